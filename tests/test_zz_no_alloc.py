"""pstgf_rmat_form_static: the single-wave call for callers that cannot allocate device memory.

Some users of this library have no way to let it call cudaMalloc: all of the GPU's memory already belongs to their
own arena (a framework's caching allocator, or the fixed slice of a GPU that several MPI ranks share, which is how the
paper runs RINIT, Fig. 2), their per-energy loop cannot stand the device-wide synchronisation an
allocation or a free may bring, or the calling thread sits inside its framework's allocator.  For them the library
keeps a 16 MiB scratch array inside its own device image and pstgf_rmat_form_static works out of that.

What is checked here, through the C ABI on cuda:0:
  * its R equals pstgf_rmat_form's -- bitwise, and in the per-energy relative measure of the parity tests at their
    1e-13 -- for pair-form waves (P, D and the pair table in the array) and for a symmetric-form wave with more items
    than CTAs (work counter in the array), each on TWO CALLS IN A ROW that are enqueued without a synchronise in
    between, with different waves, so the second call runs over what the first left in the array;
  * one of the waves against the CPU oracle as well;
  * a wave beyond the array's size is refused with PSTGF_ERR_STATIC_LIMIT and R_out is left alone;
  * the free device memory does not move over a round of calls (after a first round has loaded the kernels).

The file name sorts last on purpose: `pytest -x` stops at the first failure, and a failure here must not hide the
parity tests.  Nothing in it depends on what ran before it in the process.
"""
import numpy as np
import pytest

torch = pytest.importorskip("torch")

pytestmark = pytest.mark.gpu

TOL_TIGHT = 1e-13    # the parity tests' bar (tests/test_parity_gpu.py)

# (seed, n_chan, n_poles, n_E).  Pair form (n_chan <= 96, n_E >= 64; more than 16 channels keeps them off the
# one-launch kernel, which needs no scratch): 6.9 MB, 1.5 MB and (odd n_poles, ragged pair tiles) 3.6 MB of scratch.
PAIR_A = (11, 40, 800, 256)
PAIR_B = (12, 24, 480, 100)
PAIR_C = (13, 33, 463, 300)
# Symmetric form, 10 tiles x 20 energy blocks = 200 items for 148 CTAs: the work counter is drawn from.
SYRK_A = (14, 200, 1000, 160)
SYRK_B = (15, 131, 524, 250)


@pytest.fixture(scope="module")
def rmat():
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1909_07321_b200 import rmat as m
    m.load()     # raises if the library is missing: no fallback
    return m


def _wave(spec):
    from paper_1909_07321_b200 import inputs
    return inputs.make_wave(*spec)


def _dev(w):
    c = lambda x: torch.from_numpy(np.ascontiguousarray(x)).cuda()
    return c(w.W), c(w.E_k), c(w.energies)


def _rel_err_per_energy(got, ref):
    num = np.abs(got - ref).reshape(ref.shape[0], -1).max(axis=1)
    den = np.abs(ref).reshape(ref.shape[0], -1).max(axis=1)
    return num / den


def _two_in_a_row(rmat, spec1, spec2):
    """static(wave 1) and static(wave 2) back to back on one stream, no synchronise in between; then the same two
    waves through pstgf_rmat_form.  Returns [(wave, R_static, R_form)] as numpy."""
    waves = [_wave(spec1), _wave(spec2)]
    dev = [_dev(w) for w in waves]
    outs = [torch.full((w.n_E, w.n_chan, w.n_chan), float("nan"), dtype=torch.float64, device="cuda") for w in waves]
    for w, d, R in zip(waves, dev, outs):
        rmat.pstgf_rmat_form_static(d[0], d[1], d[2], w.a, R)
    torch.cuda.synchronize()
    refs = [rmat.pstgf_rmat_form(d[0], d[1], d[2], w.a) for w, d in zip(waves, dev)]
    torch.cuda.synchronize()
    return [(w, R.cpu().numpy(), ref.cpu().numpy()) for w, R, ref in zip(waves, outs, refs)]


def _assert_same(got, ref):
    assert np.all(np.isfinite(got))
    err = _rel_err_per_energy(got, ref)
    assert err.max() <= TOL_TIGHT, f"static vs pstgf_rmat_form: max rel err {err.max():.3e} at energy {int(err.argmax())}"
    assert np.array_equal(got, ref), "same plan, same kernels: the two calls should agree bitwise"
    assert np.array_equal(got, np.swapaxes(got, 1, 2))


@pytest.mark.parametrize("first,second", [(PAIR_A, PAIR_B), (PAIR_B, PAIR_A), (PAIR_C, PAIR_C)])
def test_pair_form_scratch_in_the_static_array(rmat, first, second):
    for _, got, ref in _two_in_a_row(rmat, first, second):
        _assert_same(got, ref)


def test_work_counter_in_the_static_array(rmat):
    for _, got, ref in _two_in_a_row(rmat, SYRK_A, SYRK_B):
        _assert_same(got, ref)
    # the counter was really used: one 16-byte memset ahead of the one persistent launch
    w = _wave(SYRK_A)
    d = _dev(w)
    R = torch.empty((w.n_E, w.n_chan, w.n_chan), dtype=torch.float64, device="cuda")
    rmat.pstgf_rmat_form_static(d[0], d[1], d[2], w.a, R)
    assert rmat.pstgf_last_launch_count() == 2
    torch.cuda.synchronize()
    # and a pair-form call ahead of a symmetric-form one: counter and scratch share the array
    for _, got, ref in _two_in_a_row(rmat, PAIR_A, SYRK_A):
        _assert_same(got, ref)


def test_against_the_oracle(rmat, oracle):
    import os
    (w1, got1, _), (w2, got2, _) = _two_in_a_row(rmat, PAIR_B, SYRK_B)
    for w, got in ((w1, got1), (w2, got2)):
        ref = oracle.rmat_form(w.W, w.E_k, w.energies, w.a, threads=os.cpu_count() or 1)
        err = _rel_err_per_energy(got, ref)
        assert err.max() <= TOL_TIGHT, f"static vs oracle: max rel err {err.max():.3e}"


def test_too_large_a_wave_is_refused(rmat):
    # BASELINE.json configs[1]: 64 x 1280 with 4096 energies wants 63 MB of pair-form scratch
    n_chan, n_poles, n_E = 64, 1280, 4096
    W = torch.zeros((n_chan, n_poles), dtype=torch.float64, device="cuda")
    E_k = torch.arange(n_poles, dtype=torch.float64, device="cuda") + 100.0
    E = torch.linspace(0.1, 20.0, n_E, dtype=torch.float64, device="cuda")
    R = torch.full((n_E, n_chan, n_chan), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(rmat.PstgfError) as ei:
        rmat.pstgf_rmat_form_static(W, E_k, E, 20.0, R)
    assert ei.value.status == rmat.PSTGF_ERR_STATIC_LIMIT
    assert "STATIC" in str(ei.value)
    torch.cuda.synchronize()
    assert bool((R == 7.0).all())                       # nothing was enqueued
    # the same wave in the symmetric form needs the counter only and goes through
    rmat.pstgf_debug_set_pair_policy(rmat.PSTGF_PAIRS_NONE)
    try:
        rmat.pstgf_rmat_form_static(W, E_k, E[:16], 20.0, R[:16])
        torch.cuda.synchronize()
        assert bool((R[:16] == 0.0).all()) and bool((R[16:] == 7.0).all())
    finally:
        rmat.pstgf_debug_set_pair_policy(rmat.PSTGF_PAIRS_AUTO)


def test_free_device_memory_does_not_move(rmat):
    specs = [PAIR_A, SYRK_A, PAIR_C, SYRK_B]
    waves = [_wave(s) for s in specs]
    dev = [_dev(w) for w in waves]
    outs = [torch.empty((w.n_E, w.n_chan, w.n_chan), dtype=torch.float64, device="cuda") for w in waves]

    def one_round():
        for w, d, R in zip(waves, dev, outs):
            rmat.pstgf_rmat_form_static(d[0], d[1], d[2], w.a, R)
        torch.cuda.synchronize()

    one_round()                                          # loads the kernels, looks the array's address up
    free_before, _ = torch.cuda.mem_get_info()
    for _ in range(3):
        one_round()
    free_after, _ = torch.cuda.mem_get_info()
    assert free_after >= free_before, f"device memory was taken during the calls: {free_before - free_after} bytes"
