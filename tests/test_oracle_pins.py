"""Pins for the CPU oracle (oracle/rmat_oracle.c) against what eq. 4
and the mathematics fix -- never against itself and never against the CUDA path.

Each pin is chosen so that a plausible mistake (dropped 1/2, 1/a vs 1/(2a),
sign of E_k - E, wrong index or stride, transposed W, missing term, skipped
last pole) fails at least one of them.
"""
import os
from fractions import Fraction

import numpy as np
import pytest

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, *vals = line.split()
            out[key] = np.array([float(v) for v in vals])
    return out


def _exact_eq4(W, E_k, energies, a):
    """Eq. 4 in exact rational arithmetic, rounded once to double."""
    C, K = W.shape
    R = np.zeros((len(energies), C, C))
    Wf = [[Fraction(float(x)) for x in row] for row in W]
    Ef = [Fraction(float(x)) for x in E_k]
    for e, E in enumerate(energies):
        Ee = Fraction(float(E))
        for n in range(C):
            for m in range(C):
                s = sum(Wf[n][k] * Wf[m][k] / (Ef[k] - Ee) for k in range(K))
                R[e, n, m] = float(s / (2 * Fraction(float(a))))
    return R


def _ulp_diff(x, y):
    scale = np.spacing(np.maximum(np.abs(x), np.abs(y)))
    return np.max(np.abs(x - y) / scale)


# ---- pin 2: hand example (tests/golden/eq4_hand_example.txt) -----------------------------
def test_hand_example_exact(oracle):
    g = _read_golden("eq4_hand_example.txt")
    W = g["W"].reshape(2, 2)
    R = oracle.rmat_form(W, g["E_k"], g["energies"], float(g["a"][0]))
    assert R.shape == (2, 2, 2)
    np.testing.assert_array_equal(R.ravel(), g["R"])


# ---- pin 1: exact rational brute force on tiny inputs ------------------------------------
@pytest.mark.parametrize("seed,C,K,N", [(0, 1, 1, 1), (1, 2, 3, 2), (2, 3, 8, 4), (3, 4, 5, 3), (4, 4, 7, 2)])
def test_exact_rational_brute_force(oracle, seed, C, K, N):
    rng = np.random.default_rng(seed)
    W = rng.normal(0, 0.3, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    energies = rng.uniform(60, 70, N) if seed % 2 else rng.uniform(-20, -10, N)
    if seed == 2:  # energies between poles: mixed-sign terms, cancellation
        energies = (E_k[:N] + E_k[1:N + 1]) / 2
    a = 7.25
    R = oracle.rmat_form(W, E_k, energies, a)
    Rx = _exact_eq4(W, E_k, energies, a)
    # compensated sum of correctly rounded terms then one division: a few ulp of the
    # result unless the sum cancels; bound relative to sum |terms| instead
    bound = np.zeros_like(Rx)
    for e, E in enumerate(energies):
        bound[e] = (np.abs(W)[:, None, :] * np.abs(W)[None, :, :] / np.abs(E_k - E)).sum(-1) / (2 * a)
    assert np.all(np.abs(R - Rx) <= 4 * np.finfo(float).eps * bound + 0.0)
    assert R.shape == (N, C, C)


def test_long_double_medium(oracle):
    """80-bit extended-precision triple loop at a size with many tiles' worth of poles."""
    rng = np.random.default_rng(11)
    C, K, N = 9, 333, 3
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    energies = np.array([0.7, 11.3, 49.2])
    a = 20.0
    Wl = W.astype(np.longdouble)
    R = oracle.rmat_form(W, E_k, energies, a)
    for e, E in enumerate(energies):
        d = 1 / (E_k.astype(np.longdouble) - np.longdouble(E))
        Rl = np.einsum("nk,mk,k->nm", Wl, Wl, d) / (2 * np.longdouble(a))
        assert np.max(np.abs(R[e] - Rl.astype(np.float64))) <= 1e-15 * np.max(np.abs(Rl))


# ---- pin 3: single-pole closed form R = w w^T / (2a (E_1 - E)) --------------------------
def test_single_pole_closed_form_bitwise(oracle):
    rng = np.random.default_rng(5)
    w = rng.normal(0, 1, (6, 1))
    E1, a = 3.125, 11.0
    energies = np.array([-1.0, 2.0, 4.5, 100.0])
    R = oracle.rmat_form(w, np.array([E1]), energies, a)
    for e, E in enumerate(energies):
        expect = (w * w.T) / (E1 - E) / (2 * a)
        np.testing.assert_array_equal(R[e], expect)
    # sign (reading R2): R_ii > 0 below the pole, < 0 above
    assert np.all(np.diagonal(R[1]) > 0) and np.all(np.diagonal(R[2]) < 0)


# ---- pin 4: symmetry, bitwise ------------------------------------------------------------
def test_symmetry_bitwise(oracle):
    rng = np.random.default_rng(6)
    W = rng.normal(0, 0.1, (13, 77))
    E_k = np.sort(rng.uniform(-5, 50, 77))
    R = oracle.rmat_form(W, E_k, np.array([0.3, 7.7]), 20.0)
    np.testing.assert_array_equal(R, np.swapaxes(R, 1, 2))


# ---- pin 5: definiteness and rank --------------------------------------------------------
def test_definiteness_and_rank(oracle):
    rng = np.random.default_rng(7)
    C, K = 10, 40
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(1, 50, K))
    R = oracle.rmat_form(W, E_k, np.array([0.5, 60.0]), 20.0)
    ev_below = np.linalg.eigvalsh(R[0])   # all E_k > E  => R >= 0
    ev_above = np.linalg.eigvalsh(R[1])   # all E_k < E  => R <= 0
    assert ev_below.min() >= -1e-13 * np.abs(ev_below).max() and ev_below.max() > 0
    assert ev_above.max() <= 1e-13 * np.abs(ev_above).max() and ev_above.min() < 0
    # rank(R) <= min(C, K)
    W2 = rng.normal(0, 0.1, (C, 4))
    R2 = oracle.rmat_form(W2, np.array([1.0, 2.0, 3.0, 4.0]), np.array([0.0]), 20.0)[0]
    ev = np.sort(np.abs(np.linalg.eigvalsh(R2)))
    assert ev[C - 4 - 1] <= 1e-14 * ev[-1] and ev[C - 4] > 1e-6 * ev[-1]


# ---- pin 6: resolvent identity and monotonicity ------------------------------------------
def test_resolvent_identity_and_monotonicity(oracle):
    rng = np.random.default_rng(8)
    C, K = 7, 50
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    gap = int(np.argmax(np.diff(E_k)))
    E1 = E_k[gap] + 0.25 * (E_k[gap + 1] - E_k[gap])
    E2 = E_k[gap] + 0.75 * (E_k[gap + 1] - E_k[gap])
    a = 20.0
    R = oracle.rmat_form(W, E_k, np.array([E1, E2]), a)
    # (R(E2)-R(E1))/(E2-E1) = (1/2a) sum_k w w^T / ((E_k-E1)(E_k-E2)): a different formula
    rhs = np.einsum("nk,mk,k->nm", W, W, 1 / ((E_k - E1) * (E_k - E2))) / (2 * a)
    lhs = (R[1] - R[0]) / (E2 - E1)
    assert np.max(np.abs(lhs - rhs)) <= 1e-12 * np.max(np.abs(rhs))
    # dR/dE >= 0 on a pole-free interval: diagonal strictly increasing, difference PSD
    assert np.all(np.diagonal(R[1]) > np.diagonal(R[0]))
    assert np.linalg.eigvalsh(R[1] - R[0]).min() >= -1e-13 * np.abs(R[1] - R[0]).max()


# ---- pin 7: exact scalings (bitwise) -----------------------------------------------------
def test_exact_scalings_bitwise(oracle):
    rng = np.random.default_rng(9)
    C, K = 5, 33
    W = rng.normal(0, 0.1, (C, K))
    # poles and energies on a 2^-20 grid so that a common shift is exact
    E_k = np.sort(np.round(rng.uniform(-5, 50, K) * 2 ** 20) / 2 ** 20)
    energies = np.round(np.array([0.37, 12.9]) * 2 ** 20) / 2 ** 20 + 2.0 ** -21
    a = 20.0
    R = oracle.rmat_form(W, E_k, energies, a)
    np.testing.assert_array_equal(oracle.rmat_form(W, E_k, energies, 2 * a), R / 2)     # 1/(2a), not 1/a^2 ...
    np.testing.assert_array_equal(oracle.rmat_form(2 * W, E_k, energies, a), 4 * R)     # quadratic in w
    np.testing.assert_array_equal(oracle.rmat_form(W, E_k + 0.5, energies + 0.5, a), R)  # depends on E_k - E only
    # a = 1/2 makes the prefactor exactly 1: R_nm = sum_k w_nk w_mk/(E_k-E)
    R1 = oracle.rmat_form(W[:, :1], E_k[:1], energies[:1], 0.5)[0]
    np.testing.assert_array_equal(R1, (W[:, :1] * W[:, :1].T) / (E_k[0] - energies[0]))


# ---- pin 8: permutations -----------------------------------------------------------------
def test_permutations(oracle):
    rng = np.random.default_rng(10)
    C, K = 6, 64
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    energies = np.array([1.234, 30.5])
    R = oracle.rmat_form(W, E_k, energies, 20.0)
    p = rng.permutation(C)
    Rp = oracle.rmat_form(W[p], E_k, energies, 20.0)
    np.testing.assert_array_equal(Rp, R[:, p][:, :, p])          # channel permutation: P R P^T bitwise
    q = rng.permutation(K)
    Rq = oracle.rmat_form(W[:, q], E_k[q], energies, 20.0)       # pole order: only rounding changes
    assert np.max(np.abs(Rq - R)) <= 1e-15 * np.max(np.abs(R))


# ---- pin 9: block structure --------------------------------------------------------------
def test_block_structure_exact_zeros(oracle):
    rng = np.random.default_rng(12)
    W = np.zeros((8, 20))
    W[:4, :10] = rng.normal(0, 0.1, (4, 10))
    W[4:, 10:] = rng.normal(0, 0.1, (4, 10))
    E_k = np.sort(rng.uniform(-5, 50, 20))
    R = oracle.rmat_form(W, E_k, np.array([0.11, 20.0]), 20.0)
    assert np.all(R[:, :4, 4:] == 0) and np.all(R[:, 4:, :4] == 0)
    assert np.all(R[:, :4, :4] != 0) and np.all(R[:, 4:, 4:] != 0)
    # and the diagonal blocks are the R-matrices of the two sub-problems
    Ra = oracle.rmat_form(W[:4, :10], E_k[:10], np.array([0.11, 20.0]), 20.0)
    np.testing.assert_array_equal(R[:, :4, :4], Ra)


# ---- pin 10: additivity over pole sets ---------------------------------------------------
def test_additivity_over_poles(oracle):
    rng = np.random.default_rng(13)
    C, K = 5, 90
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    energies = np.array([2.2, 44.0])
    R = oracle.rmat_form(W, E_k, energies, 20.0)
    RA = oracle.rmat_form(W[:, :37], E_k[:37], energies, 20.0)
    RB = oracle.rmat_form(W[:, 37:], E_k[37:], energies, 20.0)
    assert np.max(np.abs(R - (RA + RB))) <= 2e-15 * np.max(np.abs(R))
    # the last pole is really included (an off-by-one in k would drop it)
    Rm = oracle.rmat_form(W[:, :-1], E_k[:-1], energies, 20.0)
    last = (W[:, -1:] * W[:, -1:].T)[None] / (E_k[-1] - energies)[:, None, None] / 40.0
    assert np.max(np.abs((R - Rm) - last)) <= 1e-15 * np.max(np.abs(R))


# ---- pin 11: degenerate poles reduce to a library SYRK; general case vs numpy ------------
def test_degenerate_poles_vs_library_syrk(oracle):
    rng = np.random.default_rng(14)
    C, K = 12, 200
    W = rng.normal(0, 0.1, (C, K))
    E0, E, a = 5.0, 1.5, 20.0
    R = oracle.rmat_form(W, np.full(K, E0), np.array([E]), a)[0]
    expect = (W @ W.T) / (2 * a * (E0 - E))
    assert np.max(np.abs(R - expect)) <= 4e-16 * K ** 0.5 * np.max(np.abs(expect))


def test_general_case_vs_numpy_matmul(oracle):
    rng = np.random.default_rng(15)
    C, K, N = 17, 340, 5
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    energies = np.linspace(0.3, 9.7, N)
    a = 20.0
    R = oracle.rmat_form(W, E_k, energies, a)
    for e, E in enumerate(energies):
        expect = ((W * (1.0 / (E_k - E))) @ W.T) / (2 * a)
        assert np.max(np.abs(R[e] - expect)) <= 1e-14 * np.max(np.abs(expect))
    # W is [n_chan, n_poles] with k contiguous: feeding the transpose's memory must differ
    Wt = np.ascontiguousarray(W.T).reshape(C, K)
    assert np.max(np.abs(oracle.rmat_form(Wt, E_k, energies, a) - R)) > 1e-3 * np.max(np.abs(R))


# ---- shapes, threads, degenerate sizes ---------------------------------------------------
def test_threads_do_not_change_bits(oracle):
    rng = np.random.default_rng(16)
    W = rng.normal(0, 0.1, (9, 60))
    E_k = np.sort(rng.uniform(-5, 50, 60))
    energies = np.linspace(50.5, 60, 11)
    np.testing.assert_array_equal(oracle.rmat_form(W, E_k, energies, 20.0, threads=1),
                                  oracle.rmat_form(W, E_k, energies, 20.0, threads=4))


def test_degenerate_sizes(oracle):
    W = np.zeros((3, 0))
    R = oracle.rmat_form(W, np.zeros(0), np.array([1.0, 2.0]), 20.0)
    assert R.shape == (2, 3, 3) and np.all(R == 0)          # empty sum
    assert oracle.rmat_form(np.zeros((0, 4)), np.arange(4.0), np.array([9.0]), 20.0).shape == (1, 0, 0)
    assert oracle.rmat_form(np.ones((2, 4)), np.arange(4.0), np.zeros(0), 20.0).shape == (0, 2, 2)
    with pytest.raises(ValueError):
        oracle.rmat_form(np.ones((2, 4)), np.arange(3.0), np.array([9.0]), 20.0)


def test_compensation_is_live(oracle):
    """Neumaier's sum recovers what a plain FP64 sum loses (the flags keep it from being optimised out)."""
    K = 3000
    w = np.ones((1, K))
    # terms 1/(E_k - E): one huge, then many small ones that a plain sum drops
    E_k = np.concatenate([[1e-16], np.full(K - 1, 1.0)])
    R = oracle.rmat_form(w, E_k, np.array([0.0]), 0.5)[0, 0, 0]
    exact = Fraction(1) / Fraction(1e-16) + (K - 1)
    assert R == float(exact)
    plain = 0.0
    for t in 1.0 / E_k:
        plain += t
    assert plain != float(exact)  # the pin would be vacuous otherwise


def test_entries_agree_with_dense_and_exact(oracle):
    """oracle_rmat_entries (sampled outputs of waves too large to form densely) is the dense routine's
    eq4_entry: bitwise equal to it, and pinned on its own against the exact rational value."""
    rng = np.random.default_rng(31)
    C, K, N = 5, 7, 3
    W = rng.normal(0, 0.1, (C, K))
    E_k = np.sort(rng.uniform(-5, 50, K))
    en = np.array([0.3, 4.4, 9.1])
    R = oracle.rmat_form(W, E_k, en, 20.0)
    e, n, m = np.meshgrid(np.arange(N), np.arange(C), np.arange(C), indexing="ij")
    got = oracle.rmat_entries(W, E_k, en, 20.0, e.ravel(), n.ravel(), m.ravel(), threads=3)
    assert np.array_equal(got.reshape(N, C, C), R)
    exact = _exact_eq4(W, E_k, en, 20.0)
    assert np.abs(got.reshape(N, C, C) - exact).max() <= 64 * np.finfo(float).eps * np.abs(exact).max()
    with pytest.raises(ValueError):
        oracle.rmat_entries(W, E_k, en, 20.0, [3], [0], [0])          # energy index out of range
    with pytest.raises(ValueError):
        oracle.rmat_entries(W, E_k, en, 20.0, [0], [0], [C])
    assert oracle.rmat_entries(W, E_k, en, 20.0, [], [], []).shape == (0,)


# ---- the leading dimension: W as a column slice of a wider array (ldw > n_poles) ------------------------------
def test_leading_dimension_is_honoured(oracle):
    """W handed over with a row stride larger than n_poles (the C routine's ldw): exact rational brute force on
    the strided array, and bitwise the compact copy's result.  The padding holds poison (NaN) so that a stride or
    bound bug (reading column n_poles, or row n with pitch n_poles) cannot go unseen."""
    rng = np.random.default_rng(77)
    C, K, N, pad = 4, 6, 3, 5
    wide = np.full((C, K + pad), np.nan)
    wide[:, :K] = rng.uniform(-1.0, 1.0, (C, K))
    Wv = wide[:, :K]
    assert Wv.strides[0] == (K + pad) * 8 and not Wv.flags.c_contiguous
    E_k = np.sort(rng.uniform(-2.0, 6.0, K))
    en = np.array([-3.0, 1.234, 7.5])
    R = oracle.rmat_form(Wv, E_k, en, 3.0)
    assert np.all(np.isfinite(R))
    exact = _exact_eq4(np.ascontiguousarray(Wv), E_k, en, 3.0)
    Wc = np.ascontiguousarray(Wv)
    for e, E in enumerate(en):          # same bound as test_exact_rational_brute_force: relative to sum |terms|
        bound = (np.abs(Wc)[:, None, :] * np.abs(Wc)[None, :, :] / np.abs(E_k - E)).sum(-1) / (2 * 3.0)
        assert np.all(np.abs(R[e] - exact[e]) <= 4 * np.finfo(float).eps * bound)
    assert np.array_equal(R, oracle.rmat_form(np.ascontiguousarray(Wv), E_k, en, 3.0))
    # the entry-by-entry routine takes the same strided W (its own ldw argument): every entry, bitwise the dense
    # result, with the NaN padding one element past every row; a W that is not contiguous along the poles is refused
    ee, nn, mm = (x.ravel() for x in np.meshgrid(np.arange(N), np.arange(C), np.arange(C), indexing="ij"))
    assert np.array_equal(oracle.rmat_entries(Wv, E_k, en, 3.0, ee, nn, mm).reshape(N, C, C), R)
    with pytest.raises(ValueError):
        oracle.rmat_entries(np.ascontiguousarray(Wv.T).T, E_k, en, 3.0, [0], [0], [0])


# ---- the diagonal addend (where a caller's Buttle correction goes) -------------------
def test_diag_add_exact_and_local(oracle):
    """R[e][n][n] = eq. 4 + diag_add[e][n]: exact rational brute force including the addend; a zero addend is
    bitwise the plain result; off-diagonal entries are bitwise untouched; the addend enters once, after the 1/(2a)
    (a -> 2a halves eq. 4's part only), on the right energy and channel (an addend that is non-zero in one slot)."""
    rng = np.random.default_rng(91)
    C, K, N, a = 3, 5, 4, 2.0
    W = rng.uniform(-1.0, 1.0, (C, K))
    E_k = np.sort(rng.uniform(-2.0, 6.0, K))
    en = np.array([-3.0, 0.77, 2.5, 9.0])
    da = rng.uniform(-0.5, 0.5, (N, C))
    plain = oracle.rmat_form(W, E_k, en, a)
    R = oracle.rmat_form(W, E_k, en, a, diag_add=da)
    assert np.array_equal(plain, oracle.rmat_form(W, E_k, en, a, diag_add=np.zeros((N, C))))
    off = ~np.eye(C, dtype=bool)
    assert np.array_equal(R[:, off], plain[:, off])
    # exact: (sum / 2a) + addend in rationals, rounded once; the oracle rounds twice (eq. 4, then the add): <= 1 ulp more
    for e in range(N):
        for n in range(C):
            s = sum(Fraction(float(W[n, k])) ** 2 / (Fraction(float(E_k[k])) - Fraction(float(en[e]))) for k in range(K))
            exact = float(s / (2 * Fraction(a)) + Fraction(float(da[e, n])))
            assert abs(R[e, n, n] - exact) <= 3 * np.spacing(max(abs(exact), abs(plain[e, n, n]), abs(da[e, n])))
            assert R[e, n, n] == plain[e, n, n] + da[e, n]            # one rounded add, after the division by 2a
    # where a and the addend enter: doubling a halves eq. 4's part and leaves the addend alone
    R2 = oracle.rmat_form(W, E_k, en, 2 * a, diag_add=da)
    idx = np.arange(C)
    assert np.array_equal(R2[:, idx, idx], plain[:, idx, idx] / 2 + da)
    # locality: one non-zero slot moves exactly one entry
    one = np.zeros((N, C))
    one[2, 1] = 0.125
    R1 = oracle.rmat_form(W, E_k, en, a, diag_add=one)
    diff = R1 != plain
    assert diff.sum() == 1 and diff[2, 1, 1]
    with pytest.raises(ValueError):
        oracle.rmat_form(W, E_k, en, a, diag_add=np.zeros((C, N)))   # transposed shape is rejected
