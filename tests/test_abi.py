"""The C-ABI boundary without a GPU: libpstgf_rmat.so loads, exports every symbol that
include/pstgf_rmat.h declares, the Python binding covers the same names, the struct layout
matches the header, and argument errors are reported before any CUDA call is made.
"""
import ctypes
import os
import re
import subprocess

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
HEADER = os.path.join(ROOT, "include", "pstgf_rmat.h")


def _declared_functions():
    src = open(HEADER).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)          # drop comments
    src = re.sub(r"^\s*#.*$", "", src, flags=re.M)            # and preprocessor lines
    names = re.findall(r"\b(pstgf_[a-z0-9_]+)\s*\(", src)
    return sorted(set(names))


@pytest.fixture(scope="module")
def lib():
    from paper_1909_07321_b200 import build
    path = build.build()              # compiles only if missing or stale (nvcc cross-compiles without a GPU)
    return ctypes.CDLL(path)


def test_header_declares_the_boundary_calls():
    names = _declared_functions()
    for required in ("pstgf_rmat_form", "pstgf_rmat_form_batch", "pstgf_rmat_batch_workspace_bytes",
                     "pstgf_status_string", "pstgf_last_cuda_error", "pstgf_version"):
        assert required in names


def test_library_exports_every_declared_symbol(lib):
    for name in _declared_functions():
        assert hasattr(lib, name), f"{name} is declared in include/pstgf_rmat.h but not exported"


def test_binding_lists_the_same_names():
    from paper_1909_07321_b200 import rmat
    assert sorted(rmat.EXPORTS) == _declared_functions()
    for name in _declared_functions():
        if name in ("pstgf_last_cuda_error",):
            continue                                           # surfaced through PstgfError only
        assert hasattr(rmat, name), f"binding lacks {name}"


def test_header_compiles_as_plain_c(tmp_path):
    """The boundary is C: no C++ or torch types in the signatures."""
    c = tmp_path / "use_header.c"
    c.write_text('#include "pstgf_rmat.h"\n'
                 "int main(void) { pstgf_wave_t w; (void)w; return sizeof(pstgf_wave_t) == 72 ? 0 : 1; }\n")
    exe = tmp_path / "use_header"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-pedantic", "-I", os.path.join(ROOT, "include"),
                    str(c), "-o", str(exe)], check=True)
    assert subprocess.run([str(exe)]).returncode == 0


def test_wave_struct_layout_matches_binding():
    from paper_1909_07321_b200 import rmat
    assert ctypes.sizeof(rmat.pstgf_wave_t) == 72
    off = {n: getattr(rmat.pstgf_wave_t, n).offset for n, _ in rmat.pstgf_wave_t._fields_}
    assert off == {"n_chan": 0, "n_poles": 4, "n_E": 8, "w_layout": 12, "ldw": 16, "a": 24, "W": 32, "E_k": 40, "energies": 48,
                   "R_out": 56, "diag_add": 64}
    m = re.search(r"#define\s+PSTGF_RMAT_VERSION\s+(\d+)", open(HEADER).read())
    assert rmat.PSTGF_RMAT_VERSION == int(m.group(1))


def test_version_and_status_strings(lib):
    lib.pstgf_version.restype = ctypes.c_int
    lib.pstgf_status_string.restype = ctypes.c_char_p
    lib.pstgf_status_string.argtypes = [ctypes.c_int]
    m = re.search(r"#define\s+PSTGF_RMAT_VERSION\s+(\d+)", open(HEADER).read())
    assert lib.pstgf_version() == int(m.group(1))
    seen = set()
    for code in range(9):
        s = lib.pstgf_status_string(code).decode()
        assert s and s not in seen
        seen.add(s)
    assert b"unknown" in lib.pstgf_status_string(99)


def test_argument_errors_need_no_device(lib):
    """Argument checks come before any CUDA call, so they can be exercised here (no compute)."""
    vp, ll, i, d = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_double
    lib.pstgf_rmat_form.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form.restype = i
    fake = 4096                                                   # never dereferenced: the call fails first
    assert lib.pstgf_rmat_form(fake, 6, fake, fake, 4, 6, 1, 0.0, fake, None) == 1      # a <= 0
    assert lib.pstgf_rmat_form(fake, 5, fake, fake, 4, 6, 1, 20.0, fake, None) == 1     # ldw < n_poles
    assert lib.pstgf_rmat_form(None, 6, fake, fake, 4, 6, 1, 20.0, fake, None) == 1     # NULL W
    assert lib.pstgf_rmat_form(fake, 6, fake, fake, -1, 6, 1, 20.0, fake, None) == 1    # negative size
    assert lib.pstgf_rmat_form(fake + 4, 6, fake, fake, 4, 6, 1, 20.0, fake, None) == 2  # misaligned
    assert lib.pstgf_rmat_form(fake, 6, fake, fake, 0, 6, 1, 20.0, fake, None) == 0     # n_chan == 0: nothing to do
    assert lib.pstgf_rmat_form(fake, 6, fake, fake, 4, 6, 0, 20.0, fake, None) == 0     # n_E == 0
    # the no-allocation call: same checks, and a wave beyond its built-in scratch is refused before any CUDA call
    lib.pstgf_rmat_form_static.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form_static.restype = i
    assert lib.pstgf_rmat_form_static(fake, 6, fake, fake, 4, 6, 1, 0.0, fake, None) == 1       # a <= 0
    assert lib.pstgf_rmat_form_static(fake + 4, 6, fake, fake, 4, 6, 1, 20.0, fake, None) == 2  # misaligned
    assert lib.pstgf_rmat_form_static(fake, 6, fake, fake, 4, 6, 0, 20.0, fake, None) == 0      # n_E == 0
    assert lib.pstgf_rmat_form_static(fake, 1280, fake, fake, 64, 1280, 4096, 20.0, fake, None) == 8   # 63 MB of pair scratch > 16 MiB
    # H.DAT record order: the leading dimension runs over channels
    lib.pstgf_rmat_form_hdat.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form_hdat.restype = i
    assert lib.pstgf_rmat_form_hdat(fake, 3, fake, fake, 4, 6, 1, 20.0, fake, None) == 1   # ldw < n_chan
    assert lib.pstgf_rmat_form_hdat(fake, 4, fake, fake, 4, 6, 0, 20.0, fake, None) == 0   # n_E == 0
    from paper_1909_07321_b200 import rmat
    lib.pstgf_rmat_form_naive.argtypes = [ctypes.POINTER(rmat.pstgf_wave_t), vp]
    lib.pstgf_rmat_form_naive.restype = i
    w = rmat.pstgf_wave_t(4, 6, 1, 7, 6, 20.0, fake, fake, fake, fake, None)
    assert lib.pstgf_rmat_form_naive(ctypes.byref(w), None) == 1                        # unknown w_layout
    w.w_layout, w.diag_add = 0, fake + 4
    assert lib.pstgf_rmat_form_naive(ctypes.byref(w), None) == 2                        # misaligned diag_add
    assert lib.pstgf_rmat_form_naive(None, None) == 1
    for name, bad in (("pstgf_debug_set_tail_policy", 5), ("pstgf_debug_set_slab_policy", 9), ("pstgf_debug_set_pair_policy", 3),
                      ("pstgf_debug_set_small_policy", 3), ("pstgf_debug_set_host_pipeline", 3)):
        f = getattr(lib, name)
        f.argtypes, f.restype = [i], i
        assert f(bad) == 1 and f(0) == 0


def test_product_library_holds_no_measurement_code(lib):
    """The FP64 throughput probe that fixes the roofline denominator is bench-side (libpstgf_probe.so): neither the
    product header nor the product library knows it."""
    assert "probe" not in open(HEADER).read()
    assert not hasattr(lib, "pstgf_fp64_probe")
    from paper_1909_07321_b200 import build
    assert hasattr(ctypes.CDLL(build.PROBE_LIB), "pstgf_fp64_probe")
    assert hasattr(ctypes.CDLL(build.PROBE_LIB), "pstgf_i8_probe") and not hasattr(lib, "pstgf_i8_probe")
    assert hasattr(ctypes.CDLL(build.PROBE_LIB), "pstgf_l2_probe") and not hasattr(lib, "pstgf_l2_probe")


def test_mesh_from_zscaled(lib):
    """input meshes are z-scaled, E/z^2.  Exact dyadic cases, aliasing, argument errors."""
    import numpy as np
    from paper_1909_07321_b200 import rmat
    e = np.array([0.0, 0.5, 1.0, -0.25, 3.0, 2.0 ** -40])
    for z in (1.0, 2.0, 3.0, 26.0, 0.5):
        out = rmat.pstgf_mesh_from_zscaled(e, z)
        assert np.array_equal(out, e * (z * z))              # exact: z*z and every product are representable here
        assert np.array_equal(out / (z * z), e)              # and E/z^2 gives the input back
    rng = np.random.default_rng(3)
    x = rng.uniform(0.0, 5.0, 1000)
    out = rmat.pstgf_mesh_from_zscaled(x, 7.0)
    assert np.array_equal(out, x * 49.0)                     # one rounding per element, as documented
    vp, ll, d = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_double
    f = lib.pstgf_mesh_from_zscaled
    f.argtypes, f.restype = [vp, ll, d, vp], ctypes.c_int
    buf = np.array([1.0, 2.0])
    assert f(buf.ctypes.data, 2, 3.0, buf.ctypes.data) == 0  # in place
    assert np.array_equal(buf, [9.0, 18.0])
    assert f(buf.ctypes.data, 2, 0.0, buf.ctypes.data) == 1  # z must be > 0
    assert f(buf.ctypes.data, 2, float("nan"), buf.ctypes.data) == 1
    assert f(buf.ctypes.data, -1, 1.0, buf.ctypes.data) == 1
    assert f(None, 2, 1.0, buf.ctypes.data) == 1
    assert f(None, 0, 1.0, None) == 0


def test_finalize_without_a_device_is_harmless(lib):
    lib.pstgf_rmat_finalize.restype = ctypes.c_int
    assert lib.pstgf_rmat_finalize() == 0
    assert lib.pstgf_rmat_finalize() == 0


def test_no_device_is_an_error_not_a_fallback(lib):
    """On a box without a GPU a well-formed call must fail loudly (there is no CPU path)."""
    torch = pytest.importorskip("torch")
    if torch.cuda.is_available():
        pytest.skip("a CUDA device is present")
    vp, ll, i, d = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_double
    lib.pstgf_rmat_form.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form.restype = i
    assert lib.pstgf_rmat_form(4096, 6, 4096, 4096, 4, 6, 1, 20.0, 4096, None) in (4, 5)


def test_product_does_not_touch_the_oracle():
    """Nothing under the package imports, links or names oracle/ (and vice versa)."""
    pkg = os.path.join(ROOT, "paper_1909_07321_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in text and "from oracle" not in text and "liboracle" not in text, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            text = open(os.path.join(ROOT, "oracle", f)).read()
            assert "import paper_1909_07321_b200" not in text and "from paper_1909_07321_b200" not in text, f
            assert "pstgf_rmat.h" not in text and "csrc/" not in text.replace("paper_1909_07321_b200/csrc", ""), f
