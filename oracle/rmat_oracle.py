"""ctypes wrapper around oracle/rmat_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.

The oracle evaluates eq. 4 of arxiv 1909.07321 entry by entry
in FP64 with Neumaier summation; see the header of ``rmat_oracle.c``.  Only
``tests/``, ``__graft_entry__.smoke()`` and ``bench.py``'s cpu_baseline /
``--impl reference`` legs may import this module.  It imports nothing from
``paper_1909_07321_b200`` and the product never imports it.
"""
from __future__ import annotations

import ctypes
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "rmat_oracle.c")
_LIB = os.path.join(_HERE, "liboracle_rmat.so")
_CFLAGS = ["-O2", "-std=c11", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared"]

_lib = None


def build(force: bool = False) -> str:
    """Compile the C oracle in-tree (gcc); returns the library path."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        tmp = _LIB + f".tmp{os.getpid()}"
        subprocess.run(["gcc", *_CFLAGS, _SRC, "-o", tmp, "-lm"], check=True)
        os.replace(tmp, _LIB)
    return _LIB


def _load():
    global _lib
    if _lib is None:
        lib = ctypes.CDLL(build())
        dp = ctypes.POINTER(ctypes.c_double)
        lib.oracle_rmat_form.argtypes = [dp, ctypes.c_longlong, dp, dp, ctypes.c_int, ctypes.c_int,
                                         ctypes.c_int, ctypes.c_double, dp, dp, ctypes.c_int]
        lib.oracle_rmat_form.restype = ctypes.c_int
        ip = ctypes.POINTER(ctypes.c_int)
        lib.oracle_rmat_entries.argtypes = [dp, ctypes.c_longlong, dp, dp, ctypes.c_int, ctypes.c_int, ctypes.c_int,
                                            ctypes.c_double, ctypes.c_longlong, ip, ip, ip, dp, ctypes.c_int]
        lib.oracle_rmat_entries.restype = ctypes.c_int
        lib.oracle_max_threads.argtypes = []
        lib.oracle_max_threads.restype = ctypes.c_int
        _lib = lib
    return _lib


def max_threads() -> int:
    return int(_load().oracle_max_threads())


def _dptr(a: np.ndarray):
    return a.ctypes.data_as(ctypes.POINTER(ctypes.c_double))


def rmat_form(W, E_k, energies, a: float, threads: int = 1, diag_add=None) -> np.ndarray:
    """R[e, n, m] of eq. 4 for one partial wave.

    W [n_chan, n_poles], E_k [n_poles], energies [n_E].  A float64 W whose rows are contiguous (unit stride
    along the poles) is passed as it is, with its row stride as the leading dimension ldw >= n_poles (a
    column slice of a wider array is NOT copied); anything else is made contiguous first.
    diag_add, if given, is [n_E, n_chan] and is added to the diagonal of each R[e] (see rmat_oracle.c).
    """
    W = np.asarray(W, dtype=np.float64)
    if W.ndim != 2:
        raise ValueError("W must be [n_chan, n_poles]")
    item = W.itemsize
    rows_ok = W.shape[1] <= 1 or W.strides[1] == item
    ld_ok = W.shape[0] <= 1 or (W.strides[0] % item == 0 and W.strides[0] // item >= W.shape[1])
    if not (rows_ok and ld_ok):
        W = np.ascontiguousarray(W)
    E_k = np.ascontiguousarray(E_k, dtype=np.float64)
    energies = np.ascontiguousarray(energies, dtype=np.float64)
    if E_k.ndim != 1 or energies.ndim != 1 or W.shape[1] != E_k.shape[0]:
        raise ValueError("shape mismatch: W [n_chan, n_poles], E_k [n_poles], energies [n_E]")
    n_chan, n_poles = W.shape
    ldw = W.strides[0] // item if n_chan > 1 else n_poles
    n_E = energies.shape[0]
    da = None
    if diag_add is not None:
        da = np.ascontiguousarray(diag_add, dtype=np.float64)
        if da.shape != (n_E, n_chan):
            raise ValueError("diag_add must be [n_E, n_chan]")
    R = np.zeros((n_E, n_chan, n_chan), dtype=np.float64)
    rc = _load().oracle_rmat_form(_dptr(W), max(ldw, n_poles), _dptr(E_k), _dptr(energies),
                                  n_chan, n_poles, n_E, float(a), _dptr(da) if da is not None else None,
                                  _dptr(R), int(threads))
    if rc != 0:
        raise ValueError(f"oracle_rmat_form rejected its arguments (rc={rc})")
    return R


def rmat_entries(W, E_k, energies, a: float, e_idx, n_idx, m_idx, threads: int = 1) -> np.ndarray:
    """R[e_idx[s], n_idx[s], m_idx[s]] of eq. 4, entry by entry (for waves too large to form densely).

    W must already be a float64 array whose rows are contiguous: it is NOT copied (6.2 GB at the paper's scale).
    As in rmat_form, a row stride larger than n_poles (a column slice of a wider array) is passed on as the C
    routine's leading dimension ldw.
    """
    if not (isinstance(W, np.ndarray) and W.dtype == np.float64 and W.ndim == 2):
        raise ValueError("W must be a float64 [n_chan, n_poles] array")
    rows_ok = W.shape[1] <= 1 or W.strides[1] == W.itemsize
    ld_ok = W.shape[0] <= 1 or (W.strides[0] % W.itemsize == 0 and W.strides[0] // W.itemsize >= W.shape[1])
    if not (rows_ok and ld_ok):
        raise ValueError("W must have unit stride along the poles and a row stride of at least n_poles elements (it is not copied)")
    E_k = np.ascontiguousarray(E_k, dtype=np.float64)
    energies = np.ascontiguousarray(energies, dtype=np.float64)
    if E_k.ndim != 1 or energies.ndim != 1 or W.shape[1] != E_k.shape[0]:
        raise ValueError("shape mismatch: W [n_chan, n_poles], E_k [n_poles], energies [n_E]")
    idx = [np.ascontiguousarray(x, dtype=np.int32) for x in (e_idx, n_idx, m_idx)]
    if not (idx[0].ndim == 1 and idx[0].shape == idx[1].shape == idx[2].shape):
        raise ValueError("e_idx, n_idx, m_idx must be 1-D and of equal length")
    n_chan, n_poles = W.shape
    ldw = max(W.strides[0] // W.itemsize, n_poles) if n_chan > 1 else n_poles
    out = np.zeros(idx[0].shape[0], dtype=np.float64)
    ip = ctypes.POINTER(ctypes.c_int)
    rc = _load().oracle_rmat_entries(_dptr(W), ldw, _dptr(E_k), _dptr(energies), n_chan, n_poles,
                                     energies.shape[0], float(a), out.shape[0],
                                     idx[0].ctypes.data_as(ip), idx[1].ctypes.data_as(ip), idx[2].ctypes.data_as(ip),
                                     _dptr(out), int(threads))
    if rc != 0:
        raise ValueError(f"oracle_rmat_entries rejected its arguments (rc={rc})")
    return out


def rmat_form_batch(waves, threads: int = 1) -> list[np.ndarray]:
    """Eq. 4 for each partial wave of a ragged batch (objects with W, E_k, energies, a)."""
    return [rmat_form(w.W, w.E_k, w.energies, w.a, threads=threads) for w in waves]
