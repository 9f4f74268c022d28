"""Thin ctypes binding over libpstgf_rmat.so (include/pstgf_rmat.h): argument marshalling only.

Every step of eq. 4 runs in the library's sm_100a kernels.  PyTorch is used for
device memory and streams.  There is no CPU fallback: a missing library or a failing call raises.
"""
from __future__ import annotations

import ctypes
import os
from typing import Sequence

import torch

from . import build as _build

PSTGF_OK = 0
PSTGF_TAIL_AUTO, PSTGF_TAIL_NONE, PSTGF_TAIL_ALL = 0, 1, 2
PSTGF_W_POLE_CONTIGUOUS, PSTGF_W_CHANNEL_CONTIGUOUS = 0, 1
PSTGF_HOST_PIPELINE_AUTO, PSTGF_HOST_PIPELINE_CHUNKED = 0, 1
PSTGF_SLAB_AUTO, PSTGF_SLAB_NONE, PSTGF_SLAB_T32, PSTGF_SLAB_T64, PSTGF_SLAB_T128 = 0, 1, 2, 3, 4
PSTGF_PAIRS_AUTO, PSTGF_PAIRS_NONE, PSTGF_PAIRS_ALWAYS = 0, 1, 2
PSTGF_SMALL_AUTO, PSTGF_SMALL_NONE, PSTGF_SMALL_ALWAYS = 0, 1, 2
PSTGF_ERR_TIMEOUT, PSTGF_ERR_CAPTURE, PSTGF_ERR_STATIC_LIMIT = 6, 7, 8
PSTGF_STATIC_SCRATCH_BYTES = 16 << 20   # include/pstgf_rmat.h
PSTGF_RMAT_VERSION = 201            # must equal include/pstgf_rmat.h; load() checks it against the library

EXPORTS = ["pstgf_rmat_form", "pstgf_rmat_form_hdat", "pstgf_rmat_form_static", "pstgf_rmat_batch_workspace_bytes", "pstgf_rmat_form_batch",
           "pstgf_rmat_form_naive", "pstgf_rmat_form_sliced", "pstgf_rmat_sliced_workspace_bytes", "pstgf_rmat_form_batch_host", "pstgf_mesh_from_zscaled", "pstgf_rmat_finalize",
           "pstgf_debug_set_tail_policy", "pstgf_debug_set_slab_policy", "pstgf_debug_set_pair_policy", "pstgf_debug_set_small_policy",
           "pstgf_debug_set_host_pipeline",
           "pstgf_debug_set_upload_timeout_ms", "pstgf_debug_stall_upload", "pstgf_last_launch_count",
           "pstgf_status_string", "pstgf_last_cuda_error", "pstgf_version"]


class PstgfError(RuntimeError):
    def __init__(self, status: int, message: str):
        super().__init__(message)
        self.status = status


class pstgf_wave_t(ctypes.Structure):
    _fields_ = [("n_chan", ctypes.c_int), ("n_poles", ctypes.c_int), ("n_E", ctypes.c_int), ("w_layout", ctypes.c_int),
                ("ldw", ctypes.c_longlong), ("a", ctypes.c_double),
                ("W", ctypes.c_void_p), ("E_k", ctypes.c_void_p), ("energies", ctypes.c_void_p),
                ("R_out", ctypes.c_void_p), ("diag_add", ctypes.c_void_p)]


_lib = None


def library_path() -> str:
    return _build.LIB


def load(build_if_missing: bool = False):
    """Load libpstgf_rmat.so (built in-tree).  Raises if it is not there, older than its sources, or of another
    ABI version than this binding: no fallback exists."""
    global _lib
    if _lib is not None:
        return _lib
    path = library_path()
    if not os.path.exists(path) or _build.is_stale():
        if build_if_missing:
            _build.build()
        else:
            what = "is missing" if not os.path.exists(path) else "was built from other sources than csrc/ and include/pstgf_rmat.h now hold"
            raise PstgfError(-1, f"{path} {what}: run `python -m paper_1909_07321_b200.build` "
                                 "(or __graft_entry__.build()); there is no CPU fallback")
    lib = ctypes.CDLL(path)
    lib.pstgf_version.restype = ctypes.c_int
    if int(lib.pstgf_version()) != PSTGF_RMAT_VERSION:
        raise PstgfError(-1, f"{path} reports ABI version {lib.pstgf_version()}, this binding is for {PSTGF_RMAT_VERSION}: rebuild")
    vp, ll, i, d, sz = ctypes.c_void_p, ctypes.c_longlong, ctypes.c_int, ctypes.c_double, ctypes.c_size_t
    lib.pstgf_rmat_form.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form.restype = i
    lib.pstgf_rmat_form_hdat.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form_hdat.restype = i
    lib.pstgf_rmat_form_static.argtypes = [vp, ll, vp, vp, i, i, i, d, vp, vp]
    lib.pstgf_rmat_form_static.restype = i
    lib.pstgf_rmat_form_naive.argtypes = [ctypes.POINTER(pstgf_wave_t), vp]
    lib.pstgf_rmat_form_naive.restype = i
    lib.pstgf_rmat_form_sliced.argtypes = [ctypes.POINTER(pstgf_wave_t), i, vp, sz, vp]
    lib.pstgf_rmat_form_sliced.restype = i
    lib.pstgf_rmat_sliced_workspace_bytes.argtypes = [i, i, i, i]
    lib.pstgf_rmat_sliced_workspace_bytes.restype = sz
    lib.pstgf_rmat_batch_workspace_bytes.argtypes = [ctypes.POINTER(pstgf_wave_t), i]
    lib.pstgf_rmat_batch_workspace_bytes.restype = sz
    lib.pstgf_rmat_form_batch.argtypes = [ctypes.POINTER(pstgf_wave_t), i, vp, sz, vp]
    lib.pstgf_rmat_form_batch.restype = i
    lib.pstgf_rmat_form_batch_host.argtypes = [ctypes.POINTER(pstgf_wave_t), i, sz, vp]
    lib.pstgf_rmat_form_batch_host.restype = i
    for name in ("pstgf_debug_set_tail_policy", "pstgf_debug_set_slab_policy", "pstgf_debug_set_pair_policy", "pstgf_debug_set_small_policy",
                 "pstgf_debug_set_host_pipeline",
                 "pstgf_debug_stall_upload"):
        getattr(lib, name).argtypes = [i]
        getattr(lib, name).restype = i
    lib.pstgf_debug_set_upload_timeout_ms.argtypes = [ctypes.c_uint]
    lib.pstgf_debug_set_upload_timeout_ms.restype = i
    lib.pstgf_mesh_from_zscaled.argtypes = [vp, ll, d, vp]
    lib.pstgf_mesh_from_zscaled.restype = i
    lib.pstgf_rmat_finalize.argtypes = []
    lib.pstgf_rmat_finalize.restype = i
    lib.pstgf_last_launch_count.restype = i
    lib.pstgf_status_string.argtypes = [i]
    lib.pstgf_status_string.restype = ctypes.c_char_p
    lib.pstgf_last_cuda_error.restype = i
    lib.pstgf_version.restype = i
    _lib = lib
    return lib


def _check(status: int):
    if status != PSTGF_OK:
        lib = load()
        msg = lib.pstgf_status_string(status).decode()
        if status == 5:
            msg += f" (cudaError_t {lib.pstgf_last_cuda_error()})"
        raise PstgfError(status, msg)


def _stream_ptr(stream) -> int:
    if stream is None:
        stream = torch.cuda.current_stream()
    return int(stream.cuda_stream) if hasattr(stream, "cuda_stream") else int(stream)


def _dev_f64(t: torch.Tensor, name: str):
    if not isinstance(t, torch.Tensor) or t.dtype != torch.float64 or not t.is_cuda:
        raise TypeError(f"{name} must be a CUDA float64 torch.Tensor")
    return t


def _w_dims(W, layout: int):
    """(n_chan, n_poles, ldw) of a 2-D W tensor: [n_chan, n_poles] pole-contiguous, or, for
    PSTGF_W_CHANNEL_CONTIGUOUS (the H.DAT record order), [n_poles, n_chan]."""
    if W.dim() != 2 or W.stride(1) != 1 and W.shape[1] > 1:
        raise ValueError("W must be 2-D with unit stride along its last dimension")
    rows, cols = int(W.shape[0]), int(W.shape[1])
    ldw = int(W.stride(0)) if rows > 1 else max(cols, int(W.stride(0)), 1)
    return (cols, rows, ldw) if layout == PSTGF_W_CHANNEL_CONTIGUOUS else (rows, cols, ldw)


def _wave_struct(W, E_k, energies, a, R_out, layout: int = PSTGF_W_POLE_CONTIGUOUS, diag_add=None) -> pstgf_wave_t:
    _dev_f64(W, "W"); _dev_f64(E_k, "E_k"); _dev_f64(energies, "energies"); _dev_f64(R_out, "R_out")
    n_chan, n_poles, ldw = _w_dims(W, layout)
    n_E = int(energies.shape[0])
    if E_k.dim() != 1 or int(E_k.shape[0]) != n_poles or not E_k.is_contiguous():
        raise ValueError("E_k must be contiguous [n_poles]")
    if energies.dim() != 1 or not energies.is_contiguous():
        raise ValueError("energies must be contiguous [n_E]")
    if tuple(R_out.shape) != (n_E, n_chan, n_chan) or not R_out.is_contiguous():
        raise ValueError("R_out must be contiguous [n_E, n_chan, n_chan]")
    if diag_add is not None:
        _dev_f64(diag_add, "diag_add")
        if tuple(diag_add.shape) != (n_E, n_chan) or not diag_add.is_contiguous():
            raise ValueError("diag_add must be contiguous [n_E, n_chan]")
    return pstgf_wave_t(n_chan, n_poles, n_E, int(layout), ldw, float(a), W.data_ptr(), E_k.data_ptr(),
                        energies.data_ptr(), R_out.data_ptr(), diag_add.data_ptr() if diag_add is not None else None)


def pstgf_rmat_form(W, E_k, energies, a: float, R_out=None, stream=None) -> torch.Tensor:
    """R[e] = (1/2a) W diag(1/(E_k - E_e)) W^T for one partial wave (eq. 4).

    W [n_chan, n_poles] (row stride = ldw), E_k [n_poles], energies [n_E]: CUDA float64 tensors.
    Returns R_out [n_E, n_chan, n_chan] (allocated if not given).  Asynchronous on ``stream``.
    """
    lib = load()
    if R_out is None:
        R_out = torch.empty((energies.shape[0], W.shape[0], W.shape[0]), dtype=torch.float64, device=W.device)
    w = _wave_struct(W, E_k, energies, a, R_out)
    with torch.cuda.device(W.device):
        _check(lib.pstgf_rmat_form(w.W, w.ldw, w.E_k, w.energies, w.n_chan, w.n_poles, w.n_E, w.a, w.R_out,
                                   _stream_ptr(stream)))
    return R_out


def pstgf_rmat_form_static(W, E_k, energies, a: float, R_out, stream=None) -> torch.Tensor:
    """pstgf_rmat_form for callers that cannot allocate device memory (no room left beside their own arena, a loop
    that cannot stand cudaMalloc's device-wide synchronisation, a thread inside its framework's allocator): the
    library's scratch is a 16 MiB array built into its device image instead.  ``R_out`` is required -- this binding
    allocates nothing either.  Same bits as pstgf_rmat_form; a pair-form wave whose scratch exceeds the array raises
    PstgfError with status PSTGF_ERR_STATIC_LIMIT.  All calls on a device share the one array: keep them ordered
    on the GPU (one stream, or events)."""
    lib = load()
    w = _wave_struct(W, E_k, energies, a, R_out)
    with torch.cuda.device(W.device):
        _check(lib.pstgf_rmat_form_static(w.W, w.ldw, w.E_k, w.energies, w.n_chan, w.n_poles, w.n_E, w.a, w.R_out,
                                          _stream_ptr(stream)))
    return R_out


def pstgf_rmat_form_hdat(Wt, E_k, energies, a: float, R_out=None, stream=None) -> torch.Tensor:
    """pstgf_rmat_form for W in the H.DAT record order: Wt [n_poles, n_chan], channels contiguous."""
    lib = load()
    if R_out is None:
        R_out = torch.empty((energies.shape[0], Wt.shape[1], Wt.shape[1]), dtype=torch.float64, device=Wt.device)
    w = _wave_struct(Wt, E_k, energies, a, R_out, PSTGF_W_CHANNEL_CONTIGUOUS)
    with torch.cuda.device(Wt.device):
        _check(lib.pstgf_rmat_form_hdat(w.W, w.ldw, w.E_k, w.energies, w.n_chan, w.n_poles, w.n_E, w.a, w.R_out,
                                        _stream_ptr(stream)))
    return R_out


def pstgf_rmat_form_naive(W, E_k, energies, a: float, R_out=None, stream=None,
                          layout: int = PSTGF_W_POLE_CONTIGUOUS, diag_add=None) -> torch.Tensor:
    """Same result from the library's term-by-term verification kernel (slow)."""
    lib = load()
    n_chan = W.shape[1] if layout == PSTGF_W_CHANNEL_CONTIGUOUS else W.shape[0]
    if R_out is None:
        R_out = torch.empty((energies.shape[0], n_chan, n_chan), dtype=torch.float64, device=W.device)
    w = _wave_struct(W, E_k, energies, a, R_out, layout, diag_add)
    with torch.cuda.device(W.device):
        _check(lib.pstgf_rmat_form_naive(ctypes.byref(w), _stream_ptr(stream)))
    return R_out


def pstgf_rmat_sliced_workspace_bytes(n_chan: int, n_poles: int, n_E: int, n_slices: int = 7) -> int:
    return int(load().pstgf_rmat_sliced_workspace_bytes(int(n_chan), int(n_poles), int(n_E), int(n_slices)))


def pstgf_rmat_form_sliced(W, E_k, energies, a: float, n_slices: int = 7, R_out=None, workspace=None, stream=None,
                           diag_add=None) -> torch.Tensor:
    """The INT8-sliced VARIANT of eq. 4 (tcgen05.mma kind::i8; not an IEEE FP64 sum, see the header); pole-contiguous W."""
    lib = load()
    if R_out is None:
        R_out = torch.empty((energies.shape[0], W.shape[0], W.shape[0]), dtype=torch.float64, device=W.device)
    w = _wave_struct(W, E_k, energies, a, R_out, PSTGF_W_POLE_CONTIGUOUS, diag_add)
    need = int(lib.pstgf_rmat_sliced_workspace_bytes(w.n_chan, w.n_poles, w.n_E, int(n_slices)))
    if workspace is None:
        workspace = torch.empty(max(need, 1024), dtype=torch.uint8, device=W.device)
    with torch.cuda.device(W.device):
        _check(lib.pstgf_rmat_form_sliced(ctypes.byref(w), int(n_slices), workspace.data_ptr(), workspace.numel(), _stream_ptr(stream)))
    return R_out


def make_wave_array(waves: Sequence[tuple]) -> "ctypes.Array[pstgf_wave_t]":
    """waves: sequence of (W, E_k, energies, a, R_out[, w_layout[, diag_add]]) tuples of CUDA tensors."""
    arr = (pstgf_wave_t * len(waves))()
    for p, wv in enumerate(waves):
        arr[p] = _wave_struct(*wv)
    return arr


def pstgf_rmat_batch_workspace_bytes(wave_array, n_waves: int | None = None) -> int:
    lib = load()
    n = len(wave_array) if n_waves is None else n_waves
    return int(lib.pstgf_rmat_batch_workspace_bytes(wave_array, n))


def pstgf_rmat_form_batch(wave_array, workspace: torch.Tensor, stream=None, n_waves: int | None = None) -> None:
    """Ragged batch over partial waves in one persistent launch.  ``wave_array`` from make_wave_array;
    ``workspace`` a CUDA uint8 tensor of at least pstgf_rmat_batch_workspace_bytes bytes (256-byte aligned)."""
    lib = load()
    n = len(wave_array) if n_waves is None else n_waves
    with torch.cuda.device(workspace.device):
        _check(lib.pstgf_rmat_form_batch(wave_array, n, workspace.data_ptr(), workspace.numel() * workspace.element_size(),
                                         _stream_ptr(stream)))


def pstgf_rmat_form_batch_host(host_waves: Sequence[tuple], max_chunk_bytes: int = 0, stream=None) -> None:
    """End-to-end call over HOST tensors (pinned recommended): (W, E_k, energies, a, R_out[, w_layout[, diag_add]])
    per wave, all CPU float64 contiguous tensors; R_out is filled on return (the call synchronises)."""
    lib = load()
    arr = (pstgf_wave_t * len(host_waves))()
    for p, wv in enumerate(host_waves):
        W, E_k, energies, a, R_out = wv[:5]
        layout = int(wv[5]) if len(wv) > 5 else PSTGF_W_POLE_CONTIGUOUS
        diag_add = wv[6] if len(wv) > 6 else None
        for t, nm in ((W, "W"), (E_k, "E_k"), (energies, "energies"), (R_out, "R_out"), (diag_add, "diag_add")):
            if t is not None and (t.dtype != torch.float64 or t.is_cuda or not t.is_contiguous()):
                raise TypeError(f"{nm} must be a contiguous CPU float64 tensor")
        n_chan, n_poles, ldw = _w_dims(W, layout)
        arr[p] = pstgf_wave_t(n_chan, n_poles, int(energies.shape[0]), layout, ldw, float(a), W.data_ptr(), E_k.data_ptr(),
                              energies.data_ptr(), R_out.data_ptr(), diag_add.data_ptr() if diag_add is not None else None)
    _check(lib.pstgf_rmat_form_batch_host(arr, len(host_waves), int(max_chunk_bytes), _stream_ptr(stream)))


def pstgf_debug_set_tail_policy(policy: int) -> None:
    """Thread-local scheduling knob: PSTGF_TAIL_AUTO / PSTGF_TAIL_NONE / PSTGF_TAIL_ALL (results are bitwise the same)."""
    _check(load().pstgf_debug_set_tail_policy(int(policy)))


def pstgf_debug_set_slab_policy(policy: int) -> None:
    """Thread-local: how the n_E mod 8 energies are cut (PSTGF_SLAB_AUTO / _NONE / _T32 / _T64 / _T128); same bits."""
    _check(load().pstgf_debug_set_slab_policy(int(policy)))


def pstgf_debug_set_pair_policy(policy: int) -> None:
    """Thread-local: which waves take the GEMM-over-channel-pairs form (PSTGF_PAIRS_AUTO / _NONE / _ALWAYS)."""
    _check(load().pstgf_debug_set_pair_policy(int(policy)))


def pstgf_debug_set_small_policy(policy: int) -> None:
    """Thread-local: whether a tiny pair-form wave takes the one-launch kernel (PSTGF_SMALL_AUTO / _NONE / _ALWAYS); same bits."""
    _check(load().pstgf_debug_set_small_policy(int(policy)))


def pstgf_debug_set_host_pipeline(mode: int) -> None:
    """Thread-local: PSTGF_HOST_PIPELINE_AUTO (signalled single launch) or PSTGF_HOST_PIPELINE_CHUNKED (one launch per piece)."""
    _check(load().pstgf_debug_set_host_pipeline(int(mode)))


def pstgf_debug_set_upload_timeout_ms(ms: int) -> None:
    _check(load().pstgf_debug_set_upload_timeout_ms(int(ms)))


def pstgf_debug_stall_upload(on: bool) -> None:
    _check(load().pstgf_debug_stall_upload(1 if on else 0))


def pstgf_mesh_from_zscaled(e_scaled, z: float):
    """E = z^2 * E_scaled for a HOST float64 array (numpy or CPU tensor): PAPER.md:431, :503."""
    import numpy as np
    src = np.ascontiguousarray(e_scaled.numpy() if isinstance(e_scaled, torch.Tensor) else e_scaled, dtype=np.float64)
    out = np.empty_like(src)
    _check(load().pstgf_mesh_from_zscaled(src.ctypes.data, src.size, float(z), out.ctypes.data))
    return out


def pstgf_rmat_finalize() -> None:
    """Free everything the library keeps between calls (it may be used again afterwards)."""
    _check(load().pstgf_rmat_finalize())


def pstgf_last_launch_count() -> int:
    return int(load().pstgf_last_launch_count())


def pstgf_version() -> int:
    return int(load().pstgf_version())


def pstgf_status_string(status: int) -> str:
    return load().pstgf_status_string(int(status)).decode()
