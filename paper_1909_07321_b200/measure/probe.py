"""ctypes binding of libpstgf_probe.so: the register-resident FP64 throughput probe that fixes the roofline
denominator of the contraction (MEASURED_PEAKS.json has no FP64 entry).  Not part of the product library."""
from __future__ import annotations

import ctypes
import os

import torch

from .. import build as _build

_lib = None


def load():
    global _lib
    if _lib is None:
        if not os.path.exists(_build.PROBE_LIB):
            raise RuntimeError(f"{_build.PROBE_LIB} is missing: run `python -m paper_1909_07321_b200.build`")
        lib = ctypes.CDLL(_build.PROBE_LIB)
        lib.pstgf_fp64_probe.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p,
                                         ctypes.POINTER(ctypes.c_double), ctypes.c_void_p]
        lib.pstgf_fp64_probe.restype = ctypes.c_int
        lib.pstgf_i8_probe.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
        lib.pstgf_i8_probe.restype = ctypes.c_double
        _lib = lib
    return _lib


def fp64_probe(kind: int, iters: int, blocks: int, threads: int, sink: torch.Tensor, stream=None) -> float:
    """Enqueue the probe (0 DMMA.8x8x4, 1 DFMA, 2 both on alternating warps); returns the FLOPs of the launch."""
    lib = load()
    if sink.dtype != torch.float64 or not sink.is_cuda or sink.numel() < blocks * threads:
        raise ValueError("sink must be a CUDA float64 tensor of at least blocks*threads elements")
    if stream is None:
        stream = torch.cuda.current_stream()
    flop = ctypes.c_double(0.0)
    with torch.cuda.device(sink.device):
        rc = lib.pstgf_fp64_probe(int(kind), int(iters), int(blocks), int(threads), sink.data_ptr(), ctypes.byref(flop),
                                  int(stream.cuda_stream))
    if rc != 0:
        raise RuntimeError(f"pstgf_fp64_probe failed (rc={rc})")
    return float(flop.value)


def i8_probe(iters: int, blocks: int, sink: torch.Tensor, stream=None) -> float:
    """Enqueue the INT8 tensor-pipe probe (tcgen05.mma kind::i8, 128 x 256 x 32, operands resident in shared memory, one
    CTA per SM); returns the INT8 operations of the launch.  Context for DESIGN.md 11.6, not used by the product."""
    lib = load()
    if sink.dtype != torch.int32 or not sink.is_cuda or sink.numel() < blocks:
        raise ValueError("sink must be a CUDA int32 tensor of at least `blocks` elements")
    if stream is None:
        stream = torch.cuda.current_stream()
    with torch.cuda.device(sink.device):
        ops = float(lib.pstgf_i8_probe(int(iters), int(blocks), sink.data_ptr(), int(stream.cuda_stream)))
    if ops < 0:
        raise RuntimeError("pstgf_i8_probe failed to launch")
    return ops
