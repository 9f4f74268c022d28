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
        lib.pstgf_l2_probe.argtypes = [ctypes.c_int] * 9 + [ctypes.c_void_p, ctypes.c_ulonglong, ctypes.c_void_p, ctypes.c_void_p]
        lib.pstgf_l2_probe.restype = ctypes.c_double
        _lib = lib
    return _lib


L2_PROBE_PITCH = 81920      # bytes per row of the probe's source array (a row of config 5's W)


def l2_probe(mode: int, inner_bytes: int, box_rows: int, boxes_per_stage: int, lanes: int, stages: int, cluster: int,
             iters: int, n_ctas: int, src: torch.Tensor, status: torch.Tensor, stream=None) -> float:
    """Enqueue the L2 -> shared-memory load-rate probe (l2_probe.cu: persistent CTAs streaming an L2-resident array
    with TMA boxes or 1-D bulk copies and doing nothing with them); returns the bytes delivered into shared memory.
    ``src``: CUDA uint8 tensor, a multiple of L2_PROBE_PITCH bytes; ``status``: zeroed CUDA int32 word, non-zero
    afterwards if a wait timed out."""
    lib = load()
    if src.dtype != torch.uint8 or not src.is_cuda or status.dtype != torch.int32 or not status.is_cuda:
        raise ValueError("src must be a CUDA uint8 tensor and status a CUDA int32 tensor")
    if stream is None:
        stream = torch.cuda.current_stream()
    with torch.cuda.device(src.device):
        b = float(lib.pstgf_l2_probe(int(mode), int(inner_bytes), int(box_rows), int(boxes_per_stage), int(lanes), int(stages),
                                     int(cluster), int(iters), int(n_ctas), src.data_ptr(), src.numel(), status.data_ptr(),
                                     int(stream.cuda_stream)))
    if b < 0:
        raise RuntimeError(f"pstgf_l2_probe refused its arguments or failed to launch (rc={b})")
    return b


# (label, mode, inner_bytes, box_rows, boxes_per_stage, lanes, stages, cluster): what bench.py --probe-l2 sweeps
L2_PROBE_SWEEP = [
    # the library's box (160 B x 32 rows = 5 KB), 160 KB in flight, by issuing lanes
    ("tma2d 160B x32 rows, 8 boxes/stage, 4 stages, 1 lane", 0, 160, 32, 8, 1, 4, 1),
    ("tma2d 160B x32 rows, 8 boxes/stage, 4 stages, 4 lanes", 0, 160, 32, 8, 4, 4, 1),
    ("tma2d 160B x32 rows, 8 boxes/stage, 4 stages, 8 lanes", 0, 160, 32, 8, 8, 4, 1),
    ("tma2d 160B x8 rows, 32 boxes/stage, 4 stages, 32 lanes", 0, 160, 8, 32, 32, 4, 1),
    # inner extent of the box at about 5 KB per box
    ("tma2d 64B x80 rows, 8 boxes/stage, 4 stages, 8 lanes", 0, 64, 80, 8, 8, 4, 1),
    ("tma2d 256B x20 rows, 8 boxes/stage, 4 stages, 8 lanes", 0, 256, 20, 8, 8, 4, 1),
    ("tma2d 512B x10 rows, 8 boxes/stage, 4 stages, 8 lanes", 0, 512, 10, 8, 8, 4, 1),
    ("tma2d 2048B x4 rows, 5 boxes/stage, 4 stages, 5 lanes", 0, 2048, 4, 5, 5, 4, 1),
    # contiguous bulk copies
    ("bulk1d 5120 B, 8 boxes/stage, 4 stages, 8 lanes", 1, 5120, 1, 8, 8, 4, 1),
    ("bulk1d 8192 B, 5 boxes/stage, 4 stages, 5 lanes", 1, 8192, 1, 5, 5, 4, 1),
    ("bulk1d 16384 B, 2 boxes/stage, 5 stages, 2 lanes", 1, 16384, 1, 2, 2, 5, 1),
    # bytes in flight: ring depth at 10 KB per stage
    ("tma2d 160B x32 rows, 2 boxes/stage, 2 stages (20 KB in flight)", 0, 160, 32, 2, 2, 2, 1),
    ("tma2d 160B x32 rows, 2 boxes/stage, 4 stages (40 KB)", 0, 160, 32, 2, 2, 4, 1),
    ("tma2d 160B x32 rows, 2 boxes/stage, 8 stages (80 KB)", 0, 160, 32, 2, 2, 8, 1),
    ("tma2d 160B x32 rows, 2 boxes/stage, 16 stages (160 KB)", 0, 160, 32, 2, 2, 16, 1),
    # multicast: each box crosses the fabric once per cluster
    ("tma2d 160B x32 rows, 8 boxes/stage, 4 stages, multicast over 2 CTAs", 0, 160, 32, 8, 4, 4, 2),
    ("tma2d 160B x32 rows, 8 boxes/stage, 4 stages, multicast over 4 CTAs", 0, 160, 32, 8, 2, 4, 4),
    ("tma2d 512B x10 rows, 8 boxes/stage, 4 stages, multicast over 4 CTAs", 0, 512, 10, 8, 2, 4, 4),
]


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
