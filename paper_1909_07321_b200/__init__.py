"""B200-native R-matrix formation (eq. 4 of arxiv 1909.07321).

``rmat``   ctypes binding over the C-ABI library ``libpstgf_rmat.so`` (include/pstgf_rmat.h)
``inputs`` seeded synthetic workloads (no method arithmetic)
``build``  in-tree nvcc build of the library

Importing the package does not load the CUDA library; ``rmat`` loads it on
first use and raises if it is missing (there is no CPU fallback).
"""
__all__ = ["rmat", "inputs", "build"]
