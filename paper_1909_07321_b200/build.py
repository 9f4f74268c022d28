"""In-tree nvcc build of libpstgf_rmat.so for sm_100a (no JIT cache: the .so travels with the tree)."""
from __future__ import annotations

import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpstgf_rmat.so")
SOURCES = [os.path.join(CSRC, "pstgf_rmat.cu"), os.path.join(CSRC, "fp64_probe.cu")]
HEADERS = [os.path.join(CSRC, "rmat_common.h"), os.path.join(CSRC, "rmat_kernel.cuh"),
           os.path.join(os.path.dirname(_HERE), "include", "pstgf_rmat.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpstgf_rmat.so cannot be built")


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(f) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ into libpstgf_rmat.so if it is missing or older than its sources."""
    if force or is_stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc_path(), *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *SOURCES, "-o", tmp]
        subprocess.run(cmd, check=True)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
