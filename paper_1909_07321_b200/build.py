"""In-tree nvcc build of libpstgf_rmat.so (the product) and libpstgf_probe.so (the FP64 throughput probe bench.py
uses) for sm_100a (no JIT cache: the .so files travel with the tree)."""
from __future__ import annotations

import hashlib
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libpstgf_rmat.so")
SOURCES = [os.path.join(CSRC, "pstgf_rmat.cu"), os.path.join(CSRC, "rmat_launch.cu"), os.path.join(CSRC, "rmat_small.cu"), os.path.join(CSRC, "rmat_sliced.cu")]
HEADERS = [os.path.join(CSRC, "rmat_common.h"), os.path.join(CSRC, "rmat_kernel.cuh"), os.path.join(CSRC, "rmat_aux.cuh"), os.path.join(CSRC, "rmat_launch.h"),
           os.path.join(os.path.dirname(_HERE), "include", "pstgf_rmat.h")]
# translation units of libpstgf_rmat.so: (source, extra flags).  The persistent kernel is compiled once per item
# family set (csrc/rmat_launch.h), each in its own unit so that the units build side by side.
UNITS = [(SOURCES[0], []), (SOURCES[1], ["-DPSTGF_FAM=0"]), (SOURCES[1], ["-DPSTGF_FAM=1"]), (SOURCES[1], ["-DPSTGF_FAM=2"]),
         (SOURCES[2], []), (SOURCES[3], [])]
PROBE_LIB = os.path.join(_HERE, "libpstgf_probe.so")
PROBE_SOURCES = [os.path.join(_HERE, "measure", "fp64_probe.cu"), os.path.join(_HERE, "measure", "i8_probe.cu"),
                 os.path.join(_HERE, "measure", "l2_probe.cu")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def nvcc_path() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libpstgf_rmat.so cannot be built")


def _source_hash(deps: list[str]) -> str:
    h = hashlib.sha256(" ".join(NVCC_FLAGS).encode())
    for f in deps:
        with open(f, "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()


def _stale(lib: str, deps: list[str]) -> bool:
    """A library is current when the hash of its sources (recorded beside it at build time) matches: file times
    do not survive a copy of the tree to another machine, contents do."""
    stamp = lib + ".srchash"
    if not os.path.exists(lib) or not os.path.exists(stamp):
        return True
    with open(stamp) as fh:
        return fh.read().strip() != _source_hash(deps)


def is_stale() -> bool:
    """True when libpstgf_rmat.so is missing or was built from other sources than the ones in the tree."""
    return _stale(LIB, SOURCES + HEADERS)


def _compile(lib: str, units: list[tuple[str, list[str]]], deps: list[str], verbose: bool) -> None:
    """Compile every unit to an object (side by side), link them into `lib`, record the hash of the sources."""
    from concurrent.futures import ThreadPoolExecutor
    tmp = lib + f".tmp{os.getpid()}"
    digest = _source_hash(deps)
    nvcc = nvcc_path()
    objs = [f"{tmp}.{i}.o" for i in range(len(units))]

    def one(i: int) -> None:
        src, extra = units[i]
        subprocess.run([nvcc, *NVCC_FLAGS, *(["-Xptxas", "-v"] if verbose else []), *extra, "-c", src, "-o", objs[i]], check=True)

    try:
        with ThreadPoolExecutor(max_workers=min(len(units), os.cpu_count() or 1)) as pool:
            list(pool.map(one, range(len(units))))
        subprocess.run([nvcc, *NVCC_FLAGS, "-shared", *objs, "-o", tmp], check=True)
        os.replace(tmp, lib)
    finally:
        for o in objs + [tmp]:
            if os.path.exists(o):
                os.remove(o)
    with open(lib + ".srchash", "w") as fh:
        fh.write(digest + "\n")


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile csrc/ into libpstgf_rmat.so (and measure/ into libpstgf_probe.so) if missing or older than the sources."""
    if force or is_stale():
        _compile(LIB, UNITS, SOURCES + HEADERS, verbose)
    if force or _stale(PROBE_LIB, PROBE_SOURCES):
        _compile(PROBE_LIB, [(src, []) for src in PROBE_SOURCES], PROBE_SOURCES, verbose)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
