"""Build libtwk.so in-tree with nvcc for sm_100a (no torch extension machinery: the boundary is a plain C ABI)."""
from __future__ import annotations

import hashlib
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libtwk.so")
LIB_DEBUG = os.path.join(HERE, "libtwk_debug.so")   # same sources with -DTWK_DEBUG: invariant counters (twk_debug_counters)
SOURCES = ["twk_api.cu"]
HEADERS = ["twk_device.cuh", "twk_contour.cuh", "twk_kernels.cuh", "twk_adaptive.cuh", "twk_refine1.cuh", "twk_stage1.cuh"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-Xcompiler", "-fPIC",
              "-shared", "-cudart", "shared"]


def _stale(lib: str = LIB) -> bool:
    if not os.path.exists(lib):
        return True
    t = os.path.getmtime(lib)
    deps = [os.path.join(CSRC, f) for f in SOURCES + HEADERS] + [os.path.join(HERE, "..", "include", "twk.h")]
    return any(os.path.getmtime(d) > t for d in deps)


def source_hash() -> str:
    """Hash of everything the library is compiled from (CUDA sources, the C header, the compiler flags).  It is compiled
    into the library (twk_version() ends in "src:<hash>") and keys the ncu instruction counts in profiles/ that
    bench.py's roofline uses: counts measured on other sources are refused."""
    h = hashlib.sha256()
    for f in sorted(SOURCES + HEADERS):
        h.update(open(os.path.join(CSRC, f), "rb").read())
    h.update(open(os.path.join(HERE, "..", "include", "twk.h"), "rb").read())
    h.update(" ".join(NVCC_FLAGS).encode())
    return h.hexdigest()[:12]


def build(force: bool = False, verbose: bool = False, debug: bool = False) -> str:
    lib = LIB_DEBUG if debug else LIB
    if not force and not _stale(lib):
        return lib
    nvcc = os.environ.get("NVCC", "nvcc")
    tmp = lib + f".tmp{os.getpid()}"
    cmd = ([nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + (["-DTWK_DEBUG"] if debug else [])
           + [f'-DTWK_SOURCE_HASH="{source_hash()}"', "-o", tmp] + [os.path.join(CSRC, f) for f in SOURCES])
    subprocess.run(cmd, check=True)
    os.replace(tmp, lib)
    return lib


if __name__ == "__main__":
    print(build(force=True, verbose=True))
