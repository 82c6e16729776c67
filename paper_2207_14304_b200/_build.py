"""Build libargus.so (the C-ABI library, include/argus.h) in-tree with nvcc for sm_100a."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libargus.so")
SOURCES = ["argus_api.cu"]
HEADERS = ["common.cuh", "plan.cuh", "plan_block.cuh", "resample.cuh", "resample_fast.cuh", "resample_unit.cuh", "segments.cuh", "background.cuh", "subtract.cuh", os.path.join("..", "..", "include", "argus.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "--shared", "-Xcompiler", "-fPIC"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


DEBUG_LIB = os.path.join(HERE, "libargus_debug.so")


def build(force: bool = False, verbose: bool = False, debug_bounds: bool = False) -> str:
    """Compile if sources are newer than the library.  Raises if nvcc is missing or fails.
    debug_bounds: the ARGUS_DEBUG_BOUNDS build (every shared-memory gather checked against its staged box) into
    libargus_debug.so; the product library is not touched."""
    if debug_bounds:
        return _compile(DEBUG_LIB, ["-DARGUS_DEBUG_BOUNDS"], verbose)
    if not force and not _stale():
        return LIB
    return _compile(LIB, [], verbose)


def _compile(out: str, defines, verbose: bool) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = "nvcc"
    tmp = out + ".tmp.%d" % os.getpid()
    extra = os.environ.get("ARGUS_NVCC_EXTRA", "").split()   # tuning macros for experiments
    cmd = [nvcc] + NVCC_FLAGS + list(defines) + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(tmp, out)
    return out


if __name__ == "__main__":
    print(build(force=True, verbose=True))
