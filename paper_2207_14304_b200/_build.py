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


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile if sources are newer than the library.  Raises if nvcc is missing or fails."""
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(nvcc):
        nvcc = "nvcc"
    tmp = LIB + ".tmp.%d" % os.getpid()
    extra = os.environ.get("ARGUS_NVCC_EXTRA", "").split()   # e.g. -DARGUS_DEBUG_BOUNDS (tests), tuning macros
    cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
    subprocess.run(cmd, check=True, cwd=CSRC)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
