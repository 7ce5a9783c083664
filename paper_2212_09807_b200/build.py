"""In-tree build of liblartpc.so (hand-written sm_100a CUDA kernels + the C-ABI of include/lartpc.h)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblartpc.so")
SOURCES = ["api.cu", "stages_segment.cu", "stage_current.cu", "stages_pixel.cu"]
HEADERS = ["common.cuh", "scan.cuh", os.path.join("..", "..", "include", "lartpc.h")]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    """Compile with nvcc for sm_100a (cross-compiles without a GPU)."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        extra = os.environ.get("LARTPC_NVCC_EXTRA", "").split()       # e.g. -DLARTPC_DEBUG_CLOCKS (measurement builds)
        cmd = [nvcc] + NVCC_FLAGS + extra + (["-Xptxas", "-v"] if verbose else []) + \
              [os.path.join(CSRC, f) for f in SOURCES] + ["-o", LIB]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
