"""In-tree build of liblartpc.so (hand-written sm_100a CUDA kernels + the C-ABI of include/lartpc.h)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblartpc.so")
SOURCES = ["api.cu", "stages_segment.cu", "stage_current.cu", "stages_pixel.cu", "light.cu"]
HEADER = os.path.join(HERE, "..", "include", "lartpc.h")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC) if f.endswith((".cu", ".cuh"))] + [HEADER]
    return any(os.path.getmtime(f) > t for f in deps)


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    """Compile with nvcc for sm_100a (cross-compiles without a GPU).  `extra`: more nvcc flags, e.g.
    ("-DLARTPC_DEBUG_CLOCKS",) for a measurement build -- an explicit argument, never the environment."""
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + list(extra) + (["-Xptxas", "-v"] if verbose else []) + \
              [os.path.join(CSRC, f) for f in SOURCES] + ["-o", LIB]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
