"""Builds the C-ABI CUDA library in-tree (libhashrender.so) for sm_100a with nvcc.  No JIT cache."""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(_HERE, "csrc", "hashrender.cu")
LIB = os.path.join(_HERE, "libhashrender.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17", "-shared",
              "-Xcompiler", "-fPIC", "--expt-relaxed-constexpr"]


def _newest_source() -> float:
    d = os.path.join(_HERE, "csrc")
    t = [os.path.getmtime(os.path.join(d, f)) for f in os.listdir(d)]
    t.append(os.path.getmtime(os.path.join(_HERE, "..", "include", "hashrender.h")))
    return max(t)


def build(force: bool = False, verbose: bool = False, extra=()) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= _newest_source():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    if not os.path.exists(os.path.join(_HERE, "csrc", "hr_kernels_tc.cuh")):
        extra = [*extra, "-DHR_NO_TC"]
    cmd = [nvcc, *NVCC_FLAGS, *extra, "-o", LIB, SRC]
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    build(force=True, verbose="-v" in sys.argv)
    print(LIB)
