"""Builds the C-ABI CUDA library (libggt.so) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  Flags that matter for correctness: --fmad=false (no silent FMA
contraction: every fused multiply-add in the kernels is an explicit fmaf, P14), default
-prec-div / -prec-sqrt / no -ftz (IEEE), -Xcompiler -ffp-contract=off for the host-side camera algebra.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libggt.so")
SOURCES = ["ggt_api.cu", "ggt_refine.cu", "ggt_weight.cu", "ggt_integrate.cu", "ggt_extract.cu", "ggt_raymarch.cu", "ggt_temporal.cu", "ggt_features.cu"]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math", "-shared", "-cudart", "shared"]


def stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, f) for f in os.listdir(CSRC)] + [os.path.join(HERE, "..", "include", "ggt.h"), __file__]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    tmp = LIB + ".tmp%d" % os.getpid()
    cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
