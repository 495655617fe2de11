"""Builds the C-ABI CUDA library (libggt.so) in-tree with nvcc for sm_100a.

nvcc cross-compiles without a GPU.  Flags that matter for correctness: --fmad=false (no silent FMA
contraction: every fused multiply-add in the kernels is an explicit fmaf, P14), default
-prec-div / -prec-sqrt / no -ftz (IEEE), -Xcompiler -ffp-contract=off for the host-side camera algebra.
Each source is compiled to an object file in its own nvcc process (in parallel); ggt_integrate.cu, whose
kernel instantiations dominate the compile time, eight times, once per storage / mode / fusion variant.
"""
from __future__ import annotations

import os
import subprocess
import sys
import tempfile
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libggt.so")
# (source, extra defines)
UNITS = [("ggt_api.cu", []), ("ggt_refine.cu", []), ("ggt_weight.cu", []), ("ggt_extract.cu", []),
         ("ggt_raymarch.cu", []), ("ggt_temporal.cu", []), ("ggt_features.cu", []), ("ggt_splat.cu", [])] + \
        [("ggt_integrate.cu", ["-DGGT_INTEGRATE_VARIANT=%d" % v]) for v in range(8)]
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "--fmad=false", "-std=c++17",
              "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math"]


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
    with tempfile.TemporaryDirectory(prefix="ggt_build_") as tmpdir:
        def compile_unit(i):
            src, defs = UNITS[i]
            obj = os.path.join(tmpdir, "u%d.o" % i)
            cmd = [nvcc] + NVCC_FLAGS + defs + os.environ.get("GGT_EXTRA_NVCC_FLAGS", "").split() + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, os.path.join(CSRC, src)]
            r = subprocess.run(cmd, capture_output=True, text=True)
            if verbose or r.returncode != 0:
                sys.stderr.write(r.stdout + r.stderr)
            if r.returncode != 0:
                raise subprocess.CalledProcessError(r.returncode, cmd)
            return obj
        with ThreadPoolExecutor(max_workers=min(len(UNITS), os.cpu_count() or 4)) as ex:
            objs = list(ex.map(compile_unit, range(len(UNITS))))
        tmp = LIB + ".tmp%d" % os.getpid()
        subprocess.check_call([nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-shared", "-cudart", "shared", "-o", tmp] + objs)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
