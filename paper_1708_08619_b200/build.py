"""Build libg3.so in-tree with nvcc for sm_100a (no JIT cache: the .so travels with the repo)."""
from __future__ import annotations

import glob
import os
import shutil
import subprocess

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libg3.so")
BENCH_LIB = os.path.join(_HERE, "libg3bench.so")      # measurement aid of bench.py (include/g3_bench.h)

NVCC_FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a",
    "-O3", "-std=c++17", "-lineinfo",
    "--fmad=false",                 # no silent FMA contraction: every fused op is written explicitly
    "-Xcompiler", "-fPIC,-O2,-Wall,-fvisibility=hidden",
    "-shared", "-cudart", "shared",
]


def _nvcc() -> str:
    for cand in (shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found: libg3 can only be built with the CUDA toolkit")


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def needs_build() -> bool:
    if not os.path.exists(LIB) or not os.path.exists(BENCH_LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = glob.glob(os.path.join(CSRC, "*")) + glob.glob(os.path.join(CSRC, "bench", "*")) + \
        glob.glob(os.path.join(_HERE, "..", "include", "*.h"))
    return any(os.path.getmtime(d) > t for d in deps)


def bench_sources():
    return sorted(glob.glob(os.path.join(CSRC, "bench", "*.cu")))


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        extra = ["-Xptxas", "-v"] if verbose else []
        subprocess.run([_nvcc()] + NVCC_FLAGS + extra + sources() + ["-o", LIB], check=True)
        subprocess.run([_nvcc()] + NVCC_FLAGS + extra + bench_sources() + ["-o", BENCH_LIB], check=True)
    return LIB


if __name__ == "__main__":
    import sys
    print(build(force=True, verbose="-v" in sys.argv))
