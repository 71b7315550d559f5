"""Build the C-ABI library (csrc/ -> libinpc_raster.so, in-tree) for sm_100a with nvcc.

nvcc cross-compiles without a GPU.  No -use_fast_math: the canonical fp32 projection needs IEEE
division, and it is written with _rn intrinsics so the default -fmad=true cannot contract it.
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libinpc_raster.so")
SOURCES = ["inpc_raster.cu"]
HEADERS = ["common.cuh", "bin.cuh", "cellsort.cuh", "tile.cuh", "blend.cuh", "back.cuh", "big.cuh", "grad.cuh", "sh.cuh", "sampler.cuh", os.path.join("..", "..", "include", "inpc_raster.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def _nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    return "nvcc"


def needs_build() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS] + [os.path.abspath(__file__)]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or needs_build():
        cmd = [_nvcc()] + NVCC_FLAGS + os.environ.get("INPC_NVCC_EXTRA", "").split() + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
