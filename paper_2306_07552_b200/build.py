"""Build libgx.so (the C-ABI library of include/gx.h) in-tree with nvcc for sm_100a.

    python -m paper_2306_07552_b200.build [--force]

nvcc cross-compiles without a GPU.  -fmad=false: only the fmaf() calls written in the kernels fuse, which
is what makes the vertex stage bit-exact against DESIGN.md section 3.
"""
from __future__ import annotations

import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "libgx.so")
SOURCES = ["gx_api.cu"]
DEPS = ["gx_api.cu", "gx_math.cuh", "gx_pipeline.cuh", "gx_fk.cuh", "gx_collide.cuh", "gx_types.h",
        os.path.join("..", "..", "include", "gx.h")]
NVCC_FLAGS = ["-shared", "-Xcompiler", "-fPIC", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3",
              "-fmad=false", "-std=c++17", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.isabs(cand) and os.path.exists(cand) or not os.path.isabs(cand)):
            return cand
    return "nvcc"


def is_stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, d)) > t for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or is_stale():
        tmp = LIB + f".tmp{os.getpid()}"
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", tmp] + SOURCES
        subprocess.run(cmd, check=True, cwd=CSRC)
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
