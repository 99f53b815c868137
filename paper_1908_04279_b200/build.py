"""Build libmm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1908_04279_b200.build [--force] [--verbose]
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SO = os.path.join(HERE, "libmm.so")
SOURCES = [os.path.join(CSRC, "mm_api.cu")]
DEPS = SOURCES + [os.path.join(CSRC, f) for f in ("mm_common.cuh", "mm_ptx.cuh", "mm_generic.cuh", "mm_stream.cuh", "mm_tile.cuh", "mm_coef.cuh", "mm_rk2.cuh", "mm_local.cuh", "mm_spread.cuh", "mm_free.cuh")] + [
    os.path.join(os.path.dirname(HERE), "include", "mm.h")]
NVCC_FLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared", "-cudart", "static"]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def up_to_date() -> bool:
    return os.path.exists(SO) and all(os.path.getmtime(SO) >= os.path.getmtime(d) for d in DEPS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or not up_to_date():
        cmd = [nvcc()] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-o", SO] + SOURCES
        subprocess.check_call(cmd)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
