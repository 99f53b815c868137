"""Build libmm.so (the C-ABI CUDA library) in-tree with nvcc for sm_100a.

    python -m paper_1908_04279_b200.build [--force] [--verbose]

One translation unit per kernel family, compiled in parallel into build/*.o (only the units whose sources changed),
then linked into libmm.so.
"""
from __future__ import annotations

import os
import re
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
OBJ = os.path.join(HERE, "build")
SO = os.path.join(HERE, "libmm.so")
MM_H = os.path.join(os.path.dirname(HERE), "include", "mm.h")
UNITS = ("mm_api", "mm_launch_tm", "mm_launch_coef", "mm_launch_stream_tile", "mm_launch_rk2", "mm_noalloc")
SOURCES = [os.path.join(CSRC, u + ".cu") for u in UNITS]
CFLAGS = ["-O3", "-std=c++17", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-Xcompiler", "-fPIC"]
LFLAGS = ["-shared", "-cudart", "static", "-gencode", "arch=compute_100a,code=sm_100a",
          "-Xlinker", "--version-script=" + os.path.join(CSRC, "libmm.map")]


def nvcc() -> str:
    for cand in (os.environ.get("NVCC"), "/usr/local/cuda/bin/nvcc", "nvcc"):
        if cand and (os.path.sep not in cand or os.path.exists(cand)):
            return cand
    raise RuntimeError("nvcc not found")


def _deps(path: str, seen: set[str] | None = None) -> set[str]:
    """The file and every local header it includes (transitively)."""
    seen = set() if seen is None else seen
    if path in seen or not os.path.exists(path):
        return seen
    seen.add(path)
    with open(path) as f:
        for inc in re.findall(r'^\s*#include\s+"([^"]+)"', f.read(), re.M):
            _deps(os.path.normpath(os.path.join(os.path.dirname(path), inc)), seen)
    return seen


def _stale(target: str, deps) -> bool:
    return not os.path.exists(target) or any(os.path.getmtime(d) > os.path.getmtime(target) for d in deps)


def up_to_date() -> bool:
    return not _stale(SO, set().union(*(_deps(s) for s in SOURCES)) | {os.path.abspath(__file__)})


def build(force: bool = False, verbose: bool = False) -> str:
    os.makedirs(OBJ, exist_ok=True)
    cc = nvcc()
    jobs = []
    for unit, src in zip(UNITS, SOURCES):
        obj = os.path.join(OBJ, unit + ".o")
        if force or _stale(obj, _deps(src) | {os.path.abspath(__file__)}):
            jobs.append([cc] + CFLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", obj, src])
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 1)) as ex:
            for rc, cmd in zip(ex.map(subprocess.call, jobs), jobs):
                if rc != 0:
                    raise subprocess.CalledProcessError(rc, cmd)
    objs = [os.path.join(OBJ, u + ".o") for u in UNITS]
    if jobs or _stale(SO, objs + [os.path.join(CSRC, "libmm.map")]):
        subprocess.check_call([cc] + LFLAGS + ["-o", SO] + objs)
    return SO


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
