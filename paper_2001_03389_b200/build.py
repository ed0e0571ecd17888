"""Build librfim.so (nvcc, sm_100a) and the synthetic-input generator twins, in-tree.

    python -m paper_2001_03389_b200.build [--force] [-v]

Every `csrc/*.cu` is one translation unit (one per kernel family plus the host plumbing and the C ABI); they are
compiled in parallel into `csrc/obj/` and linked into `librfim.so`.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
OBJ = os.path.join(CSRC, "obj")
LIB = os.path.join(_HERE, "librfim.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC"]


def _stale(target: str, sources) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def _includes(unit: str) -> list:
    """Headers of csrc/ a unit includes, transitively (by scanning `#include "..."` lines)."""
    seen, todo = set(), [unit]
    while todo:
        f = todo.pop()
        for line in open(f, encoding="utf-8"):
            line = line.strip()
            if line.startswith('#include "'):
                h = os.path.normpath(os.path.join(os.path.dirname(f), line.split('"')[1]))
                if h not in seen and os.path.exists(h):
                    seen.add(h)
                    todo.append(h)
    return sorted(seen)


def build_librfim(force: bool = False, verbose: bool = False) -> str:
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    os.makedirs(OBJ, exist_ok=True)
    units = sorted(glob.glob(os.path.join(CSRC, "*.cu")))
    jobs = []
    for u in units:
        o = os.path.join(OBJ, os.path.basename(u)[:-3] + ".o")
        if force or _stale(o, [u] + _includes(u)):
            jobs.append([nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + ["-c", "-o", o, u])
    if jobs:
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            for rc, cmd in zip(ex.map(lambda c: subprocess.run(c).returncode, jobs), jobs):
                if rc != 0:
                    raise subprocess.CalledProcessError(rc, cmd)
    objs = [os.path.join(OBJ, os.path.basename(u)[:-3] + ".o") for u in units]
    if jobs or _stale(LIB, objs):
        subprocess.check_call([nvcc, "-shared", "-o", LIB] + objs)
    return LIB


def build_all(force: bool = False, verbose: bool = False) -> None:
    from . import synth
    build_librfim(force, verbose)
    synth.build_host(force)
    synth.build_cuda(force)


if __name__ == "__main__":
    build_all(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
