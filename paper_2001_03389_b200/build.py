"""Build librfim.so (nvcc, sm_100a) and the synthetic-input generator twins, in-tree.

    python -m paper_2001_03389_b200.build [--force]
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

_HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(_HERE, "csrc")
LIB = os.path.join(_HERE, "librfim.so")
NVCC_FLAGS = ["-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
              "-Xcompiler", "-fPIC", "-shared"]


def _stale(target: str, sources) -> bool:
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build_librfim(force: bool = False, verbose: bool = False) -> str:
    sources = glob.glob(os.path.join(CSRC, "*.cu")) + glob.glob(os.path.join(CSRC, "*.cuh")) + [
        os.path.join(os.path.dirname(_HERE), "include", "rfim.h")]
    if force or _stale(LIB, sources):
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc] + NVCC_FLAGS + (["-Xptxas", "-v"] if verbose else []) + [
            "-o", LIB, os.path.join(CSRC, "rfim_api.cu")]
        subprocess.check_call(cmd)
    return LIB


def build_all(force: bool = False, verbose: bool = False) -> None:
    from . import synth
    build_librfim(force, verbose)
    synth.build_host(force)
    synth.build_cuda(force)


if __name__ == "__main__":
    build_all(force="--force" in sys.argv, verbose="-v" in sys.argv)
    print(LIB)
