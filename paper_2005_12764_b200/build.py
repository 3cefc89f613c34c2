"""Build step: compile the CUDA kernels and the C-ABI into paper_2005_12764_b200/liblb_b200.so.

nvcc cross-compiles for sm_100a without a GPU.  Run as `python -m paper_2005_12764_b200.build`
or through __graft_entry__.build().
"""
from __future__ import annotations

import os
import shutil
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "liblb_b200.so")
SOURCES = ["lb_api.cu"]
HEADERS = ["lb_kernels.cuh", "lb_lattice.cuh", os.path.join("..", "..", "include", "lb.h")]

NVCC_FLAGS = ["-std=c++17", "-O3", "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo",
              "-Xcompiler", "-fPIC", "-shared"]


def _nvcc():
    for cand in (os.environ.get("NVCC"), shutil.which("nvcc"), "/usr/local/cuda/bin/nvcc"):
        if cand and os.path.exists(cand):
            return cand
    raise RuntimeError("nvcc not found; cannot build the CUDA extension")


SUBSET_STAMP = LIB + ".subset"     # present beside a library that was built with LB_BUILD_SUBSET=1


def _subset():
    return os.environ.get("LB_BUILD_SUBSET") == "1"


def stale():
    if not os.path.exists(LIB):
        return True
    if os.path.exists(SUBSET_STAMP) != _subset():   # a developer build never stands in for the full one
        return True
    t = os.path.getmtime(LIB)
    deps = [os.path.join(CSRC, s) for s in SOURCES + HEADERS]
    return any(os.path.getmtime(d) > t for d in deps)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or stale():
        tmp = LIB + ".tmp%d" % os.getpid()
        # LB_BUILD_SUBSET=1: developer builds that compile a fifth of the k_fused instantiations (lb_api.cu)
        subset = ["-DLB_BUILD_SUBSET"] if _subset() else []
        cmd = [_nvcc()] + NVCC_FLAGS + subset + (["-Xptxas", "-v"] if verbose else []) + \
              ["-o", tmp] + [os.path.join(CSRC, s) for s in SOURCES]
        subprocess.check_call(cmd)
        os.replace(tmp, LIB)
        if _subset():
            open(SUBSET_STAMP, "w").close()
        elif os.path.exists(SUBSET_STAMP):
            os.remove(SUBSET_STAMP)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
