"""Build libarachne_attn.so in-tree with nvcc for sm_100a (cross-compiles without a GPU)."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(CSRC, "libarachne_attn.so")
SOURCES = ["arachne_attn.cu"]
HEADERS = ["sm100.cuh", "common.cuh", "rawtile.cuh", "normrope.cuh", "prep.cuh", "fwd.cuh", "bwd_fused.cuh", os.path.join("..", "..", "include", "arachne_attn.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if force or _stale():
        nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
        cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
               "-shared", "-Xcompiler", "-fPIC", "--use_fast_math", "-o", LIB] + [os.path.join(CSRC, s) for s in SOURCES]
        if verbose:
            cmd.insert(1, "-Xptxas=-v")
        subprocess.run(cmd, check=True)
    return LIB


SCHED_LIB = os.path.join(CSRC, "libarachne_sched.so")
SCHED_SRC = [os.path.join(CSRC, "cascade_sched.cpp"), os.path.join(HERE, "..", "include", "arachne_sched.h")]


def build_sched(force: bool = False) -> str:
    """libarachne_sched.so: the host-only cascade scheduler (include/arachne_sched.h).  -ffp-contract=off: the makespans
    are compared value for value with the Python oracle."""
    if force or not os.path.exists(SCHED_LIB) or any(os.path.getmtime(f) > os.path.getmtime(SCHED_LIB) for f in SCHED_SRC):
        subprocess.run(["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-o", SCHED_LIB,
                        SCHED_SRC[0]], check=True)
    return SCHED_LIB


if __name__ == "__main__":
    build_sched(force="--force" in sys.argv)
    print(build(force="--force" in sys.argv, verbose="-v" in sys.argv))
