"""Builds libmoebius.so (host planner + sm_100a kernel) in-tree with nvcc.  No GPU needed."""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
LIB = os.path.join(HERE, "libmoebius.so")
SOURCES = ["moebius_plan.cpp", "moebius_policy.cpp", "moebius_cuda.cu", "moebius_arena.cu", "moebius_naive.cu", "moebius_static.cu"]
HEADERS = ["moebius_units.h", "moebius_host.h", os.path.join("..", "..", "include", "moebius.h")]


def _stale() -> bool:
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(CSRC, f)) > t for f in SOURCES + HEADERS)


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and not _stale():
        return LIB
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    cmd = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo", "-O3", "-std=c++17",
           "-shared", "-Xcompiler", "-fPIC,-fvisibility=hidden,-Wall", "-cudart", "static",
           "-o", LIB] + [os.path.join(CSRC, f) for f in SOURCES]
    extra = os.environ.get("MOEBIUS_NVCC_FLAGS", "").split()   # e.g. -DMOEBIUS_PIPE_STATS (profiling aid)
    cmd[1:1] = extra
    if verbose:
        cmd.insert(1, "-Xptxas=-v")
        print(" ".join(cmd))
    r = subprocess.run(cmd, capture_output=True, text=True)
    if r.returncode != 0:
        sys.stderr.write(r.stdout + r.stderr)
        raise RuntimeError("nvcc failed building libmoebius.so")
    if verbose:
        print(r.stdout + r.stderr)
    return LIB


if __name__ == "__main__":
    print(build(force=True, verbose=True))
