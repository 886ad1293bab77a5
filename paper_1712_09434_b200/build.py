"""Builds ``libtpc_tracker.so`` (the C ABI of include/tpc_tracker.h) in-tree for sm_100a.

    python -m paper_1712_09434_b200.build [--force] [--verbose]

Flags that matter for parity (docs/ARITH_SPEC.md section 0): ``-fmad=false`` (no FMA
contraction), IEEE division and square root, denormals kept.
"""
from __future__ import annotations

import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
SRC = os.path.join(CSRC, "tpc_tracker.cu")
LIB = os.path.join(HERE, "libtpc_tracker.so")
NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
FLAGS = [
    "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-std=c++17", "-lineinfo",
    "-fmad=false", "-prec-div=true", "-prec-sqrt=true", "-ftz=false",
    "--shared", "-Xcompiler", "-fPIC,-ffp-contract=off,-fno-fast-math", "-cudart", "shared",
]


def _sources():
    inc = os.path.join(os.path.dirname(HERE), "include", "tpc_tracker.h")
    return [SRC, inc, *glob.glob(os.path.join(CSRC, "*.cuh"))]


def build(force: bool = False, verbose: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(
            os.path.getmtime(LIB) >= os.path.getmtime(s) for s in _sources()):
        return LIB
    cmd = [NVCC, *FLAGS, *(["-Xptxas", "-v"] if verbose else []), SRC, "-o", LIB]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv, verbose="--verbose" in sys.argv))
