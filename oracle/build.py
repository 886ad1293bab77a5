"""Builds the CPU oracle shared library (test infrastructure, not the product).

    python -m oracle.build

Flags: -O2, no fast-math, no FMA contraction (docs/ARITH_SPEC.md section 0).

TPC_ORACLE_SANITIZE=1 builds (and loads) a second library with -fsanitize=address,undefined instead; run the CPU
suite on it with  LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)"
(the summary of such a run is kept in profiles/).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tpc_oracle.cpp")
LIB = os.path.join(HERE, "libtpc_oracle.so")
FLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall"]


def build(force: bool = False) -> str:
    lib, flags = LIB, FLAGS
    if os.environ.get("TPC_ORACLE_SANITIZE") == "1":
        lib = os.path.join(HERE, "libtpc_oracle_asan.so")
        flags = [*FLAGS, "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    if (not force and os.path.exists(lib)
            and os.path.getmtime(lib) >= os.path.getmtime(SRC)):
        return lib
    cmd = ["g++", *flags, SRC, "-o", lib]
    subprocess.run(cmd, check=True)
    return lib


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
