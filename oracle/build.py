"""Compile the CPU oracle ``oracle/mro.c`` into ``oracle/libmro.so`` with gcc (test infrastructure only).

``-O2``, no fast-math, ``-ffp-contract=off`` so that the oracle evaluates exactly the operations written in the
source (no fused multiply-adds), OpenMP only so that the timing harness can use the host cores.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mro.c")
LIB = os.path.join(HERE, "libmro.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-std=c99", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
