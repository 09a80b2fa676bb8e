"""Compile oracle/qr_oracle.c into oracle/libqr_oracle.so with gcc (test infrastructure only).

-ffp-contract=off: only the fmaf() calls written in the source fuse, so the fp32 decision
arithmetic has the operation order DESIGN.md fixes.  No -ffast-math, no -march flags (the
library is built on one box and may be loaded on another).
"""
from __future__ import annotations

import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "qr_oracle.c")
LIB = os.path.join(HERE, "libqr_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
