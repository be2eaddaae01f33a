"""Compile oracle/sr_oracle.c into oracle/libsr_oracle.so with gcc (FP64, OpenMP).

Building the checker is not using it: __graft_entry__.build() calls this too.
No -ffast-math and no -march flags: the oracle's arithmetic is plain IEEE double.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sr_oracle.c")
LIB = os.path.join(HERE, "libsr_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-ffp-contract=off",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
