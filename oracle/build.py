"""Compile the CPU oracle (test infrastructure) into oracle/libbh_oracle.so with g++.

-ffp-contract=off keeps every floating-point operation of bh_oracle.cpp a single IEEE operation
(no fused multiply-add unless fmaf() is written), which the bit-exact steps rely on.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bh_oracle.cpp")
LIB = os.path.join(HERE, "libbh_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-shared", "-fPIC", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
