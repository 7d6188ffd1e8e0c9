"""Builds oracle/libpimd_oracle.so from pimd_oracle.c with gcc (TEST INFRASTRUCTURE).

`-ffp-contract=off` is required: the neighbour predicate must not
be contracted into fused multiply-adds.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pimd_oracle.c")
LIB = os.path.join(HERE, "libpimd_oracle.so")
FLAGS = ["-O3", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11", "-Wall", "-Wno-unknown-pragmas"]


def build(force: bool = False) -> str:
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < os.path.getmtime(SRC):
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
