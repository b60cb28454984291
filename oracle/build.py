"""Compile the CPU oracle (test infrastructure) into oracle/libazint_oracle.so with gcc.

Usage: python oracle/build.py            (also called by __graft_entry__.build()).
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "azint_oracle.c")
LIB = os.path.join(HERE, "libazint_oracle.so")
# -ffp-contract=off: no fused multiply-add, so every operation rounds once as written
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-shared", "-fPIC", "-std=c99", "-Wall"]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    subprocess.check_call(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
