"""Compile oracle/asym_oracle.c into oracle/libasym_oracle.so (gcc, no CUDA)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "asym_oracle.c")
INC = os.path.join(HERE, "asym_substep.inc")
LIB = os.path.join(HERE, "libasym_oracle.so")
# -ffp-contract=off: no FMA contraction, every operation rounds as written.
CFLAGS = ["-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c11"]


def build(force: bool = False) -> str:
    newest = max(os.path.getmtime(SRC), os.path.getmtime(INC), os.path.getmtime(__file__))
    if force or not os.path.exists(LIB) or os.path.getmtime(LIB) < newest:
        tmp = LIB + f".tmp{os.getpid()}"
        subprocess.check_call(["gcc", *CFLAGS, SRC, "-o", tmp, "-lm"])
        os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
