"""Compile the C oracle (test infrastructure) into oracle/libsldg_oracle.so with gcc.

Building the checker is not using it: __graft_entry__.build() calls this; the product path never
loads the result.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "sldg_oracle.c")
LIB = os.path.join(HERE, "libsldg_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    # -O2, no -ffast-math, no FMA contraction: the oracle is plain IEEE fp64 arithmetic as written.
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-D_GNU_SOURCE", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
