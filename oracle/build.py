"""Compile the C part of the oracle (gcc, OpenMP) into oracle/_fdd_oracle_c.so.

Run as ``python -m oracle.build``; ``__graft_entry__.build()`` calls ``build()`` too.
Building the checker is not using it: nothing on the product path loads this library.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "fdd_oracle_c.c")
LIB = os.path.join(HERE, "_fdd_oracle_c.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-std=c11", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
