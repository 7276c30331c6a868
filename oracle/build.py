"""Compile oracle/bh_oracle.c into oracle/libbh_oracle.so (gcc, -ffp-contract=off, OpenMP).

Test infrastructure: called by __graft_entry__.build() and by tests/conftest.py when the library
is missing.  No -march flags: the built library travels to the GPU box, whose CPU may differ.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "bh_oracle.c")
LIB = os.path.join(HERE, "libbh_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC",
           "-shared", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
