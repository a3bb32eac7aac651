"""Compile the fp64 C oracle into oracle/libnpfem_oracle.so (gcc -O2 -fopenmp).

TEST INFRASTRUCTURE: building the checker is not using it.  Called by __graft_entry__.build()
and lazily by oracle/npfem_oracle.py.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "npfem_oracle.c")
LIB = os.path.join(HERE, "libnpfem_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
           "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
