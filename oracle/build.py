"""Builds oracle/libpsdf_oracle.so (g++ -O2 -fopenmp, no -ffast-math).

The oracle is test infrastructure (see psdf_oracle.cpp header).  `__graft_entry__.build()`
calls this too: building the checker is not using it.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "psdf_oracle.cpp")
LIB = os.path.join(HERE, "libpsdf_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-shared", "-fPIC", "-Wall", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
