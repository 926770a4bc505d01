"""Compile the CPU oracle (test infrastructure) into oracle/libgothic_oracle.so.

g++ -O2 -std=c++17 -fopenmp -ffp-contract=off: contraction is disabled because the oracle spells out
every fused multiply-add that decides an integer (R11)."""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "gothic_oracle.cpp")
LIB = os.path.join(HERE, "libgothic_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
