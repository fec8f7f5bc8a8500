"""Compile oracle/twk_oracle.cpp into oracle/libtwk_oracle.so (g++ -O2 -fopenmp).  TEST INFRASTRUCTURE ONLY.

Called by oracle.api on first use and by __graft_entry__.build() (building the checker is not using it).
-O2 without -ffast-math: the oracle's arithmetic must stay in the order it is written.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "twk_oracle.cpp")
LIB = os.path.join(HERE, "libtwk_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-o", tmp, SRC]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
