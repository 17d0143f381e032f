"""Compile the CPU oracle (oracle/etics_oracle.cpp) into oracle/libetics_oracle.so.

TEST INFRASTRUCTURE.  Flags: -O2 -ffp-contract=off (no implicit FMA contraction, so the only fused
operations are the std::fma calls that pin the sort key's rounding), -fopenmp for the threaded figure.
"""
from __future__ import annotations

import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "etics_oracle.cpp")
LIB = os.path.join(HERE, "libetics_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", SRC, "-o", LIB + ".tmp"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
