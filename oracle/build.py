"""Build the CPU oracle (test infrastructure) into oracle/libmd_oracle.so with g++.

    python oracle/build.py

Flags: -O2 -ffp-contract=off (no fused multiply-adds may be formed from the source's * and +: the oracle's
floating-point steps are exactly the ones written), no -ffast-math, OpenMP for the row loops.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "md_oracle.cpp")
LIB = os.path.join(HERE, "libmd_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
