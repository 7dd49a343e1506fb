"""Builds oracle/libcavmag_oracle.so from cavmag_oracle.cpp with g++ (test infrastructure).

-ffp-contract=off keeps every cell's arithmetic identical (no FMA contraction that could
differ between boundary and interior code paths).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "cavmag_oracle.cpp")
LIB = os.path.join(HERE, "libcavmag_oracle.so")


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-fopenmp", "-shared", "-fPIC", "-std=c++17",
           "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
