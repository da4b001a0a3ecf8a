"""Build the CPU oracle (test infrastructure) into oracle/libox.so with g++.

Flags follow DESIGN.md reading R21: -O2 -ffp-contract=off (no FMA contraction), IEEE
division and square root, OpenMP over the outermost grid index.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ox_oracle.cpp")
HDR = os.path.join(HERE, "ox.h")
LIB = os.path.join(HERE, "libox.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        if os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR)):
            return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
