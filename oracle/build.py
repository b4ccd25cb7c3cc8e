"""Build the CPU oracle (TEST INFRASTRUCTURE) into oracle/liboracle_tdse.so.

Flags follow SURVEY §8(c): -O2 -ffp-contract=off, no fast-math, so every sum is
evaluated exactly in the order the source states.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "tdse_oracle.cpp")
HDR = os.path.join(HERE, "tdse_oracle.h")
LIB = os.path.join(HERE, "liboracle_tdse.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp",
           "-shared", "-fPIC", "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
