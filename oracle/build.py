"""Builds the CPU oracle shared library (test infrastructure, not the product).

    python -m oracle.build

g++ -O2 -ffp-contract=off: no FMA contraction, so the marker index arithmetic of step I-1
 is reproducible operation by operation.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libfs_oracle.so")
SRC = os.path.join(HERE, "fs_oracle.cpp")
HDR = os.path.join(HERE, "fs_oracle.h")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["g++", "-O2", "-ffp-contract=off", "-std=c++17", "-Wall", "-shared", "-fPIC", SRC, "-o", LIB]
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
