"""Build the CPU oracle (test infrastructure) into oracle/liboracle_mpc.so.

Flags follow reading U1: no contraction, no fast-math, so that every fused
multiply-add in the binning expression is the explicit fmaf written in the source.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mpc_oracle.cpp")
LIB = os.path.join(HERE, "liboracle_mpc.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", LIB, SRC]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
