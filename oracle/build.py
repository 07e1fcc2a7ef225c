"""Build the CPU oracle (test infrastructure) into oracle/liboracle_mpc.so.

Flags follow reading U1: no contraction, no fast-math, so that every fused
multiply-add in the binning expression is the explicit fmaf written in the source.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mpc_oracle.cpp")
LIB = os.path.join(HERE, "liboracle_mpc.so")


LIB_SAN = os.path.join(HERE, "liboracle_mpc_san.so")


def build(force: bool = False, sanitize: bool = False) -> str:
    """sanitize=True: a second library built with -fsanitize=address,undefined (tests/test_oracle_sanitize.py loads it in a
    child process that preloads the sanitizer runtimes); same arithmetic flags."""
    lib = LIB_SAN if sanitize else LIB
    if not force and os.path.exists(lib) and os.path.getmtime(lib) >= os.path.getmtime(SRC):
        return lib
    cmd = ["g++", "-O1" if sanitize else "-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared", "-Wall", "-Wextra"]
    if sanitize:
        cmd += ["-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
    subprocess.run(cmd + ["-o", lib, SRC], check=True)
    return lib


if __name__ == "__main__":
    print(build(force=True))
