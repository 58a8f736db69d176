"""Builds oracle/libpwa_oracle.so from oracle/pwa_oracle.c with gcc.

TEST INFRASTRUCTURE: the oracle is the independent CPU checker, not product code.
Plain `-O2`, no `-ffast-math`, FMA contraction off, so the compensated sums survive.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "pwa_oracle.c")
LIB = os.path.join(HERE, "libpwa_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= os.path.getmtime(SRC)):
        return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", "-Wall", "-Wextra", "-o", LIB, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
