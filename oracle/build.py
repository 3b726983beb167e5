"""Compile the CPU oracle (oracle/skv_oracle.c) into oracle/libskv_oracle.so with gcc.

TEST INFRASTRUCTURE: building the checker is not using it.  Flags: no fast-math, no FMA
contraction (the quantizer's fp32 steps are specified as separately rounded operations).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "skv_oracle.c")
LIB = os.path.join(HERE, "libskv_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off",
           "-fno-fast-math", "-Wall", "-Wextra", "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
