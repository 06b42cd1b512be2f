"""Compile the CPU oracle (oracle/ds_oracle.c) into oracle/libds_oracle.so with gcc.

TEST INFRASTRUCTURE.  Plain -O2, no fast-math, no FMA contraction, OpenMP only for the
timed multi-thread baseline (results are bit-identical at any thread count).
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "ds_oracle.c")
LIB = os.path.join(HERE, "libds_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + f".tmp{os.getpid()}"
    cmd = ["gcc", "-std=c99", "-O2", "-fno-fast-math", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-o", tmp, SRC, "-lm"]
    subprocess.run(cmd, check=True)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
