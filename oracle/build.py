"""Compile the C oracle (TEST INFRASTRUCTURE) into oracle/liboracle_hpmc.so with gcc.

-ffp-contract=off and no fast-math: the fp32 pins (cell_of, translation fmaf, wrap) need IEEE
single-precision operations exactly as written.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "hpmc_oracle.c")
HDR = os.path.join(HERE, "hpmc_oracle.h")
LIB = os.path.join(HERE, "liboracle_hpmc.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB):
        newest = max(os.path.getmtime(SRC), os.path.getmtime(HDR))
        if os.path.getmtime(LIB) >= newest:
            return LIB
    cmd = ["gcc", "-O2", "-std=c99", "-Wall", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-o", LIB, SRC, "-lm"]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
