"""Build the CPU oracle (test infrastructure) into oracle/libmg_oracle.so with g++ -O2 -fopenmp.

-ffp-contract=off: no fused multiply-adds, so the fp64 arithmetic is exactly what the source says.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mg_oracle.cpp")
LIB = os.path.join(HERE, "libmg_oracle.so")


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    cmd = ["g++", "-O2", "-fopenmp", "-ffp-contract=off", "-fPIC", "-shared", "-std=c++17", "-Wall", "-o", LIB, SRC]
    subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
