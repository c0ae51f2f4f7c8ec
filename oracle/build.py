"""Builds oracle/libgrim_oracle.so from grim_oracle.c (ORACLE = test infrastructure, not the product).

    python oracle/build.py

Flags: -O2 -ffp-contract=off (no FMA contraction: every +,-,*,/,sqrt is a separately rounded IEEE
operation, which is what the GPU library's strict arithmetic mode reproduces bit for bit) -fopenmp.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "grim_oracle.c")
HDR = os.path.join(HERE, "grim_oracle.h")
LIB = os.path.join(HERE, "libgrim_oracle.so")


def build(force: bool = False) -> str:
    if (not force and os.path.exists(LIB)
            and os.path.getmtime(LIB) >= max(os.path.getmtime(SRC), os.path.getmtime(HDR))):
        return LIB
    cmd = ["gcc", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared", "-std=gnu11", "-Wall",
           "-o", LIB + ".tmp", SRC, "-lm"]
    subprocess.check_call(cmd)
    os.replace(LIB + ".tmp", LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
