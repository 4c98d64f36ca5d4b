"""Compile oracle/nbody_oracle.c into oracle/liboracle.so (TEST INFRASTRUCTURE, not the product).

Flags are normative for bit-reproducibility (SURVEY.md 8c header, c-14): -O2 -ffp-contract=off,
no -ffast-math, OpenMP over particles only.  Called by tests/conftest.py, __graft_entry__.build()
and bench.py's cpu_baseline / --impl reference legs; never by the product package.
"""
import os
import subprocess

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "nbody_oracle.c")
LIB = os.path.join(HERE, "liboracle.so")
FLAGS = ["-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared", "-std=c11"]


def build(force: bool = False) -> str:
    if (not force) and os.path.exists(LIB) and os.path.getmtime(LIB) >= os.path.getmtime(SRC):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()
    subprocess.check_call(["gcc", *FLAGS, SRC, "-o", tmp, "-lm"])
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force=True))
