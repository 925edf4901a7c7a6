"""ORACLE — TEST INFRASTRUCTURE ONLY.  Compiles oracle/libmfc_oracle.so with g++.

-O2 -ffp-contract=off: no FMA contraction, so every operation is rounded exactly as
written in mfc_oracle.hpp (DESIGN.md §3 N1).  OpenMP only spreads independent lines /
cells over host cores; it does not change any arithmetic.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libmfc_oracle.so")
SRC = [os.path.join(HERE, "mfc_oracle_capi.cpp")]
DEPS = SRC + [os.path.join(HERE, "mfc_oracle.hpp")]


def build(force: bool = False) -> str:
    if not force and os.path.exists(LIB) and all(os.path.getmtime(LIB) >= os.path.getmtime(d) for d in DEPS):
        return LIB
    tmp = LIB + ".tmp.%d" % os.getpid()  # complete before it takes the library's name (several processes may build at once)
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-Wextra", "-Wno-maybe-uninitialized", "-o", tmp] + SRC
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
