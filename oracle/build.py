"""Build the CPU oracle (test infrastructure) into oracle/libora.so.

g++ -O2 -ffp-contract=off: no FMA contraction, so the oracle is a fixed IEEE reference
(SURVEY.md §8(c)).  OpenMP only parallelises loops over independent cells/faces, so the
result is identical for any thread count.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "libora.so")
SOURCES = ["ora_capi.cpp"]
HEADERS = ["ora.h", "ora_core.hpp", "ora_solver.hpp", "ora_naive.hpp"]


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SOURCES + HEADERS + ["build.py"])


def build(force=False):
    if not force and not needs_build():
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", LIB] + [os.path.join(HERE, s) for s in SOURCES]
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
