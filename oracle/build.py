"""Builds the CPU oracle shared library (test infrastructure; see swe_oracle.cpp header).

    python -m oracle.build

g++ -O2 -ffp-contract=off keeps the arithmetic reproducible across hosts (no FMA contraction);
OpenMP only parallelises the loops over cells, each cell's arithmetic is unchanged.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRCS = [os.path.join(HERE, "swe_oracle.cpp")]
LIB = os.path.join(HERE, "liborc.so")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.exists(s) and os.path.getmtime(s) > t for s in SRCS)


def build(force=False, verbose=False):
    if not force and not needs_build():
        return LIB
    srcs = [s for s in SRCS if os.path.exists(s)]
    tmp = LIB + ".tmp.%d" % os.getpid()
    cmd = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
           "-Wall", "-o", tmp] + srcs
    if verbose:
        print(" ".join(cmd))
    subprocess.check_call(cmd)
    os.replace(tmp, LIB)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
