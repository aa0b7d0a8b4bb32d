"""Build the CPU oracle (TEST INFRASTRUCTURE, not product code).

    python oracle/build.py          ->  oracle/liboracle.so, oracle/flopcount

-ffp-contract=off: the oracle evaluates every expression exactly as written (no FMA
contraction), so that it is a fixed point of reference for the CUDA path's parity tests.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
LIB = os.path.join(HERE, "liboracle.so")
FLOP = os.path.join(HERE, "flopcount")
CXXFLAGS = ["-O2", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-fopenmp", "-Wall"]


def _stale(target, sources):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(s) > t for s in sources)


def build(force=False, verbose=False):
    core = os.path.join(HERE, "oracle_core.hpp")
    src = os.path.join(HERE, "oracle.cpp")
    if force or _stale(LIB, [core, src, __file__]):
        cmd = ["g++", *CXXFLAGS, "-shared", "-fPIC", src, "-o", LIB]
        if verbose:
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    fsrc = os.path.join(HERE, "flopcount.cpp")
    if os.path.exists(fsrc) and (force or _stale(FLOP, [core, fsrc, __file__])):
        cmd = ["g++", "-O1", "-std=c++17", "-ffp-contract=off", fsrc, "-o", FLOP]
        if verbose:
            print(" ".join(cmd))
        subprocess.check_call(cmd)
    return LIB


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
    print(LIB)
