"""Build the oracle shared library (test infrastructure only; see oracle/README.md).

    python oracle/build.py

Compiles oracle/oracle_api.cpp with g++ (-O2, OpenMP, IEEE arithmetic: no -ffast-math) into
oracle/liboracle.so.  Called by __graft_entry__.build() and, lazily, by oracle/oracle.py.
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = ["oracle_api.cpp"]
HDR = ["su3.hpp", "kin.hpp", "rambo.hpp", "diagrams.hpp", "colour.hpp", "eval.hpp", "berends_giele.hpp"]
LIB = os.path.join(HERE, "liboracle.so")


def needs_build():
    if not os.path.exists(LIB):
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SRC + HDR)


def build(force=False):
    if not force and not needs_build():
        return LIB
    cmd = ["g++", "-std=c++17", "-O2", "-fopenmp", "-fPIC", "-shared", "-Wall",
           "-o", LIB] + [os.path.join(HERE, s) for s in SRC]
    subprocess.check_call(cmd, cwd=HERE)
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
