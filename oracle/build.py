"""Build the oracle shared library (test infrastructure only; see oracle/README.md).

    python oracle/build.py

Compiles oracle/oracle_api.cpp with g++ (-O3 -march=native as BASELINE.md section 3 states for the timed CPU baseline, OpenMP,
IEEE arithmetic: no -ffast-math) into oracle/liboracle.so.  Called by __graft_entry__.build() and, lazily, by oracle/oracle.py.
The library is specific to the CPU it was built on: a stamp (flags of this CPU + the command line) sits beside it, and a
library carried over from another machine (the GPU box receives this tree) is rebuilt there.
"""
import hashlib
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = ["oracle_api.cpp"]
HDR = ["su3.hpp", "kin.hpp", "rambo.hpp", "diagrams.hpp", "colour.hpp", "eval.hpp", "berends_giele.hpp"]
LIB = os.path.join(HERE, "liboracle.so")


STAMP = os.path.join(HERE, "liboracle.stamp")
CMD = ["g++", "-std=c++17", "-O3", "-march=native", "-fopenmp", "-fPIC", "-shared", "-Wall"]


def _stamp():
    flags = ""
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("flags") or line.startswith("model name"):
                    flags += line
                    if line.startswith("flags"):
                        break
    except OSError:
        pass
    return hashlib.sha256((flags + " ".join(CMD)).encode()).hexdigest()


def needs_build():
    if not os.path.exists(LIB) or not os.path.exists(STAMP):
        return True
    if open(STAMP).read().strip() != _stamp():
        return True
    t = os.path.getmtime(LIB)
    return any(os.path.getmtime(os.path.join(HERE, f)) > t for f in SRC + HDR)


def build(force=False):
    if not force and not needs_build():
        return LIB
    tmp = LIB + ".%d.tmp" % os.getpid()
    subprocess.check_call(CMD + ["-o", tmp] + [os.path.join(HERE, s) for s in SRC], cwd=HERE)
    os.replace(tmp, LIB)
    with open(STAMP, "w") as f:
        f.write(_stamp() + "\n")
    return LIB


if __name__ == "__main__":
    print(build(force="--force" in sys.argv))
