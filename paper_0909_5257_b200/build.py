"""Build the heget-b200 native code in-tree for sm_100a.

    python -m paper_0909_5257_b200.build [--only TAG ...] [--force] [--jobs N]

1. g++   csrc/gen/hegetgen.cpp                      -> bin/hegetgen        (process generator, step a0)
2. nvcc  csrc/api.cu + csrc/gen/genlib.cpp          -> libheget.so         (C-ABI of include/heget.h + RAMBO kernel)
3. for every process in PROCESSES: hegetgen -> kernels/gen_<tag>.cu, then one nvcc per precision
                                                   -> kernels/heget_<tag>_f64.so, _f32.so, _f32p.so (packed f32x2)
Up-to-date outputs (newer than every source they depend on) are skipped.  Processes not listed here are generated and
compiled by heget_process_create at first use (needs nvcc at run time).
(`ptxas -O1` halves the compile time of the big processes but costs 10-35 % of their speed -- measured, not used.)
"""
import argparse
import concurrent.futures as cf
import os
import subprocess
import sys
import time

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
KDIR = os.path.join(HERE, "kernels")
BIN = os.path.join(HERE, "bin")
LIB = os.path.join(HERE, "libheget.so")
NVCC = os.environ.get("HEGET_NVCC", "nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a", "-lineinfo"]

# BASELINE.json configs C1..C4 first (C5: SLOW_PROCESSES), then the small processes the parity tests use
PROCESSES = [
    "u u~ > g g",
    "g g > g g g",
    "u u > u u g g",
    "g g > g g g g",
    "g g > g g",
    "u u > u u",
    "u u~ > g g g",
    "u u > u u g",
    "u u~ > g g g g",
    "u g > u g g",          # a crossing of u u~ > g g g
]


# The straight-line kernels of the 7-leg config take ~10 minutes of ptxas per precision; the table back end (no compilation)
# is what serves processes with >= 6 legs, so they are only built on request: `python -m paper_0909_5257_b200.build --slow`.
SLOW_PROCESSES = ["u u~ > g g g g g"]

# The packed-FP32 path (HEGET_FP32X2) is an experiment that did not pay: pre-built only for the two
# processes its tests use; any other process is compiled on demand by heget_process_create.
PACKED_PROCESSES = ["u u~ > g g", "g g > g g g"]


def tag_of(process):
    return "".join("_" if c == ">" else "x" if c == "~" else c for c in process if c != " ")


def n_legs(process):
    return len([t for t in process.split() if t != ">"])


def _newer(target, deps):
    if not os.path.exists(target):
        return False
    t = os.path.getmtime(target)
    return all(os.path.getmtime(d) <= t for d in deps)


def _run(cmd, log=None):
    t0 = time.time()
    r = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    if log:
        with open(log, "w") as f:
            f.write(" ".join(cmd) + "\n" + r.stdout)
    if r.returncode != 0:
        raise RuntimeError("command failed: %s\n%s" % (" ".join(cmd), r.stdout[-4000:]))
    return time.time() - t0


def gen_sources():
    g = os.path.join(CSRC, "gen")
    return [os.path.join(g, f) for f in sorted(os.listdir(g))]


def dev_sources():
    d = os.path.join(CSRC, "device")
    return [os.path.join(d, f) for f in sorted(os.listdir(d))]


def build_generator(force=False):
    os.makedirs(BIN, exist_ok=True)
    exe = os.path.join(BIN, "hegetgen")
    if force or not _newer(exe, gen_sources()):
        _run(["g++", "-std=c++17", "-O2", "-o", exe, os.path.join(CSRC, "gen", "hegetgen.cpp")])
    return exe


def build_library(force=False):
    deps = gen_sources() + dev_sources() + [os.path.join(CSRC, "api.cu"), os.path.join(CSRC, "rambo.cuh"),
                                            os.path.join(HERE, "..", "include", "heget.h")]
    if force or not _newer(LIB, deps):
        _run([NVCC, "-std=c++17", "-O3"] + ARCH + ["-shared", "-Xcompiler", "-fPIC", "-o", LIB,
             os.path.join(CSRC, "api.cu"), os.path.join(CSRC, "gen", "genlib.cpp"), "-ldl"])
    return LIB


def _compile_plugin(cu, so, prec, nlegs):
    cmd = [NVCC, "-std=c++17", "-O3"] + ARCH + ["-shared", "-Xcompiler", "-fPIC", "-Xptxas", "-v",
           "-DHG_ONLY_PREC=%d" % prec] + (["-DHG_NO_LANES1"] if nlegs >= 6 else []) + \
          ["-I" + os.path.join(CSRC, "device"), "-o", so + ".tmp", cu]
    dt = _run(cmd, log=so[:-3] + ".log")
    os.replace(so + ".tmp", so)
    return so, dt


def build_kernels(processes=None, force=False, jobs=None, verbose=True):
    exe = build_generator(force)
    os.makedirs(KDIR, exist_ok=True)
    todo = []
    for proc in (processes or PROCESSES):
        tag = tag_of(proc)
        cu = os.path.join(KDIR, "gen_%s.cu" % tag)
        if force or not _newer(cu, [exe]):
            _run([exe, tag, proc, cu])
        precs = [(0, "f64"), (1, "f32")] + ([(2, "f32p")] if proc in PACKED_PROCESSES else [])
        for prec, suf in precs:
            so = os.path.join(KDIR, "heget_%s_%s.so" % (tag, suf))
            if force or not _newer(so, [cu] + dev_sources()):
                todo.append((cu, so, prec, n_legs(proc)))
    # biggest first so the long compiles start at once
    todo.sort(key=lambda t: -os.path.getsize(t[0]))
    jobs = jobs or max(1, (os.cpu_count() or 2))
    with cf.ThreadPoolExecutor(max_workers=jobs) as ex:
        futs = [ex.submit(_compile_plugin, *t) for t in todo]
        for f in cf.as_completed(futs):
            so, dt = f.result()
            if verbose:
                print("built %s in %.0f s" % (os.path.relpath(so, HERE), dt), flush=True)
    return KDIR


def build_all(processes=None, force=False, jobs=None, verbose=True):
    build_library(force)
    build_kernels(processes, force, jobs, verbose)
    return LIB


if __name__ == "__main__":
    ap = argparse.ArgumentParser()
    ap.add_argument("--only", nargs="*", help="process strings to build (default: the configured list)")
    ap.add_argument("--force", action="store_true")
    ap.add_argument("--slow", action="store_true", help="also build the straight-line kernels of SLOW_PROCESSES")
    ap.add_argument("--jobs", type=int, default=None)
    a = ap.parse_args()
    print(build_all(a.only or (PROCESSES + SLOW_PROCESSES if a.slow else None), a.force, a.jobs))
