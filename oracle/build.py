"""Build the CPU oracle shared libraries (test infrastructure, not the product).

    python oracle/build.py          # builds libmfo.so (1 thread) and libmfo_omp.so (-fopenmp, bit-identical)

g++ -O2 -ffp-contract=off: the written order of operations is the executed one (A16).
"""
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
SRC = os.path.join(HERE, "mfo_oracle.cpp")
HDR = os.path.join(HERE, "mfo_oracle.h")
LIB = os.path.join(HERE, "libmfo.so")
LIB_OMP = os.path.join(HERE, "libmfo_omp.so")

BASE = ["g++", "-std=c++17", "-O2", "-ffp-contract=off", "-fno-fast-math", "-fPIC", "-shared",
        "-Wall", "-Wextra", "-Wno-unknown-pragmas"]


def _stale(out):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(p) > t for p in (SRC, HDR, __file__))


def build(force=False, verbose=False):
    """Compile both variants if missing or older than the sources. Returns (LIB, LIB_OMP)."""
    for out, extra in ((LIB, []), (LIB_OMP, ["-fopenmp"])):
        if force or _stale(out):
            cmd = BASE + extra + [SRC, "-o", out + ".tmp"]
            if verbose:
                print(" ".join(cmd), file=sys.stderr)
            subprocess.run(cmd, check=True)
            os.replace(out + ".tmp", out)
    return LIB, LIB_OMP


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose=True)
