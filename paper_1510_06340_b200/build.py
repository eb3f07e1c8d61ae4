"""Compile csrc/*.cu into the C-ABI shared library for sm_100a, in tree.

    python -m paper_1510_06340_b200.build [--force] [--verbose]

Outputs (git-ignored, shipped to the GPU box by gpurun):
    paper_1510_06340_b200/libmustaforce.so          the product
    paper_1510_06340_b200/libmustaforce_strict.so   same sources with --fmad=false -DMF_STRICT: no FMA contraction, so that
                                                    its results can be compared bit-for-bit with the oracle (a debugging aid
                                                    used by tests/test_parity_strict.py; never timed)
nvcc cross-compiles without a GPU.
"""
import glob
import os
import subprocess
import sys

HERE = os.path.dirname(os.path.abspath(__file__))
CSRC = os.path.join(HERE, "csrc")
INCLUDE = os.path.join(os.path.dirname(HERE), "include")
LIB = os.path.join(HERE, "libmustaforce.so")
LIB_STRICT = os.path.join(HERE, "libmustaforce_strict.so")

NVCC = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
ARCH = ["-gencode", "arch=compute_100a,code=sm_100a"]
COMMON = ["-O3", "-std=c++17", "-lineinfo", "-Xcompiler", "-fPIC", "-shared", "-I", INCLUDE, "-I", CSRC,
          "-Xptxas", "-v", "--resource-usage"]


def sources():
    return sorted(glob.glob(os.path.join(CSRC, "*.cu")))


def _deps():
    return sources() + glob.glob(os.path.join(CSRC, "*.h")) + glob.glob(os.path.join(CSRC, "*.cuh")) + \
        [os.path.join(INCLUDE, "mustaforce.h"), os.path.abspath(__file__)]


def _stale(out):
    if not os.path.exists(out):
        return True
    t = os.path.getmtime(out)
    return any(os.path.getmtime(p) > t for p in _deps())


def _compile(out, extra, verbose):
    cmd = [NVCC] + ARCH + COMMON + extra + sources() + ["-o", out + ".tmp"]
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    log = out.replace(".so", ".build.log")
    with open(log, "w") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout)
    if res.returncode != 0:
        sys.stderr.write(res.stdout)
        raise RuntimeError("nvcc failed for %s (log: %s)" % (out, log))
    if verbose:
        sys.stderr.write(res.stdout)
    os.replace(out + ".tmp", out)


def build(force=False, verbose=False, strict=True):
    if force or _stale(LIB):
        _compile(LIB, [], verbose)
    if strict and (force or _stale(LIB_STRICT)):
        _compile(LIB_STRICT, ["--fmad=false", "-DMF_STRICT"], verbose)
    return LIB, LIB_STRICT


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(LIB)
