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


def _newer(target, deps):
    if not os.path.exists(target):
        return True
    t = os.path.getmtime(target)
    return any(os.path.getmtime(p) > t for p in deps)


def _run(cmd, log, verbose):
    if verbose:
        print(" ".join(cmd), file=sys.stderr)
    res = subprocess.run(cmd, stdout=subprocess.PIPE, stderr=subprocess.STDOUT, text=True)
    with open(log, "a") as f:
        f.write(" ".join(cmd) + "\n" + res.stdout)
    if res.returncode != 0:
        sys.stderr.write(res.stdout)
        raise RuntimeError("nvcc failed: %s (log: %s)" % (cmd[-1], log))
    if verbose:
        sys.stderr.write(res.stdout)


def _compile(out, extra, verbose, force):
    """One object per .cu (compiled in parallel, kept under build/ next to the library, rebuilt when a source or header is newer),
    then one link."""
    tag = os.path.basename(out).replace(".so", "")
    objdir = os.path.join(HERE, "build", tag)
    os.makedirs(objdir, exist_ok=True)
    log = out.replace(".so", ".build.log")
    open(log, "w").close()
    headers = [p for p in _deps() if not p.endswith(".cu")]
    flags = [f for f in COMMON if f != "-shared"]
    jobs, objs = [], []
    for src in sources():
        obj = os.path.join(objdir, os.path.basename(src).replace(".cu", ".o"))
        objs.append(obj)
        if force or _newer(obj, [src] + headers):
            jobs.append([NVCC] + ARCH + flags + extra + ["-c", src, "-o", obj])
    if jobs:
        from concurrent.futures import ThreadPoolExecutor
        with ThreadPoolExecutor(max_workers=min(len(jobs), os.cpu_count() or 4)) as ex:
            list(ex.map(lambda cmd: _run(cmd, log, verbose), jobs))
    if jobs or force or _newer(out, objs):
        _run([NVCC] + ARCH + ["-shared", "-Xcompiler", "-fPIC"] + objs + ["-o", out + ".tmp"], log, verbose)
        os.replace(out + ".tmp", out)


def build(force=False, verbose=False, strict=True):
    from concurrent.futures import ThreadPoolExecutor
    with ThreadPoolExecutor(max_workers=2) as ex:                    # the two variants side by side
        futs = [ex.submit(_compile, LIB, [], verbose, force)]
        if strict:
            futs.append(ex.submit(_compile, LIB_STRICT, ["--fmad=false", "-DMF_STRICT"], verbose, force))
        for f in futs:
            f.result()
    return LIB, LIB_STRICT


if __name__ == "__main__":
    build(force="--force" in sys.argv, verbose="--verbose" in sys.argv)
    print(LIB)
