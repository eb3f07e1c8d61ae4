"""Helpers of the GPU parity tests: drive the CUDA path (through the C ABI) and the oracle from the same
seeded host arrays, and compare with the norm of DESIGN.md reading A17."""
import numpy as np

from oracle.mfo import Oracle
from paper_1510_06340_b200.binding import MustaForce

TOL = 1e-11          # BASELINE.json north_star: max relative difference <= 1e-11 per field after 100 steps


def make_pair(st, omp=True, path="auto", strict=False, **over):
    """(gpu, oracle) contexts for a workload dict from paper_1510_06340_b200.workloads."""
    nz, ny, nx = st["shape"]
    kw = dict(st["scheme"])
    kw.update(over)
    g = MustaForce(nx, ny, nz, dx=st["dx"], path=path, strict=strict, **kw)
    o = Oracle(nx, ny, nz, dx=st["dx"], omp=omp, **kw)
    for h in (g, o):
        h.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
        if "jet" in st:
            j = st["jet"]
            h.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
    return g, o


def field_scales(ref):
    ref = [np.asarray(a, dtype=np.float64) for a in ref]
    return np.abs(ref[0]).max(), np.sqrt(ref[1] ** 2 + ref[2] ** 2 + ref[3] ** 2).max(), np.abs(ref[4]).max()


def rel_diff(got, ref, scales=None):
    """A17: per-field max|G-O| / max|O|; the three momentum components share max|M|; a field whose oracle
    max-norm is 0 is measured against max|E|.  Returns (rel_E, rel_M, rel_R).  `scales` = the max-norms of the
    WHOLE field when got/ref are only a window of it."""
    got = [np.asarray(a, dtype=np.float64) for a in got]
    ref = [np.asarray(a, dtype=np.float64) for a in ref]
    sE, sM, sR = scales if scales is not None else field_scales(ref)
    if sM == 0.0:
        sM = sE
    if sR == 0.0:
        sR = sE
    dM = max(np.abs(got[q] - ref[q]).max() for q in (1, 2, 3))
    return np.abs(got[0] - ref[0]).max() / sE, dM / sM, np.abs(got[4] - ref[4]).max() / sR


def assert_parity(got, ref, tol=TOL, what="", scales=None):
    assert all(np.all(np.isfinite(a)) for a in got), "non-finite GPU state " + what
    r = rel_diff(got, ref, scales)
    assert max(r) <= tol, "parity %s: rel diff (E, M, R) = %s > %g" % (what, r, tol)
    return r
