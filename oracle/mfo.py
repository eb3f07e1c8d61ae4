"""ctypes front end of the CPU oracle (oracle/mfo_oracle.cpp).  TEST INFRASTRUCTURE ONLY.

May be imported by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs, never by the product package.  It imports nothing from paper_1510_06340_b200.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

LIM = {"none": 0, "minmod": 1, "superbee": 2, "vanalbada": 3, "vanleer": 4, "mc": 5, "first": 6}
BC = {"outflow": 0, "periodic": 1}
EOS_CS2, EOS_TABLE = 0, 1
OK, EINVAL, ENOMEM, ESTATE = 0, -1, -2, -4

_dp = C.POINTER(C.c_double)
_libs = {}


def _load(omp):
    if omp in _libs:
        return _libs[omp]
    import importlib.util
    spec = importlib.util.spec_from_file_location("_mfo_build", os.path.join(_HERE, "build.py"))
    b = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(b)
    lib_path, omp_path = b.build()
    lib = C.CDLL(omp_path if omp else lib_path)
    vp = C.c_void_p
    d5 = [_dp] * 5
    sig = {
        "mfo_create": (vp, [C.c_int] * 3 + [C.c_double] + [C.c_int] * 3),
        "mfo_destroy": (None, [vp]),
        "mfo_set_state": (C.c_int, [vp] + d5),
        "mfo_get_state": (C.c_int, [vp] + d5),
        "mfo_set_state_prim": (C.c_int, [vp] + d5),
        "mfo_get_state_prim": (C.c_int, [vp] + d5),
        "mfo_step": (C.c_int, [vp, C.c_int, C.c_double]),
        "mfo_step_dt": (C.c_int, [vp, C.c_int, C.c_double]),
        "mfo_conserved_totals": (C.c_int, [vp, _dp]),
        "mfo_get_time": (C.c_int, [vp, _dp, _dp, C.POINTER(C.c_longlong)]),
        "mfo_max_signal_speed": (C.c_int, [vp, _dp]),
        "mfo_set_rk": (C.c_int, [vp, C.c_int]),
        "mfo_set_boundary": (C.c_int, [vp, C.c_int]),
        "mfo_set_cs2": (C.c_int, [vp, C.c_double]),
        "mfo_set_predictor": (C.c_int, [vp, C.c_int]),
        "mfo_set_state_precision": (C.c_int, [vp, C.c_int]),
        "mfo_set_alpha": (C.c_int, [vp, C.c_double]),
        "mfo_set_jet_source": (C.c_int, [vp] + [C.c_double] * 5),
        "mfo_set_eos_table": (C.c_int, [vp, C.c_int, C.c_int] + [C.c_double] * 4 + [_dp]),
        "mfo_eos": (C.c_int, [vp, C.c_double, C.c_double, _dp]),
        "mfo_sync": (C.c_int, [vp]),
        "mfo_last_error": (C.c_char_p, [vp]),
        "mfo_slope": (C.c_double, [C.c_int, C.c_double, C.c_double]),
        "mfo_flux": (C.c_int, [vp, C.c_int, _dp, _dp]),
        "mfo_con2prim": (C.c_int, [vp, _dp, _dp]),
        "mfo_prim2con": (C.c_int, [vp, _dp, _dp]),
        "mfo_musta_flux": (C.c_int, [vp, C.c_int, C.c_double, _dp, _dp, _dp]),
        "mfo_eval_L": (C.c_int, [vp, C.c_double] + d5),
        "mfo_eval_faces": (C.c_int, [vp, C.c_double, C.c_int, C.c_int, _dp]),
        "mfo_num_threads": (C.c_int, []),
    }
    for name, (res, args) in sig.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _libs[omp] = lib
    return lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a, n=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if n is not None and a.size != n:
        raise ValueError("array has %d elements, expected %d" % (a.size, n))
    return a


class OracleError(RuntimeError):
    pass


class Oracle:
    """One oracle context.  Arrays are numpy float64 of shape (nz, ny, nx) (x fastest) or flat."""

    def __init__(self, nx, ny=1, nz=1, dx=1.0, limiter="minmod", k_stages=2, rk=2, bc="outflow",
                 predictor=True, alpha=None, cs2=None, omp=False, eos_table=None, state_bits=64):
        self.lib = _load(omp)
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        lim = LIM[limiter] if isinstance(limiter, str) else int(limiter)
        self.h = self.lib.mfo_create(nx, ny, nz, float(dx), EOS_CS2 if eos_table is None else EOS_TABLE, lim, int(k_stages))
        if not self.h:
            raise OracleError("mfo_create failed (bad arguments)")
        self._chk(self.lib.mfo_set_rk(self.h, int(rk)))
        self._chk(self.lib.mfo_set_boundary(self.h, BC[bc] if isinstance(bc, str) else int(bc)))
        self._chk(self.lib.mfo_set_predictor(self.h, 1 if predictor else 0))
        if alpha is not None:
            self._chk(self.lib.mfo_set_alpha(self.h, float(alpha)))
        if cs2 is not None:
            self._chk(self.lib.mfo_set_cs2(self.h, float(cs2)))
        if eos_table is not None:
            self.set_eos_table(eos_table)
        if state_bits != 64:
            self._chk(self.lib.mfo_set_state_precision(self.h, int(state_bits)))

    def _chk(self, rc, allow=()):
        if rc != OK and rc not in allow:
            raise OracleError("oracle error %d: %s" % (rc, self.lib.mfo_last_error(self.h).decode()))
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.lib.mfo_destroy(self.h)
            self.h = None

    __del__ = close

    def set_state(self, E, Mx, My, Mz, R):
        a = [_f64(x, self.n) for x in (E, Mx, My, Mz, R)]
        self._chk(self.lib.mfo_set_state(self.h, *[_p(x) for x in a]))

    def set_state_prim(self, e, vx, vy, vz, n):
        a = [_f64(x, self.n) for x in (e, vx, vy, vz, n)]
        self._chk(self.lib.mfo_set_state_prim(self.h, *[_p(x) for x in a]))

    def get_state(self):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self.lib.mfo_get_state(self.h, *[_p(x) for x in out]), allow=(ESTATE,))
        return out

    def get_state_prim(self):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self.lib.mfo_get_state_prim(self.h, *[_p(x) for x in out]), allow=(ESTATE,))
        return out

    def step(self, n, cfl):
        return self._chk(self.lib.mfo_step(self.h, int(n), float(cfl)), allow=(ESTATE,))

    def step_dt(self, n, dt):
        return self._chk(self.lib.mfo_step_dt(self.h, int(n), float(dt)), allow=(ESTATE,))

    def totals(self):
        out = np.empty(5)
        self._chk(self.lib.mfo_conserved_totals(self.h, _p(out)), allow=(ESTATE,))
        return out

    def time(self):
        t, dt, s = C.c_double(), C.c_double(), C.c_longlong()
        self._chk(self.lib.mfo_get_time(self.h, C.byref(t), C.byref(dt), C.byref(s)), allow=(ESTATE,))
        return t.value, dt.value, s.value

    def max_signal_speed(self):
        s = C.c_double()
        rc = self._chk(self.lib.mfo_max_signal_speed(self.h, C.byref(s)), allow=(ESTATE,))
        return s.value, rc

    def set_jet_source(self, dEdx, sigma, x0, y0, z0):
        self._chk(self.lib.mfo_set_jet_source(self.h, dEdx, sigma, x0, y0, z0))

    def set_eos_table(self, tb):
        """tb: dict(ln_e0, dln_e, n0, dn, ln_p) with ln_p of shape (nn, ne) (see workloads.crossover_eos_table)."""
        ln_p = _f64(tb["ln_p"])
        nn, ne = (1, ln_p.size) if ln_p.ndim == 1 else ln_p.shape
        self._chk(self.lib.mfo_set_eos_table(self.h, ne, nn, tb["ln_e0"], tb["dln_e"], tb.get("n0", 0.0), tb.get("dn", 1.0), _p(ln_p)))

    def eos(self, e, n=0.0):
        out = np.empty(3)
        self._chk(self.lib.mfo_eos(self.h, float(e), float(n), _p(out)))
        return out

    def status(self):
        return self.lib.mfo_sync(self.h)

    # ---- pieces ----
    def flux(self, d, U):
        U = _f64(U, 5)
        F = np.empty(5)
        self._chk(self.lib.mfo_flux(self.h, d, _p(U), _p(F)))
        return F

    def con2prim(self, U):
        U = _f64(U, 5)
        P = np.empty(5)
        self._chk(self.lib.mfo_con2prim(self.h, _p(U), _p(P)))
        return P

    def prim2con(self, P):
        P = _f64(P, 5)
        U = np.empty(5)
        self._chk(self.lib.mfo_prim2con(self.h, _p(P), _p(U)))
        return U

    def musta_flux(self, d, lam, UL, UR):
        UL, UR = _f64(UL, 5), _f64(UR, 5)
        F = np.empty(5)
        self._chk(self.lib.mfo_musta_flux(self.h, d, float(lam), _p(UL), _p(UR), _p(F)))
        return F

    def eval_L(self, dt):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self.lib.mfo_eval_L(self.h, float(dt), *[_p(x) for x in out]))
        return out

    def eval_faces(self, dt, d, side):
        out = np.empty((5,) + self.shape)
        self._chk(self.lib.mfo_eval_faces(self.h, float(dt), d, side, _p(out)))
        return out


def slope(limiter, a, b, omp=False):
    lim = LIM[limiter] if isinstance(limiter, str) else int(limiter)
    return _load(omp).mfo_slope(lim, float(a), float(b))


def num_threads(omp=False):
    return _load(omp).mfo_num_threads()
