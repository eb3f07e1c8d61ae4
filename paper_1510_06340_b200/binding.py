"""Thin ctypes binding over the C-ABI library (include/mustaforce.h): same names, argument marshalling only.

Every step of the path runs in the CUDA kernels of libmustaforce.so.  There is no CPU fallback: if the library
is missing it is built with nvcc, and if that or the GPU is missing the calls raise.  This module never imports
oracle/.
"""
import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))

MF_OK, MF_EINVAL, MF_ENOMEM, MF_ECUDA, MF_ESTATE = 0, -1, -2, -3, -4
MF_EOS_CS2, MF_EOS_TABLE = 0, 1
LIM = {"none": 0, "minmod": 1, "superbee": 2, "vanalbada": 3, "vanleer": 4, "mc": 5, "first": 6}
BC = {"outflow": 0, "periodic": 1}
PATH = {"auto": 0, "staged": 1, "fused": 2, "hybrid": 3, "sweep": 4, "small": 5}

_dp = C.POINTER(C.c_double)
_vp = C.c_void_p
_d5 = [_dp] * 5
_v5 = [_vp] * 5

# name -> (restype, argtypes); the list is checked against include/mustaforce.h by tests/test_abi.py
SIGNATURES = {
    "mf_create": (_vp, [C.c_int] * 3 + [C.c_double] + [C.c_int] * 3),
    "mf_create_batch": (_vp, [C.c_int] * 4 + [C.c_double] + [C.c_int] * 3),
    "mf_batch_size": (C.c_int, [_vp]),
    "mf_destroy": (None, [_vp]),
    "mf_set_state": (C.c_int, [_vp] + _d5),
    "mf_get_state": (C.c_int, [_vp] + _d5),
    "mf_set_state_async": (C.c_int, [_vp] + _d5),
    "mf_get_state_async": (C.c_int, [_vp] + _d5),
    "mf_set_state_device": (C.c_int, [_vp] + _v5),
    "mf_get_state_device": (C.c_int, [_vp] + _v5),
    "mf_set_state_prim": (C.c_int, [_vp] + _d5),
    "mf_get_state_prim": (C.c_int, [_vp] + _d5),
    "mf_step": (C.c_int, [_vp, C.c_int, C.c_double]),
    "mf_step_dt": (C.c_int, [_vp, C.c_int, C.c_double]),
    "mf_conserved_totals": (C.c_int, [_vp, _dp]),
    "mf_conserved_totals_event": (C.c_int, [_vp, C.c_int, _dp]),
    "mf_get_time": (C.c_int, [_vp, _dp, _dp, C.POINTER(C.c_longlong)]),
    "mf_get_time_event": (C.c_int, [_vp, C.c_int, _dp, _dp, C.POINTER(C.c_longlong)]),
    "mf_max_signal_speed": (C.c_int, [_vp, _dp]),
    "mf_set_rk": (C.c_int, [_vp, C.c_int]),
    "mf_set_boundary": (C.c_int, [_vp, C.c_int]),
    "mf_set_cs2": (C.c_int, [_vp, C.c_double]),
    "mf_set_eos_table": (C.c_int, [_vp, C.c_int, C.c_int] + [C.c_double] * 4 + [_dp]),
    "mf_set_predictor": (C.c_int, [_vp, C.c_int]),
    "mf_set_alpha": (C.c_int, [_vp, C.c_double]),
    "mf_set_jet_source": (C.c_int, [_vp] + [C.c_double] * 5),
    "mf_set_path": (C.c_int, [_vp, C.c_int]),
    "mf_get_path": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "mf_set_low_storage": (C.c_int, [_vp, C.c_int]),
    "mf_set_state_precision": (C.c_int, [_vp, C.c_int]),
    "mf_get_state_precision": (C.c_int, [_vp, C.POINTER(C.c_int)]),
    "mf_set_graph": (C.c_int, [_vp, C.c_int]),
    "mf_graph_stats": (C.c_int, [_vp, C.POINTER(C.c_longlong), C.POINTER(C.c_longlong)]),
    "mf_memory_bytes": (C.c_int, [_vp, C.POINTER(C.c_longlong)]),
    "mf_set_stream": (C.c_int, [_vp, _vp]),
    "mf_sync": (C.c_int, [_vp]),
    "mf_last_error": (C.c_char_p, [_vp]),
    "mf_eval_L": (C.c_int, [_vp, C.c_double] + _d5),
    "mf_launch_count": (C.c_int, [_vp, C.POINTER(C.c_longlong)]),
    "mf_profile": (C.c_int, [_vp, C.c_int]),
    "mf_profile_read": (C.c_int, [_vp, _dp, C.POINTER(C.c_longlong)]),
    "mf_probe_fp64": (C.c_int, [_dp]),
    "mf_totals_static": (C.c_int, [C.c_void_p] * 5 + [C.c_longlong, C.c_double, C.c_void_p, C.c_void_p]),
    "mf_static_last_error": (C.c_char_p, []),
    "mf_version": (C.c_char_p, []),
}

_libs = {}


class MustaForceError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__("mustaforce error %d: %s" % (code, msg))
        self.code = code


def load(strict=False):
    """dlopen the in-tree library (building it with nvcc first if it is missing or stale)."""
    if strict in _libs:
        return _libs[strict]
    from . import build as _build
    lib_path, strict_path = _build.build(strict=strict)
    lib = C.CDLL(strict_path if strict else lib_path)
    for name, (res, args) in SIGNATURES.items():
        f = getattr(lib, name)
        f.restype, f.argtypes = res, args
    _libs[strict] = lib
    return lib


def _p(a):
    return a.ctypes.data_as(_dp)


def _f64(a, n):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.size != n:
        raise ValueError("array has %d elements, expected %d" % (a.size, n))
    return a


def probe_fp64(strict=False):
    out = np.zeros(8)
    rc = load(strict).mf_probe_fp64(_p(out))
    if rc != MF_OK:
        raise MustaForceError(rc, "mf_probe_fp64 failed (no GPU?)")
    return dict(dfma_per_s=out[0], dadd_per_s=out[1], dmul_per_s=out[2], rcp_per_s=out[3], sqrt_per_s=out[4],
                sm_clock_hz=out[5], sms=int(out[6]), dfma3_per_s=out[7])


def totals_static(device_ptrs, ncells, scale, out_ptr, stream=None, strict=False):
    """mf_totals_static: allocation-free conserved totals of five DEVICE arrays (integers such as torch's data_ptr()) into the device
    array out_ptr (5 doubles), on `stream` (a cudaStream_t as int, None = default stream).  Argument marshalling only."""
    lib = load(strict)
    rc = lib.mf_totals_static(*[C.c_void_p(int(p)) for p in device_ptrs], int(ncells), float(scale), C.c_void_p(int(out_ptr)),
                              C.c_void_p(int(stream)) if stream else None)
    if rc != MF_OK:
        raise MustaForceError(rc, lib.mf_static_last_error().decode())
    return rc


def version(strict=False):
    return load(strict).mf_version().decode()


class MustaForce:
    """One mf_ctx.  Host arrays are numpy float64, shape (nz, ny, nx) or flat, x fastest; with batch=B (mf_create_batch: B independent
    events stepped by the same launches, each on its own clock) every array has shape (B, nz, ny, nx)."""

    def __init__(self, nx, ny=1, nz=1, dx=1.0, limiter="minmod", k_stages=2, rk=2, bc="outflow", predictor=True,
                 alpha=None, cs2=None, path="auto", stream=None, strict=False, eos_table=None, batch=None, state_bits=64):
        self.lib = load(strict)
        self.batch = batch
        self.shape = (nz, ny, nx) if batch is None else (int(batch), nz, ny, nx)
        self.n = nx * ny * nz * (1 if batch is None else int(batch))
        lim = LIM[limiter] if isinstance(limiter, str) else int(limiter)
        eos = MF_EOS_CS2 if eos_table is None else MF_EOS_TABLE
        if batch is None:
            self.h = self.lib.mf_create(nx, ny, nz, float(dx), eos, lim, int(k_stages))
        else:
            self.h = self.lib.mf_create_batch(int(batch), nx, ny, nz, float(dx), eos, lim, int(k_stages))
        if not self.h:
            raise MustaForceError(MF_EINVAL, self.lib.mf_last_error(None).decode())
        self._chk(self.lib.mf_set_rk(self.h, int(rk)))
        self._chk(self.lib.mf_set_boundary(self.h, BC[bc] if isinstance(bc, str) else int(bc)))
        self._chk(self.lib.mf_set_predictor(self.h, 1 if predictor else 0))
        if alpha is not None:
            self._chk(self.lib.mf_set_alpha(self.h, float(alpha)))
        if cs2 is not None:
            self._chk(self.lib.mf_set_cs2(self.h, float(cs2)))
        self._chk(self.lib.mf_set_path(self.h, PATH[path] if isinstance(path, str) else int(path)))
        if stream is not None:
            self.set_stream(stream)
        if eos_table is not None:
            self.set_eos_table(eos_table)
        if state_bits != 64:
            self.set_state_precision(state_bits)

    def _chk(self, rc, allow=()):
        if rc != MF_OK and rc not in allow:
            raise MustaForceError(rc, self.lib.mf_last_error(self.h).decode())
        return rc

    def close(self):
        if getattr(self, "h", None):
            self.lib.mf_destroy(self.h)
            self.h = None

    __del__ = close

    # ---- state
    def set_state(self, E, Mx, My, Mz, R):
        a = [_f64(x, self.n) for x in (E, Mx, My, Mz, R)]
        self._chk(self.lib.mf_set_state(self.h, *[_p(x) for x in a]))

    def get_state(self, out=None):
        out = out if out is not None else [np.empty(self.shape) for _ in range(5)]
        rc = self._chk(self.lib.mf_get_state(self.h, *[_p(x) for x in out]), allow=(MF_ESTATE,))
        self.last_status = rc
        return out

    def set_state_device(self, ptrs):
        """ptrs: five device addresses (ints), e.g. torch tensors' data_ptr()."""
        self._chk(self.lib.mf_set_state_device(self.h, *[C.c_void_p(int(p)) for p in ptrs]))

    def get_state_device(self, ptrs):
        return self._chk(self.lib.mf_get_state_device(self.h, *[C.c_void_p(int(p)) for p in ptrs]), allow=(MF_ESTATE,))

    def set_state_prim(self, e, vx, vy, vz, n):
        a = [_f64(x, self.n) for x in (e, vx, vy, vz, n)]
        self._chk(self.lib.mf_set_state_prim(self.h, *[_p(x) for x in a]))

    def get_state_prim(self):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self.lib.mf_get_state_prim(self.h, *[_p(x) for x in out]), allow=(MF_ESTATE,))
        return out

    # ---- stepping
    def step(self, n, cfl):
        self._chk(self.lib.mf_step(self.h, int(n), float(cfl)))

    def step_dt(self, n, dt):
        self._chk(self.lib.mf_step_dt(self.h, int(n), float(dt)))

    def sync(self):
        return self._chk(self.lib.mf_sync(self.h), allow=(MF_ESTATE,))

    def totals(self, event=None):
        out = np.empty(5)
        if event is None:
            self._chk(self.lib.mf_conserved_totals(self.h, _p(out)), allow=(MF_ESTATE,))
        else:
            self._chk(self.lib.mf_conserved_totals_event(self.h, int(event), _p(out)), allow=(MF_ESTATE,))
        return out

    def time(self, event=0):
        t, dt, s = C.c_double(), C.c_double(), C.c_longlong()
        self._chk(self.lib.mf_get_time_event(self.h, int(event), C.byref(t), C.byref(dt), C.byref(s)), allow=(MF_ESTATE,))
        return t.value, dt.value, s.value

    def batch_size(self):
        return self.lib.mf_batch_size(self.h)

    def max_signal_speed(self):
        s = C.c_double()
        rc = self._chk(self.lib.mf_max_signal_speed(self.h, C.byref(s)), allow=(MF_ESTATE,))
        return s.value, rc

    def eval_L(self, dt):
        out = [np.empty(self.shape) for _ in range(5)]
        self._chk(self.lib.mf_eval_L(self.h, float(dt), *[_p(x) for x in out]))
        return out

    # ---- options
    def set_jet_source(self, dEdx, sigma, x0, y0, z0):
        self._chk(self.lib.mf_set_jet_source(self.h, dEdx, sigma, x0, y0, z0))

    def set_eos_table(self, tb):
        """tb: dict(ln_e0, dln_e, n0, dn, ln_p) with ln_p of shape (nn, ne), e.g. workloads.crossover_eos_table()."""
        ln_p = np.ascontiguousarray(tb["ln_p"], dtype=np.float64)
        nn, ne = (1, ln_p.size) if ln_p.ndim == 1 else ln_p.shape
        self._chk(self.lib.mf_set_eos_table(self.h, ne, nn, float(tb["ln_e0"]), float(tb["dln_e"]), float(tb.get("n0", 0.0)),
                                            float(tb.get("dn", 1.0)), _p(ln_p)))

    def set_state_async(self, E, Mx, My, Mz, R):
        """No synchronisation: the five float64 arrays (pinned, contiguous, of the context's size) must stay alive and untouched until sync()."""
        for x in (E, Mx, My, Mz, R):
            if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"] or x.size != self.n:
                raise ValueError("set_state_async needs contiguous float64 arrays of %d elements (no copy can be made here)" % self.n)
        self._chk(self.lib.mf_set_state_async(self.h, *[_p(x) for x in (E, Mx, My, Mz, R)]))

    def get_state_async(self, out):
        """Enqueue the copy of the state into the five (pinned) float64 arrays `out`; they are complete after sync()."""
        for x in out:
            if x.dtype != np.float64 or not x.flags["C_CONTIGUOUS"] or x.size != self.n:
                raise ValueError("get_state_async needs contiguous float64 arrays of %d elements" % self.n)
        self._chk(self.lib.mf_get_state_async(self.h, *[_p(x) for x in out]))

    def set_stream(self, stream):
        """stream: a raw cudaStream_t as int (e.g. torch.cuda.current_stream().cuda_stream); 0/None = own stream."""
        self._chk(self.lib.mf_set_stream(self.h, C.c_void_p(int(stream) if stream else None)))

    def set_path(self, path):
        self._chk(self.lib.mf_set_path(self.h, PATH[path] if isinstance(path, str) else int(path)))

    def set_low_storage(self, on):
        self._chk(self.lib.mf_set_low_storage(self.h, 1 if on else 0))

    def set_state_precision(self, bits):
        self._chk(self.lib.mf_set_state_precision(self.h, int(bits)))

    def state_precision(self):
        b = C.c_int()
        self._chk(self.lib.mf_get_state_precision(self.h, C.byref(b)))
        return b.value

    def set_graph(self, on):
        self._chk(self.lib.mf_set_graph(self.h, 1 if on else 0))

    def graph_stats(self):
        cap, rep = C.c_longlong(), C.c_longlong()
        self._chk(self.lib.mf_graph_stats(self.h, C.byref(cap), C.byref(rep)))
        return cap.value, rep.value

    def memory_bytes(self):
        b = C.c_longlong()
        self._chk(self.lib.mf_memory_bytes(self.h, C.byref(b)))
        return b.value

    def path(self):
        p = C.c_int()
        self._chk(self.lib.mf_get_path(self.h, C.byref(p)))
        return {v: k for k, v in PATH.items()}[p.value]

    def profile(self, on):
        self._chk(self.lib.mf_profile(self.h, 1 if on else 0))

    def profile_read(self):
        """{class name: (milliseconds, event-bracketed launch groups)} since the last read."""
        ms = np.zeros(8)
        cnt = (C.c_longlong * 8)()
        self._chk(self.lib.mf_profile_read(self.h, _p(ms), cnt))
        names = ["cfl", "cell_stage", "flux_stage", "combine", "fused_stage", "scalars", "_6", "_7"]
        return {names[i]: (float(ms[i]), int(cnt[i])) for i in range(8) if cnt[i]}

    def launch_count(self):
        n = C.c_longlong()
        self._chk(self.lib.mf_launch_count(self.h, C.byref(n)))
        return n.value
