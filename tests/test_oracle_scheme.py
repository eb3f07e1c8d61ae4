"""Pins for the oracle's scheme as a whole: exact Riemann solution under
refinement (Q1), conservation (Q2), uniform state (Q3), axis permutation (Q4), limiter / k ordering (Q8),
numpy transcription on tiny inputs (Q9), jet-source budget (Q10), convergence order on exact linear
advection of the charge, and bit-identity of the OpenMP build.  CPU only."""
import itertools
import os

import numpy as np
import pytest

import exact_riemann
import np_transcription as npt
from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads

GOLD = os.path.join(os.path.dirname(__file__), "golden", "riemann_p_e3.txt")


def run_to(o, dx, t_end, cfl):
    """Config-1 driver: mf_step(1,cfl) until t+dt > t_end, then mf_step_dt(1, t_end-t)."""
    while True:
        t = o.time()[0]
        if t >= t_end - 1e-12:
            return
        smax, _ = o.max_signal_speed()
        dt = cfl * dx / smax
        if t + dt > t_end:
            o.step_dt(1, t_end - t)
        else:
            o.step(1, cfl)


def shock_tube_l1(nx, limiter="minmod", k=2, rk=2, predictor=True, cfl=0.4, fixed_lambda=None):
    st = workloads.shock_tube_1d(nx=nx)
    dx = st["dx"]
    o = Oracle(nx, dx=dx, limiter=limiter, k_stages=k, rk=rk, predictor=predictor)
    o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    if fixed_lambda is None:
        run_to(o, dx, 12.0, cfl)
    else:
        nsteps = int(round(12.0 / (fixed_lambda * dx)))
        o.step_dt(nsteps, 12.0 / nsteps)
    assert o.time()[0] == pytest.approx(12.0, abs=1e-9)
    e, vx, _, _, n = [a.ravel() for a in o.get_state_prim()]
    x = workloads.centres(nx, dx)
    ee, ve, ne = exact_riemann.exact(x / 12.0, 10.0, 1.0, 10.0, 1.0)
    return dx * np.abs(e - ee).sum(), dx * np.abs(vx - ve).sum(), dx * np.abs(n - ne).sum()


# ---------------------------------------------------------------- Q1
def test_exact_solver_reproduces_fixture_and_rankine_hugoniot():
    gold = {}
    for line in open(GOLD):
        if line.strip() and not line.startswith("#"):
            key, val = line.split()
            gold[key] = float(val)
    lm = exact_riemann.landmarks(10.0, 1.0)
    for key, val in gold.items():
        assert lm[key] == pytest.approx(val, rel=2e-14), key
    # lab-frame Rankine-Hugoniot: v_sh [U] = [F] for energy and momentum, p = e/3
    def cons(e, v):
        g2 = 1 / (1 - v * v)
        w = e * 4 / 3 * g2
        return np.array([w - e / 3, w * v]), np.array([w * v, w * v * v + e / 3])
    U2, F2 = cons(gold["e_star"], gold["v_star"])
    U1, F1 = cons(1.0, 0.0)
    assert np.all(np.abs(gold["v_shock"] * (U2 - U1) - (F2 - F1)) < 1e-13)


@pytest.mark.parametrize("predictor", [True, False])
def test_shock_tube_converges_to_exact_solution(predictor):
    """Config 1 (minmod, k=2, RK2, cfl 0.4): L1 error at t=12 shrinks under refinement 200->400->800->1600."""
    errs = [shock_tube_l1(n, predictor=predictor) for n in (200, 400, 800, 1600)]
    for prev, cur in zip(errs, errs[1:]):
        for q in range(3):
            assert cur[q] / prev[q] <= 0.70, (errs, q)
    e400 = errs[1]
    if predictor:
        assert e400[0] <= 2.0 and e400[1] <= 0.25 and e400[2] <= 2.4
    else:
        assert e400[0] <= 1.2 and e400[1] <= 0.15


def test_star_state_plateau_matches_exact_values():
    """Between contact and shock the numerical plateau sits on (e*, v*) and n on n*_R."""
    nx = 1600
    st = workloads.shock_tube_1d(nx=nx)
    o = Oracle(nx, dx=st["dx"], limiter="minmod", k_stages=2, rk=2)
    o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    run_to(o, st["dx"], 12.0, 0.4)
    e, vx, _, _, n = [a.ravel() for a in o.get_state_prim()]
    x = workloads.centres(nx, st["dx"])
    lm = exact_riemann.landmarks(10.0, 1.0)
    mid = np.abs(x - 0.5 * 12 * (lm["v_star"] + lm["v_shock"])).argmin()
    assert e[mid] == pytest.approx(lm["e_star"], rel=2e-3)
    assert vx[mid] == pytest.approx(lm["v_star"], rel=2e-3)
    assert n[mid] == pytest.approx(lm["nR_star_over_nR"], rel=5e-3)
    left = np.abs(x - 0.5 * 12 * (lm["xi_tail"] + lm["v_star"])).argmin()
    assert n[left] == pytest.approx(10 * lm["nL_star_over_nL"], rel=5e-3)


# ---------------------------------------------------------------- Q8
def test_limiter_and_stage_ordering():
    """Minbee most diffusive, Superbee sharpest; more MUSTA stages reduce the error (fixed lambda)."""
    e_mm = shock_tube_l1(400, "minmod", predictor=False, fixed_lambda=0.4)[0]
    e_mc = shock_tube_l1(400, "mc", predictor=False, fixed_lambda=0.4)[0]
    e_sb = shock_tube_l1(400, "superbee", predictor=False, fixed_lambda=0.4)[0]
    assert e_mm > e_mc > e_sb
    by_k = [shock_tube_l1(400, "minmod", k=k)[0] for k in range(4)]
    assert by_k[0] > by_k[1] > by_k[2] > by_k[3]


# ---------------------------------------------------------------- Q3
@pytest.mark.parametrize("limiter,k,rk,bc", [("minmod", 2, 2, "outflow"), ("superbee", 3, 3, "periodic"),
                                            ("vanalbada", 4, 3, "outflow"), ("none", 1, 2, "periodic"),
                                            ("mc", 2, 2, "periodic"), ("vanleer", 0, 3, "outflow")])
@pytest.mark.parametrize("moving", [False, True])
def test_uniform_state_is_a_fixed_point(limiter, k, rk, bc, moving):
    shape = (5, 6, 7)
    n = int(np.prod(shape))
    o = Oracle(shape[2], shape[1], shape[0], dx=0.1, limiter=limiter, k_stages=k, rk=rk, bc=bc)
    v = (0.3, -0.2, 0.5) if moving else (0.0, 0.0, 0.0)
    o.set_state_prim(np.full(n, 2.0), np.full(n, v[0]), np.full(n, v[1]), np.full(n, v[2]), np.full(n, 1.5))
    before = o.get_state()
    o.step(3, 0.3)
    after = o.get_state()
    for b, a in zip(before, after):
        if rk == 2:
            assert np.array_equal(a, b)
        else:
            assert np.allclose(a, b, rtol=3 * 4 * 2.3e-16, atol=0)      # <= 4 ulp per step (convex sums round)


# ---------------------------------------------------------------- Q2
def test_conservation_on_periodic_box():
    st = workloads.gaussian_hot_spot(shape=(12, 14, 16), dx=0.4)
    nz, ny, nx = st["shape"]
    o = Oracle(nx, ny, nz, dx=st["dx"], limiter="superbee", k_stages=3, rk=3, bc="periodic")
    o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    t0 = o.totals()
    o.step(40, 0.3)
    t1 = o.totals()
    assert abs(t1[0] - t0[0]) / t0[0] <= 1e-13
    assert abs(t1[4] - t0[4]) / t0[4] <= 1e-13
    for q in (1, 2, 3):
        assert abs(t1[q]) / t0[0] <= 1e-13
    E = o.get_state()[0]
    assert np.abs(E - st["E"]).max() > 0.05               # it did evolve


def test_totals_are_cell_sums_times_volume():
    st = workloads.lumpy_event(shape=(6, 5, 4), dx=0.5, n_gauss=3)
    o = Oracle(4, 5, 6, dx=0.5)
    o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    assert o.totals()[0] == pytest.approx(st["E"].sum() * 0.125, rel=1e-14)
    assert o.totals()[4] == pytest.approx(st["R"].sum() * 0.125, rel=1e-14)


# ---------------------------------------------------------------- Q4
def _lumpy_moving(shape, seed):
    rng = np.random.default_rng(seed)
    st = workloads.lumpy_event(shape=shape, dx=0.4, n_gauss=5, radius=1.5, half_z=1.0, background=1.0)
    e = st["E"]
    v = [0.3 * np.sin(0.7 * e), 0.2 * np.cos(0.4 * e), -0.25 * np.sin(0.3 * e + 1)]
    return e, v, 1.0 + rng.uniform(size=e.shape)


@pytest.mark.parametrize("perm", [(1, 0, 2), (2, 1, 0), (1, 2, 0)])
def test_axis_permutation_symmetry(perm):
    """Permuting (x,y,z) of the data together with (Mx,My,Mz) permutes the result (<= 1e-13 relative)."""
    shape = (6, 7, 8)                                            # (nz, ny, nx)
    e, v, n = _lumpy_moving(shape, 11)
    kw = dict(dx=0.4, limiter="vanleer", k_stages=2, rk=3, bc="periodic")
    a = Oracle(shape[2], shape[1], shape[0], **kw)
    a.set_state_prim(e, v[0], v[1], v[2], n)
    a.step_dt(5, 0.08)
    ref = a.get_state()
    # new axis d' takes old axis perm[d'];  numpy axes are (z,y,x) = 2-d
    np_axes = tuple(2 - perm[2 - ax] for ax in range(3))
    tr = lambda f: np.ascontiguousarray(np.transpose(f, np_axes))
    e2, n2 = tr(e), tr(n)
    v2 = [tr(v[perm[d]]) for d in range(3)]
    s2 = e2.shape
    b = Oracle(s2[2], s2[1], s2[0], **kw)
    b.set_state_prim(e2, v2[0], v2[1], v2[2], n2)
    b.step_dt(5, 0.08)
    got = b.get_state()
    scale = np.abs(ref[0]).max()
    assert np.abs(got[0] - tr(ref[0])).max() <= 1e-13 * scale
    assert np.abs(got[4] - tr(ref[4])).max() <= 1e-13 * scale
    for d in range(3):
        assert np.abs(got[1 + d] - tr(ref[1 + perm[d]])).max() <= 1e-13 * scale


@pytest.mark.parametrize("axis", [1, 2])
def test_1d_problem_embedded_in_3d(axis):
    """1D data along y or z of a 3D grid with alpha=1 reproduces the 1D run along x."""
    st = workloads.shock_tube_1d(nx=48, length=4.8)
    kw = dict(dx=st["dx"], limiter="mc", k_stages=2, rk=2, bc="outflow")
    a = Oracle(48, **kw)
    a.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    a.step_dt(20, 0.03)
    ref = [f.ravel() for f in a.get_state()]
    dims = [5, 5, 5]
    dims[axis] = 48
    b = Oracle(dims[0], dims[1], dims[2], alpha=1.0, **kw)
    shp = (dims[2], dims[1], dims[0])
    prof = [1, 1, 1]
    prof[2 - axis] = 48
    E = np.broadcast_to(st["E"].reshape(prof), shp)
    R = np.broadcast_to(st["R"].reshape(prof), shp)
    z = np.zeros(shp)
    b.set_state(E, z, z, z, R)
    b.step_dt(20, 0.03)
    got = b.get_state()
    line = [slice(2, 3)] * 3
    line[2 - axis] = slice(None)
    assert np.abs(got[0][tuple(line)].ravel() - ref[0]).max() <= 1e-13 * 10
    assert np.abs(got[1 + axis][tuple(line)].ravel() - ref[1]).max() <= 1e-13 * 10
    assert np.abs(got[4][tuple(line)].ravel() - ref[4]).max() <= 1e-13 * 10
    other = [q for q in (1, 2, 3) if q != 1 + axis]
    for q in other:
        assert np.abs(got[q]).max() <= 1e-13


# ---------------------------------------------------------------- Q9
CASES = list(itertools.product(["minmod", "superbee", "vanalbada", "vanleer", "mc", "none", "first"], [True, False]))


@pytest.mark.parametrize("limiter,predictor", CASES)
def test_L_matches_numpy_transcription_1d(limiter, predictor):
    rng = np.random.default_rng(21)
    nx, dx, dt = 8, 0.1, 0.03
    e = 1 + 5 * rng.uniform(size=nx)
    v = 0.6 * (rng.uniform(size=nx) - 0.5)
    n = 1 + rng.uniform(size=nx)
    for bc in ("outflow", "periodic"):
        o = Oracle(nx, dx=dx, limiter=limiter, k_stages=2, bc=bc, predictor=predictor)
        o.set_state_prim(e, v, 0 * v, 0 * v, n)
        U = np.array(o.get_state())
        L = np.array(o.eval_L(dt))
        ref = npt.L_op(U, dt, dx, 2, limiter, predictor, 1.0, bc)
        assert np.abs(L - ref).max() <= 1e-13 * np.abs(ref).max()


@pytest.mark.parametrize("shape", [(4, 4, 4), (4, 5, 6), (1, 6, 5), (5, 1, 4)])
@pytest.mark.parametrize("bc", ["outflow", "periodic"])
def test_step_matches_numpy_transcription_3d(shape, bc):
    rng = np.random.default_rng(22)
    nz, ny, nx = shape
    e = 1 + 5 * rng.uniform(size=shape)
    v = [0.5 * (rng.uniform(size=shape) - 0.5) for _ in range(3)]
    n = 1 + rng.uniform(size=shape)
    alpha = float(sum(s > 1 for s in shape))
    for limiter, k, rk, predictor in (("mc", 2, 2, True), ("superbee", 3, 3, True), ("minmod", 1, 3, False)):
        o = Oracle(nx, ny, nz, dx=0.1, limiter=limiter, k_stages=k, rk=rk, bc=bc, predictor=predictor)
        o.set_state_prim(e, v[0], v[1], v[2], n)
        U = np.array(o.get_state())
        smax, _ = o.max_signal_speed()
        assert smax == pytest.approx(npt.smax(U), rel=1e-15)
        o.step(1, 0.3)
        dt = o.time()[1]
        assert dt == pytest.approx(0.3 * 0.1 / smax, rel=1e-15)
        ref = npt.step(U, dt, 0.1, k, limiter, rk, predictor, alpha, bc)
        got = np.array(o.get_state())
        assert np.abs(got - ref).max() <= 1e-13 * np.abs(ref).max()


def test_guarded_states_match_transcription():
    """Near-vacuum / superluminal cells go through the A12 guard the same way in both."""
    rng = np.random.default_rng(23)
    shape = (4, 4, 6)
    U = np.zeros((5,) + shape)
    U[0] = 10 ** rng.uniform(-14, 0, size=shape)
    for q in (1, 2, 3):
        U[q] = U[0] * rng.uniform(-0.7, 0.7, size=shape)
    U[4] = 1.0
    o = Oracle(6, 4, 4, dx=0.1, limiter="minmod", k_stages=2, bc="outflow")
    o.set_state(*U)
    L = np.array(o.eval_L(0.02))
    ref = npt.L_op(U, 0.02, 0.1, 2, "minmod", True, 3.0, "outflow")
    assert np.all(np.isfinite(L))
    assert np.abs(L - ref).max() <= 1e-12 * np.abs(ref).max()


# ---------------------------------------------------------------- Q10
def test_jet_source_energy_budget():
    """Outflow box, wave far from the boundary: d/dt sum(E) dx^3 = d/dt sum(Mx) dx^3 = dE/dx (A14)."""
    n, dx = 24, 0.25
    o = Oracle(n, n, n, dx=dx, limiter="mc", k_stages=1, rk=3, bc="outflow")
    e = np.full((n, n, n), 1.0)
    z = np.zeros_like(e)
    o.set_state(e, z, z, z, e)
    o.set_jet_source(5.0, 0.35, -0.5, 0.0, 0.0)
    t0 = o.totals()
    o.step_dt(10, 0.05)
    t1 = o.totals()
    t = o.time()[0]
    assert t1[0] - t0[0] == pytest.approx(5.0 * t, rel=1e-8)
    assert t1[1] - t0[1] == pytest.approx(5.0 * t, rel=1e-8)
    assert abs(t1[2]) < 1e-12 and abs(t1[3]) < 1e-12
    assert t1[4] == pytest.approx(t0[4], rel=1e-10)            # only the far Gaussian tail reaches the outflow faces
    ref = np.array([e, z, z, z, e])
    for s in range(2):
        ref = npt.step(ref, 0.05, dx, 1, "mc", 3, True, 3.0, "outflow", t=0.05 * s, src=(5.0, 0.35, (-0.5, 0.0, 0.0)))
    o2 = Oracle(n, n, n, dx=dx, limiter="mc", k_stages=1, rk=3, bc="outflow")
    o2.set_state(e, z, z, z, e)
    o2.set_jet_source(5.0, 0.35, -0.5, 0.0, 0.0)
    o2.step_dt(2, 0.05)
    assert np.abs(np.array(o2.get_state()) - ref).max() <= 1e-13


# ---------------------------------------------------------------- exact linear advection of the charge
def _advection_error(nx, limiter, predictor, rk, diag3d=False):
    """Uniform (e, v), varying n: E, M stay uniform and R is advected exactly, R(x,t) = R0(x - v t)."""
    L, v0, t_end = 1.0, 0.5, 0.4
    dx = L / nx
    if diag3d:
        shape = (nx, nx, nx)
        x = workloads.centres(nx, dx)
        X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
        vv = (v0 / np.sqrt(3),) * 3
        prof = lambda t: 1 + 0.3 * np.sin(2 * np.pi * (X - vv[0] * t)) * np.sin(2 * np.pi * (Y - vv[1] * t)) * np.cos(2 * np.pi * (Z - vv[2] * t))
        o = Oracle(nx, nx, nx, dx=dx, limiter=limiter, k_stages=2, rk=rk, bc="periodic", predictor=predictor)
    else:
        shape = (1, 1, nx)
        x = workloads.centres(nx, dx).reshape(shape)
        vv = (v0, 0.0, 0.0)
        prof = lambda t: 1 + 0.3 * np.sin(2 * np.pi * (x - v0 * t))
        o = Oracle(nx, dx=dx, limiter=limiter, k_stages=2, rk=rk, bc="periodic", predictor=predictor)
    full = lambda c: np.full(shape, c)
    o.set_state_prim(full(2.0), full(vv[0]), full(vv[1]), full(vv[2]), prof(0.0))
    nsteps = int(round(t_end / (0.25 * dx)))
    o.step_dt(nsteps, t_end / nsteps)
    n = o.get_state_prim()[4]
    return np.abs(n - prof(t_end)).mean()


def test_second_order_convergence_on_linear_advection():
    """Eq.14 slopes + RK2 without the Hancock step are second order; first-order slopes are first order."""
    e = [_advection_error(n, "none", False, 2) for n in (32, 64, 128)]
    assert e[0] / e[1] > 3.6 and e[1] / e[2] > 3.6
    f = [_advection_error(n, "first", False, 2) for n in (32, 64, 128)]
    assert 1.6 < f[0] / f[1] < 2.4 and 1.6 < f[1] / f[2] < 2.4
    assert e[2] < 0.05 * f[2]


def test_advection_in_3d_along_the_diagonal_converges():
    e = [_advection_error(n, "none", False, 3, diag3d=True) for n in (8, 16)]
    assert e[0] / e[1] > 3.0


# ---------------------------------------------------------------- OpenMP build is the same oracle
@pytest.mark.parametrize("rk", [2, 3])
@pytest.mark.parametrize("k,predictor", [(0, False), (2, True)])
def test_runge_kutta_step_is_the_taylor_polynomial_of_a_linear_operator(rk, k, predictor):
    """Eq.6 / Eq.7 against what the mathematics fixes: for a LINEAR spatial operator the TVD RK2 step is
    (1 + z + z^2/2) U and the TVD RK3 step (1 + z + z^2/2 + z^3/6) U with z = dt L (their stability polynomials).  L is linear in the charge R
    when (e, v) are uniform (R is advected, flux v_d R) and the slope is the central one (Eq.14), whatever k and the half step do; powers of L
    are taken with mfo_eval_L on states whose R is the previous result.  A wrong coefficient anywhere in Eq.6 or Eq.7 changes the polynomial."""
    shape = (5, 6, 8)
    nz, ny, nx = shape
    dx, dt = 0.5, 0.12
    v = (0.3, -0.2, 0.25)
    full = lambda c: np.full(shape, c)
    rng = np.random.default_rng(3)
    kw = dict(dx=dx, limiter="none", k_stages=k, predictor=predictor, bc="periodic", rk=rk)
    o = Oracle(nx, ny, nz, **kw)
    o.set_state_prim(full(2.0), full(v[0]), full(v[1]), full(v[2]), 1.0 + rng.uniform(size=shape))
    E, Mx, My, Mz, R0 = o.get_state()

    def L(R):                                                             # the oracle's own spatial operator on (E, M, R)
        h = Oracle(nx, ny, nz, **kw)
        h.set_state(E, Mx, My, Mz, R)
        out = h.eval_L(dt)
        assert all(np.abs(out[q]).max() < 1e-13 for q in range(4))       # uniform E, M: nothing moves, so L acts on R alone
        return out[4]

    L1 = L(R0); L2 = L(L1); L3 = L(L2)
    assert np.allclose(L(2.0 * R0 - 0.5 * L1), 2.0 * L1 - 0.5 * L2, rtol=0, atol=1e-12 * np.abs(L1).max())    # L is linear indeed
    want = R0 + dt * L1 + 0.5 * dt ** 2 * L2 + ((dt ** 3 / 6.0) * L3 if rk == 3 else 0.0)
    o.step_dt(1, dt)
    got = o.get_state()[4]
    assert np.allclose(got, want, rtol=0, atol=1e-13 * np.abs(want).max())
    assert np.abs(got - (want + (dt ** 3 / 6.0) * L3 * (1 if rk == 2 else -1))).max() > 1e-8          # (and the orders differ measurably)


@pytest.mark.parametrize("shift", [(3, 0, 0), (0, -2, 0), (0, 0, 5), (1, 2, -3)])
def test_periodic_box_is_translation_invariant(shift):
    """Ghost cells of a periodic box are the cells modulo n on every axis (reading A11): shifting the initial data cyclically shifts the result,
    bit for bit (every cell runs the same arithmetic on the same numbers).  A wrap that is off by one on any side of any axis breaks it."""
    st = workloads.lumpy_event(shape=(7, 6, 9), dx=0.2, n_gauss=5, radius=0.6, half_z=0.4, background=0.5)
    nz, ny, nx = st["shape"]
    kw = dict(dx=st["dx"], limiter="mc", k_stages=2, rk=3, bc="periodic")
    F = ("E", "Mx", "My", "Mz", "R")
    a, b = Oracle(nx, ny, nz, **kw), Oracle(nx, ny, nz, **kw)
    roll = lambda x: np.roll(x, shift, axis=(0, 1, 2))                   # shift = (z, y, x)
    a.set_state(*[st[f] for f in F])
    b.set_state(*[np.ascontiguousarray(roll(st[f])) for f in F])
    a.step_dt(6, 0.02)
    b.step_dt(6, 0.02)
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.array_equal(roll(x), y)
    assert not np.array_equal(a.get_state()[0], st["E"])


@pytest.mark.parametrize("axis", [0, 1, 2])
def test_outflow_boundaries_are_mirror_symmetric(axis):
    """Outflow ghosts are the clamped index on both sides of every axis (A11): data that are mirror symmetric about the middle of an axis stay so,
    with the momentum component along that axis antisymmetric.  A clamp that treats the two ends differently breaks it."""
    st = workloads.lumpy_event(shape=(8, 6, 10), dx=0.2, n_gauss=5, radius=0.5, half_z=0.4, background=0.5)
    nz, ny, nx = st["shape"]
    npax = {0: 2, 1: 1, 2: 0}[axis]                                       # direction -> numpy axis of (nz, ny, nx)
    sym = lambda x: 0.5 * (x + np.flip(x, axis=npax))
    e = sym(st["E"])
    o = Oracle(nx, ny, nz, dx=st["dx"], limiter="superbee", k_stages=3, rk=3, bc="outflow")
    zero = np.zeros_like(e)
    o.set_state(e, zero, zero, zero, sym(st["R"]))
    o.step(12, 0.3)
    out = o.get_state()
    scale = np.abs(out[0]).max()
    for q, x in enumerate(out):
        sign = -1.0 if q == 1 + axis else 1.0
        assert np.abs(x - sign * np.flip(x, axis=npax)).max() <= 1e-13 * scale
    assert np.abs(out[1 + axis]).max() > 1e-3 * scale                    # something moved, and it reached the boundary cells
    edge = np.take(out[1 + axis], [0], axis=npax)
    assert np.abs(edge).max() > 0.0


def test_openmp_build_is_bit_identical():
    st = workloads.lumpy_event(shape=(10, 9, 12), dx=0.3, n_gauss=6, radius=1.2, half_z=1.0)
    out = []
    for omp in (False, True):
        o = Oracle(12, 9, 10, dx=0.3, limiter="superbee", k_stages=3, rk=3, bc="outflow", omp=omp)
        o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
        o.step(6, 0.3)
        out.append(np.array(o.get_state()))
    assert np.array_equal(out[0], out[1])
