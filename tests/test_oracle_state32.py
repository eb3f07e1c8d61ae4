"""Pins for the oracle's single-precision STATE mode ("The state of the system is saved as
5 single precision floating-point numbers per lattice cell"; reading A19: every stored state value - the state handed in and
the result of every Runge-Kutta stage - is rounded to float, the arithmetic between a load and the next store stays double).  CPU only.

What fixes the mode independently of its own code: (i) the stored values are floats; (ii) one step is the composition, written out
here with numpy's float32 rounding, of the 64-bit oracle's own spatial operator (mfo_eval_L, pinned elsewhere) and Eq.6 / Eq.7;
(iii) a uniform state is a fixed point; (iv) conservation and the distance to the 64-bit run are at single-precision round-off,
neither better (the rounding is really applied) nor worse (it is applied to the state only)."""
import numpy as np
import pytest

from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w

F32 = lambda a: np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)


def _pair(st, **over):
    nz, ny, nx = st["shape"]
    kw = dict(st["scheme"])
    kw.update(over)
    o32 = Oracle(nx, ny, nz, dx=st["dx"], state_bits=32, **kw)
    o64 = Oracle(nx, ny, nz, dx=st["dx"], **kw)
    for o in (o32, o64):
        o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    return o32, o64


def test_stored_state_is_single_precision():
    st = w.lumpy_event(shape=(8, 10, 12), dx=0.2, n_gauss=4, radius=0.8, half_z=0.5, background=0.5)
    o32, o64 = _pair(st)
    for a, b in zip(o32.get_state(), (st["E"], st["Mx"], st["My"], st["Mz"], st["R"])):
        assert np.array_equal(a, F32(b))                               # the state handed in is rounded once
    o32.step(3, 0.3)
    U = o32.get_state()
    assert all(np.array_equal(a, F32(a)) for a in U)
    o64.step(3, 0.3)
    assert not np.array_equal(o64.get_state()[0], F32(o64.get_state()[0]))   # the 64-bit run does not happen to be float-valued


@pytest.mark.parametrize("rk", [2, 3])
@pytest.mark.parametrize("predictor", [True, False])
def test_one_step_is_eq6_eq7_with_float_rounding_of_every_stage(rk, predictor):
    """U1 = f32(U + dt L(U)); RK2: U' = f32((U + U1 + dt L(U1))/2); RK3: U2 = f32(3/4 U + 1/4 U1 + 1/4 dt L(U1)),
    U' = f32(1/3 U + 2/3 U2 + 2/3 dt L(U2)) (Eq.6, Eq.7), with L taken from a 64-bit oracle context."""
    st = w.lumpy_event(shape=(6, 7, 9), dx=0.2, n_gauss=4, radius=0.6, half_z=0.4, background=0.5)
    kw = dict(limiter="mc", k_stages=2, rk=rk, bc="periodic", predictor=predictor)
    o32, oL = _pair(st, **kw)
    dt = 0.02

    def L(U):
        oL.set_state(*U)
        return [np.asarray(a) for a in oL.eval_L(dt)]

    U0 = [F32(st[k]) for k in ("E", "Mx", "My", "Mz", "R")]
    U1 = [F32(u + dt * l) for u, l in zip(U0, L(U0))]
    if rk == 2:
        want = [F32(0.5 * (u + u1 + dt * l)) for u, u1, l in zip(U0, U1, L(U1))]
    else:
        U2 = [F32(0.75 * u + 0.25 * u1 + (0.25 * dt) * l) for u, u1, l in zip(U0, U1, L(U1))]
        want = [F32((1.0 / 3.0) * u + (2.0 / 3.0) * u2 + ((2.0 / 3.0) * dt) * l) for u, u2, l in zip(U0, U2, L(U2))]
    o32.step_dt(1, dt)
    for a, b in zip(o32.get_state(), want):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("rk", [2, 3])
def test_uniform_state_is_a_fixed_point(rk):
    o = Oracle(8, 6, 5, dx=0.1, limiter="superbee", k_stages=3, rk=rk, bc="periodic", state_bits=32)
    shape = (5, 6, 8)
    full = lambda c: np.full(shape, c)
    o.set_state_prim(full(2.0), full(0.3), full(-0.2), full(0.5), full(1.5))
    before = o.get_state()
    o.step(5, 0.3)
    for a, b in zip(o.get_state(), before):
        assert np.array_equal(a, b)


def test_conservation_and_distance_to_the_64_bit_run_are_at_float_round_off():
    """Config-3-like periodic hot spot, 100 steps: total E drifts by single-precision round-off of the state (each cell's stored value is
    off by <= 2^-24 relative, the errors are unbiased), and the state stays within ~1e-6 of the 64-bit run - but not closer than 1e-9,
    or the rounding would not be there."""
    st = w.gaussian_hot_spot(shape=(20, 18, 22), dx=0.2)
    o32, o64 = _pair(st)
    t0 = o32.totals()
    o32.step(100, st["cfl"])
    o64.step(100, st["cfl"])
    t1 = o32.totals()
    assert abs(t1[0] - t0[0]) / t0[0] < 2e-6
    assert abs(t1[4] - t0[4]) / t0[4] < 2e-6
    a, b = o32.get_state(), o64.get_state()
    rel = max(np.abs(x - y).max() for x, y in zip(a, b)) / np.abs(b[0]).max()
    assert 1e-9 < rel < 5e-6, rel
    assert o32.time()[0] == pytest.approx(o64.time()[0], rel=1e-6)


def test_precision_argument_is_checked():
    o = Oracle(8, dx=0.1)
    assert o.lib.mfo_set_state_precision(o.h, 16) != 0
    assert o.lib.mfo_set_state_precision(o.h, 32) == 0
    assert o.lib.mfo_set_state_precision(o.h, 64) == 0
