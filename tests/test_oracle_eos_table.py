"""Pins for the oracle's tabulated equation of state and its Newton con2prim (A18).  CPU only.

* the table lookup against scipy's RegularGridInterpolator on (ln e, n) -> ln p (a library routine);
* a table of p = cs2*e must reproduce the closed-form path (lookup is exact for it; Newton must land on the closed-form root);
* Eq.4 -> Eq.23 round trip on a non-trivial table; the root against plain bisection written here;
* conservation, uniform state and a 1D shock tube against the closed-form run."""
import math

import numpy as np
import pytest
from scipy.interpolate import RegularGridInterpolator

from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w


@pytest.fixture(scope="module")
def cross():
    return w.crossover_eos_table()


def test_lookup_matches_library_interpolator(cross):
    o = Oracle(8, dx=1.0, eos_table=cross)
    nn, ne = cross["ln_p"].shape
    ln_e = cross["ln_e0"] + cross["dln_e"] * np.arange(ne)
    n = cross["n0"] + cross["dn"] * np.arange(nn)
    interp = RegularGridInterpolator((n, ln_e), cross["ln_p"], method="linear")
    rng = np.random.default_rng(1)
    for _ in range(2000):
        e = math.exp(rng.uniform(ln_e[0], ln_e[-1]))
        nv = rng.uniform(0, n[-1])
        p, p_e, p_n = o.eos(e, nv)
        assert p == pytest.approx(math.exp(interp([nv, math.log(e)])[0]), rel=1e-13)
        h = 1e-6                                                    # derivatives against central differences inside one cell
        pm, pp = o.eos(e * (1 - h), nv)[0], o.eos(e * (1 + h), nv)[0]
        assert p_e == pytest.approx((pp - pm) / (2 * h * e), rel=2e-4, abs=1e-9)
    # outside the n range the value is held, outside the e range ln p continues linearly in ln e
    assert o.eos(2.0, 50.0)[0] == pytest.approx(o.eos(2.0, n[-1])[0], rel=1e-14)
    e_hi = math.exp(ln_e[-1])
    slope = (cross["ln_p"][0, -1] - cross["ln_p"][0, -2]) / cross["dln_e"]
    assert o.eos(4 * e_hi, 0.0)[0] == pytest.approx(o.eos(e_hi, 0.0)[0] * 4 ** slope, rel=1e-12)


@pytest.mark.parametrize("nn", [1, 5])
@pytest.mark.parametrize("cs2", [1.0 / 3.0, 0.2])
def test_linear_table_reproduces_closed_form(cs2, nn):
    """ln p = ln cs2 + ln e is linear, so the table is exact and Newton must find the closed-form root of Eq.23."""
    tab = Oracle(8, dx=1.0, eos_table=w.linear_eos_table(cs2=cs2, nn=nn))
    ref = Oracle(8, dx=1.0, cs2=cs2)
    rng = np.random.default_rng(2)
    for _ in range(1000):
        e, n = 10 ** rng.uniform(-3, 2.5), 10 ** rng.uniform(-2, 1)
        v = rng.normal(size=3)
        v *= rng.choice([0.0, rng.uniform(0, 0.9), rng.uniform(0.9, 0.999)]) / np.linalg.norm(v)
        U = ref.prim2con([e, *v, n])
        assert np.allclose(tab.prim2con([e, *v, n]), U, rtol=1e-13)
        g2 = 1 / (1 - v @ v)
        assert np.allclose(tab.con2prim(U), ref.con2prim(U), rtol=1e-12 * g2, atol=1e-13 * g2)
        for d in range(3):
            assert np.allclose(tab.flux(d, U), ref.flux(d, U), rtol=1e-12 * g2, atol=1e-13 * g2 * U[0])


def test_round_trip_and_residual_on_crossover_table(cross):
    o = Oracle(8, dx=1.0, eos_table=cross)
    rng = np.random.default_rng(3)
    for _ in range(2000):
        e, n = 10 ** rng.uniform(-2, 2), rng.uniform(0, 10)
        v = rng.normal(size=3)
        vm = rng.choice([1e-9, rng.uniform(0, 0.9), rng.uniform(0.9, 0.995)])
        v *= vm / np.linalg.norm(v)
        U = o.prim2con([e, *v, n])
        back = o.con2prim(U)
        g2 = 1 / (1 - vm * vm)
        assert back[0] == pytest.approx(e, rel=2e-13 * g2)
        assert np.allclose(back[1:4], v, atol=2e-14 * g2)
        assert back[4] == pytest.approx(n, rel=2e-13 * g2)
        # Eq.23 itself: v = M/(E + p(e, n)) with e = E - M.v, n = R sqrt(1 - v^2)
        p = o.eos(back[0], back[4])[0]
        assert np.allclose(back[1:4], U[1:4] / (U[0] + p), atol=1e-13)


def test_newton_root_against_bisection(cross):
    o = Oracle(8, dx=1.0, eos_table=cross)
    rng = np.random.default_rng(4)
    for _ in range(200):
        E = 10 ** rng.uniform(-1, 2)
        M = E * rng.uniform(0.0, 0.98)
        R = rng.uniform(0, 8)
        f = lambda v: v * (E + o.eos(E - M * v, R * math.sqrt(1 - v * v))[0]) - M
        lo, hi = 0.0, M / E
        for _ in range(80):
            mid = 0.5 * (lo + hi)
            if f(mid) > 0:
                hi = mid
            else:
                lo = mid
        prim = o.con2prim([E, M, 0.0, 0.0, R])
        assert prim[1] == pytest.approx(0.5 * (lo + hi), abs=3e-15)


def test_shock_tube_with_linear_table_matches_closed_form_run():
    st = w.shock_tube_1d()
    a = Oracle(400, dx=st["dx"], limiter="minmod", k_stages=2, rk=2)
    b = Oracle(400, dx=st["dx"], limiter="minmod", k_stages=2, rk=2, eos_table=w.linear_eos_table())
    for o in (a, b):
        o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
        o.step(100, 0.4)
    ta, tb = a.time()[0], b.time()[0]
    assert tb == pytest.approx(ta, rel=1e-12)                       # same S_max: cs^2 from the table is 1/3
    for x, y in zip(a.get_state(), b.get_state()):
        assert np.abs(x - y).max() <= 1e-11 * 10


def test_table_run_conserves_and_keeps_uniform_state(cross):
    st = w.gaussian_hot_spot(shape=(10, 12, 14), dx=0.4)
    o = Oracle(14, 12, 10, dx=0.4, limiter="vanleer", k_stages=2, rk=3, bc="periodic", eos_table=cross)
    o.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
    t0 = o.totals()
    o.step(20, 0.3)
    t1 = o.totals()
    assert abs(t1[0] - t0[0]) / t0[0] <= 1e-13 and abs(t1[4] - t0[4]) / t0[4] <= 1e-13
    assert np.abs(o.get_state()[0] - st["E"]).max() > 0.05
    n = 14 * 12 * 10
    o.set_state_prim(np.full(n, 2.0), np.full(n, 0.3), np.full(n, -0.2), np.full(n, 0.5), np.full(n, 1.5))
    before = o.get_state()
    o.step(3, 0.3)
    for x, y in zip(o.get_state(), before):
        assert np.allclose(x, y, rtol=1e-13, atol=0)


def test_signal_speed_uses_the_tables_sound_speed(cross):
    """At rest S_max = c_s with c_s^2 = dp/de + n/(e+p) dp/dn from the table (reading A18)."""
    o = Oracle(8, dx=1.0, eos_table=cross)
    e, n = 3.0, 2.0
    o.set_state_prim(np.full(8, e), np.zeros(8), np.zeros(8), np.zeros(8), np.full(8, n))
    p, p_e, p_n = o.eos(e, n)
    assert o.max_signal_speed()[0] == pytest.approx(math.sqrt(p_e + n * p_n / (e + p)), rel=1e-13)
