"""GPU parity of the sweep path (MF_PATH_SWEEP): per-direction sweep kernels that limit the slopes themselves from
a +-2-cell halo of the state, PAPER.md:33 ("each dimension separately"), Eq.12, 15-22 (:155-211), Eq.8-11 (:123-151).

With the Hancock half step off (reading A4) it is the path MF_PATH_AUTO takes; the oracle runs the same scheme with
predictor=False.  Bar: 1e-11 per field after 100 steps in the A17 norm; the strict build must match the oracle bit for bit.
"""
import numpy as np
import pytest

import parity
from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w
from paper_1510_06340_b200.binding import MustaForce, MustaForceError

pytestmark = pytest.mark.gpu

FIELDS = ("E", "Mx", "My", "Mz", "R")


def _scaled(index):
    if index == 1:
        return w.shock_tube_1d()
    if index == 2:
        return w.diagonal_shock_3d(shape=(40, 36, 44))
    if index == 3:
        return w.gaussian_hot_spot(shape=(40, 36, 44), dx=0.2)
    if index == 4:
        return w.lumpy_event(shape=(36, 44, 40), dx=0.1, n_gauss=10, radius=1.2, half_z=0.8)
    st = w.lumpy_event(event=1000, shape=(36, 40, 44), dx=0.1, n_gauss=10, radius=1.2, half_z=0.8)
    st.update(scheme=dict(limiter="mc", k_stages=3, rk=3, bc="outflow"), cfl=0.3,
              jet=dict(dEdx=5.0, sigma=0.3, x0=-1.5, y0=0.0, z0=0.0))
    return st


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_predictor_off_takes_the_sweep_path_and_matches_the_oracle(index):
    """The five configs' schemes without the Hancock step, 100 steps at parity sizes, path chosen by MF_PATH_AUTO."""
    st = _scaled(index)
    g, o = parity.make_pair(st, predictor=False)
    assert g.path() == ("small" if index == 1 else "sweep")               # (config 1 is a launch-bound 1D grid: MF_PATH_AUTO runs it in one block)
    g.step(100, st["cfl"])
    o.step(100, st["cfl"])
    got, ref = g.get_state(), o.get_state()
    assert g.last_status == 0 and o.status() == 0
    r = parity.assert_parity(got, ref, what="config %d, predictor off, sweep path" % index)
    assert g.time()[0] == pytest.approx(o.time()[0], rel=1e-12)
    print("config", index, "sweep: rel diff E,M,R =", r)


@pytest.mark.parametrize("limiter", ["minmod", "superbee", "mc", "vanleer", "vanalbada", "none", "first"])
def test_every_limiter_on_a_2d_grid(limiter):
    """All seven slope functions through the sweep kernels' run-time limiter switch, on an x-y grid with ragged extents."""
    st = w.lumpy_event(shape=(1, 37, 45), dx=0.2, n_gauss=6, radius=1.5, half_z=0.1, background=0.5)
    cfl = 0.2 if limiter == "none" else 0.3
    g, o = parity.make_pair(st, predictor=False, limiter=limiter, k_stages=2, rk=3, bc="periodic")
    assert g.path() == "sweep"
    g.step(30, cfl)
    o.step(30, cfl)
    parity.assert_parity(g.get_state(), o.get_state(), what="limiter %s on the sweep path" % limiter)


def test_sweep_equals_staged_bit_for_bit_without_predictor():
    """Same arithmetic per interface (A = U + H, B = U - H, the same MUSTA): the two paths must agree to the last bit."""
    st = w.diagonal_shock_3d(shape=(20, 24, 28))
    out = {}
    for path in ("sweep", "staged"):
        g = MustaForce(28, 24, 20, dx=st["dx"], path=path, predictor=False, **{k: v for k, v in st["scheme"].items() if k != "predictor"})
        g.set_state(*[st[f] for f in FIELDS])
        g.step(20, 0.3)
        assert g.path() == path
        out[path] = g.get_state()
    for a, b in zip(out["sweep"], out["staged"]):
        assert np.array_equal(a, b)


def test_sweep_with_predictor_matches_the_oracle():
    """Predictor on (3D): the increment of Eq.13 comes from the predictor kernel, the sweeps add it to both face states (A3)."""
    st = _scaled(3)
    g, o = parity.make_pair(st, path="sweep")
    assert g.path() == "sweep"
    g.step(100, st["cfl"])
    o.step(100, st["cfl"])
    parity.assert_parity(g.get_state(), o.get_state(), what="config 3, predictor on, sweep path")


def test_batched_events_on_the_sweep_path():
    shape = (20, 28, 24)
    events = [w.lumpy_event(shape=shape, event=ev, dx=0.1, n_gauss=8, radius=1.0, half_z=0.7) for ev in range(3)]
    events[2]["E"] = events[2]["E"] * 2.5                               # its own S_max history and clock
    nz, ny, nx = shape
    kw = dict(dx=0.1, limiter="minmod", k_stages=2, rk=2, bc="outflow", predictor=False)
    g = MustaForce(nx, ny, nz, batch=3, **kw)
    assert g.path() == "sweep"
    g.set_state(*[np.stack([ev[f] for ev in events]) for f in FIELDS])
    g.step(40, 0.3)
    got = g.get_state()
    for ev, st in enumerate(events):
        o = Oracle(nx, ny, nz, omp=True, **kw)
        o.set_state(*[st[f] for f in FIELDS])
        o.step(40, 0.3)
        parity.assert_parity([a[ev] for a in got], o.get_state(), what="event %d of a batch on the sweep path" % ev)
        assert g.time(ev)[0] == pytest.approx(o.time()[0], rel=1e-12)


def test_path_selection_rules():
    g = MustaForce(16, 16, 16, dx=0.1)
    assert g.path() == "staged"                                           # predictor on: AUTO stays on the staged path
    g = MustaForce(16, 16, 16, dx=0.1, predictor=False)
    assert g.path() == "sweep"
    g = MustaForce(1, 16, 16, dx=0.1, predictor=False)                    # no x axis: the x sweep cannot finish the cells
    assert g.path() == "staged"
    with pytest.raises(MustaForceError):
        MustaForce(1, 16, 16, dx=0.1, predictor=False, path="sweep")
    with pytest.raises(MustaForceError):
        MustaForce(64, dx=0.1, path="sweep")                              # 1D with the predictor on: no predictor kernel for it
    g = MustaForce(64, dx=0.1, predictor=False, path="sweep")
    with pytest.raises(MustaForceError):
        g._chk(g.lib.mf_set_predictor(g.h, 1))                            # refused while the sweep path is selected
    assert g.path() == "sweep"
    g = MustaForce(16, 16, 16, dx=0.1, predictor=False, eos_table=w.crossover_eos_table())
    assert g.path() == "staged"                                           # tabulated EOS: staged path only
    # launch-bound 1D grids: MF_PATH_AUTO runs them in one block, whatever the predictor setting; larger ones and other options do not qualify
    assert MustaForce(400, dx=0.1).path() == "small" and MustaForce(400, dx=0.1, predictor=False).path() == "small"
    assert MustaForce(767, dx=0.1).path() == "staged" and MustaForce(767, dx=0.1, predictor=False).path() == "sweep"
    assert MustaForce(400, dx=0.1, state_bits=32).path() == "staged"
    assert MustaForce(400, dx=0.1, eos_table=w.crossover_eos_table()).path() == "staged"
    with pytest.raises(MustaForceError):
        MustaForce(16, 16, 1, dx=0.1, path="small")


def test_sweep_conserves_and_keeps_a_uniform_state():
    st = w.gaussian_hot_spot(shape=(48, 40, 56), dx=0.15)
    g = MustaForce(56, 40, 48, dx=0.15, limiter="superbee", k_stages=3, rk=3, bc="periodic", predictor=False)
    assert g.path() == "sweep"
    g.set_state(*[st[f] for f in FIELDS])
    t0 = g.totals()
    g.step(50, 0.3)
    t1 = g.totals()
    assert abs(t1[0] - t0[0]) / t0[0] <= 1e-12 and abs(t1[4] - t0[4]) / t0[4] <= 1e-12
    assert max(abs(t1[q]) for q in (1, 2, 3)) / t0[0] <= 1e-12
    n = 56 * 40 * 48
    g.set_state_prim(np.full(n, 2.0), np.full(n, 0.3), np.full(n, -0.2), np.full(n, 0.5), np.full(n, 1.5))
    before = g.get_state()
    g.step(3, 0.3)
    for a, b in zip(g.get_state(), before):
        assert np.allclose(a, b, rtol=3e-15, atol=0)


def test_full_size_config3_256_predictor_off_window():
    """The configuration `bench.py --predictor off` times (256^3, superbee, k=3, RK3, periodic, sweep path): the last two steps re-run by
    the oracle on a window around the hot spot with the GPU's own dt sequence."""
    from test_parity_gpu import _windowed_parity
    st = w.gaussian_hot_spot()
    st["scheme"] = dict(st["scheme"], predictor=False)
    r = _windowed_parity(st, (128, 128, 128))
    print("256^3 sweep window", r)
