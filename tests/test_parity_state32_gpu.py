"""GPU parity of the single-precision STATE mode (reading A19) against the oracle's
32-bit state mode (pinned in tests/test_oracle_state32.py).

Bars.  The strict build (no FMA contraction, IEEE divide and root, the oracle's operation order) computes every stage result to the
same double as the oracle and rounds it to float in the same way: BIT-IDENTICAL.  The product build differs from the oracle by ~1e-16
relative before the store; rounding to float turns that into a difference of one float ulp (6e-8 relative) in the rare cells whose
value sits on a rounding boundary, which the scheme then carries along like any other perturbation (shocks amplify it).  Its bar is the
mode's own noise floor: after 100 steps the product build must be no further from the 32-bit oracle than twice the distance of the 32-bit oracle from the
64-bit oracle (the effect of rounding EVERY cell at EVERY stage, 1e-6 .. 2e-5 in the A17 norm on these workloads), and below 5e-5 in any
case.  What must hold exactly on both builds: every stored value is a float.
"""
import numpy as np
import pytest

import parity
from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w
from paper_1510_06340_b200.binding import MustaForce, MustaForceError

pytestmark = pytest.mark.gpu

F32 = lambda a: np.asarray(a, dtype=np.float64).astype(np.float32).astype(np.float64)
FIELDS = ("E", "Mx", "My", "Mz", "R")


def _pair(st, strict=False, **over):
    nz, ny, nx = st["shape"]
    kw = dict(st["scheme"])
    kw.update(over)
    g = MustaForce(nx, ny, nz, dx=st["dx"], strict=strict, state_bits=32, **kw)
    o = Oracle(nx, ny, nz, dx=st["dx"], omp=True, state_bits=32, **kw)
    for h in (g, o):
        h.set_state(*[st[f] for f in FIELDS])
        if "jet" in st:
            j = st["jet"]
            h.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
    return g, o


CASES = [("minmod", 2, 2, "outflow", True), ("superbee", 3, 3, "periodic", True), ("mc", 2, 3, "outflow", False),
         ("vanleer", 1, 2, "periodic", True)]


@pytest.mark.parametrize("limiter,k,rk,bc,predictor", CASES)
@pytest.mark.parametrize("shape", [(1, 1, 37), (9, 11, 13), (1, 12, 10), (12, 10, 1), (4, 5, 6)])
def test_strict_build_is_bit_identical_in_32_bit_state_mode(shape, limiter, k, rk, bc, predictor):
    st = w.lumpy_event(shape=shape, dx=0.25, n_gauss=4, radius=0.8, half_z=0.6, background=0.5)
    g, o = _pair(st, strict=True, limiter=limiter, k_stages=k, rk=rk, bc=bc, predictor=predictor)
    # without the Hancock step MF_PATH_AUTO takes the sweep path (when the x axis is active), otherwise the staged path: both carry the state type
    assert g.path() == ("sweep" if (not predictor and shape[2] > 1) else "staged") and g.state_precision() == 32
    for a, b in zip(g.get_state(), [st[f] for f in FIELDS]):
        assert np.array_equal(a, F32(b).reshape(a.shape))                # the state handed in is rounded once
    g.step(7, 0.3)
    o.step(7, 0.3)
    got, ref = g.get_state(), o.get_state()
    for a, b in zip(got, ref):
        assert np.array_equal(a, b.reshape(a.shape))
        assert np.array_equal(a, F32(a))                                 # every stored value is a float
    assert g.time() == o.time()                                          # the same dt sequence, bit for bit (S_max from the rounded state)
    g.step_dt(3, 0.01)
    o.step_dt(3, 0.01)
    for a, b in zip(g.get_state(), o.get_state()):
        assert np.array_equal(a, b.reshape(a.shape))


@pytest.mark.parametrize("index", [1, 2, 3, 4, 5])
def test_product_build_100_steps_32_bit_state(index):
    from test_parity_gpu import _scaled
    st = _scaled(index)
    g, o = _pair(st)
    g.step(100, st["cfl"])
    o.step(100, st["cfl"])
    got, ref = g.get_state(), o.get_state()
    assert g.last_status == 0 and o.status() == 0
    assert all(np.array_equal(a, F32(a)) for a in got)
    nz, ny, nx = st["shape"]
    o64 = Oracle(nx, ny, nz, dx=st["dx"], omp=True, **st["scheme"])
    o64.set_state(*[st[f] for f in FIELDS])
    if "jet" in st:
        j = st["jet"]
        o64.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
    o64.step(100, st["cfl"])
    noise = max(parity.rel_diff(ref, o64.get_state()))                   # what single-precision storage itself costs on this workload
    assert 1e-9 < noise < 5e-5, noise
    r = parity.assert_parity(got, ref, tol=2.0 * noise, what="config %d, 32-bit state (noise floor %.2g)" % (index, noise))
    assert g.time()[0] == pytest.approx(o.time()[0], rel=1e-5)
    print("config", index, "32-bit state: rel diff E,M,R =", r, "32-vs-64-bit oracle:", noise)


def test_32_bit_state_against_the_64_bit_run_and_conservation():
    """Neither better nor worse than single-precision round-off of the state: within 5e-6 of the 64-bit GPU run after 100 steps but not
    closer than 1e-9, totals conserved to float round-off on a periodic box."""
    st = w.gaussian_hot_spot(shape=(40, 36, 44), dx=0.2)
    nz, ny, nx = st["shape"]
    g32 = MustaForce(nx, ny, nz, dx=st["dx"], state_bits=32, **st["scheme"])
    g64 = MustaForce(nx, ny, nz, dx=st["dx"], **st["scheme"])
    for g in (g32, g64):
        g.set_state(*[st[f] for f in FIELDS])
    t0 = g32.totals()
    g32.step(100, st["cfl"])
    g64.step(100, st["cfl"])
    t1 = g32.totals()
    assert abs(t1[0] - t0[0]) / t0[0] < 2e-6 and abs(t1[4] - t0[4]) / t0[4] < 2e-6
    a, b = g32.get_state(), g64.get_state()
    rel = max(np.abs(x - y).max() for x, y in zip(a, b)) / np.abs(b[0]).max()
    assert 1e-9 < rel < 5e-6, rel


def test_switching_precision_converts_the_state_and_other_paths_refuse():
    st = w.lumpy_event(shape=(8, 10, 12), dx=0.2, n_gauss=4, radius=0.8, half_z=0.5, background=0.5)
    nz, ny, nx = st["shape"]
    g = MustaForce(nx, ny, nz, dx=st["dx"], limiter="mc", k_stages=2, rk=3)
    g.set_state(*[st[f] for f in FIELDS])
    g.step(2, 0.3)
    before = g.get_state()
    g.set_state_precision(32)
    assert g.path() == "staged"
    for a, b in zip(g.get_state(), before):
        assert np.array_equal(a, F32(b))
    g.set_state_precision(64)
    for a, b in zip(g.get_state(), before):
        assert np.array_equal(a, F32(b))                                 # widening is exact
    g.set_state_precision(32)
    for p in ("sweep", "fused", "hybrid"):                               # (the sweep path takes the 32-bit state only without the Hancock step)
        with pytest.raises(MustaForceError):
            g.set_path(p)
    with pytest.raises(MustaForceError):
        g.set_state_precision(16)
    # low storage and batches run the same kernels
    g.set_low_storage(True)
    g.step(3, 0.3)
    assert g.sync() == 0 and all(np.array_equal(a, F32(a)) for a in g.get_state())
    g2 = MustaForce(nx, ny, nz, dx=st["dx"], limiter="mc", k_stages=2, rk=3, state_bits=32)
    g2.set_state(*[st[f] for f in FIELDS])
    g2.set_low_storage(True)
    g2.step(5, 0.3)
    o2 = Oracle(nx, ny, nz, dx=st["dx"], limiter="mc", k_stages=2, rk=3, state_bits=32)
    o2.set_state(*[st[f] for f in FIELDS])
    o2.step(5, 0.3)
    parity.assert_parity(g2.get_state(), o2.get_state(), tol=5e-5, what="32-bit state, low storage")


@pytest.mark.parametrize("path", ["staged", "sweep"])
def test_predictor_off_paths_agree_bit_for_bit_in_32_bit_state_mode(path):
    st = w.lumpy_event(shape=(9, 11, 13), dx=0.25, n_gauss=4, radius=0.8, half_z=0.6, background=0.5)
    nz, ny, nx = st["shape"]
    kw = dict(limiter="superbee", k_stages=3, rk=3, bc="periodic", predictor=False)
    g = MustaForce(nx, ny, nz, dx=st["dx"], strict=True, state_bits=32, path=path, **kw)
    o = Oracle(nx, ny, nz, dx=st["dx"], state_bits=32, **kw)
    for h in (g, o):
        h.set_state(*[st[f] for f in FIELDS])
        h.step(8, 0.3)
    assert g.path() == path
    for a, b in zip(g.get_state(), o.get_state()):
        assert np.array_equal(a, b.reshape(a.shape)) and np.array_equal(a, F32(a))
    L = g.eval_L(0.01)                                                   # L itself stays double (not rounded to float)
    Lo = o.eval_L(0.01)
    assert all(np.array_equal(a, np.asarray(b).reshape(a.shape)) for a, b in zip(L, Lo))
    assert not all(np.array_equal(a, F32(a)) for a in L)


def test_tabulated_eos_with_32_bit_state_strict():
    """The two widening rows together: tabulated p(e, n) with Newton con2prim (reading A18) on a single-precision state (A19)."""
    st = w.lumpy_event(shape=(9, 11, 13), dx=0.25, n_gauss=4, radius=0.8, half_z=0.6, background=0.5)
    nz, ny, nx = st["shape"]
    table = w.crossover_eos_table()
    kw = dict(limiter="mc", k_stages=2, rk=3, bc="outflow")
    g = MustaForce(nx, ny, nz, dx=st["dx"], strict=True, state_bits=32, eos_table=table, **kw)
    o = Oracle(nx, ny, nz, dx=st["dx"], state_bits=32, eos_table=table, **kw)
    for h in (g, o):
        h.set_state(*[st[f] for f in FIELDS])
        h.step(5, 0.3)
    for a, b in zip(g.get_state(), o.get_state()):
        assert np.all(np.isfinite(a)) and np.array_equal(a, F32(a))
        assert np.abs(a - b.reshape(a.shape)).max() <= 1e-6 * np.abs(b).max()      # (log/exp of the table path are library calls: not bit-comparable)


def test_batch_of_events_32_bit_state():
    evs = [w.lumpy_event(event=e, shape=(10, 12, 14), dx=0.2, n_gauss=4, radius=0.8, half_z=0.5, background=0.5) for e in range(3)]
    nz, ny, nx = evs[0]["shape"]
    g = MustaForce(nx, ny, nz, dx=0.2, batch=3, strict=True, state_bits=32, limiter="minmod", k_stages=2, rk=2)
    g.set_state(*[np.stack([ev[f] for ev in evs]) for f in FIELDS])
    g.step(6, 0.3)
    got = g.get_state()
    for e, ev in enumerate(evs):
        o = Oracle(nx, ny, nz, dx=0.2, limiter="minmod", k_stages=2, rk=2, state_bits=32)
        o.set_state(*[ev[f] for f in FIELDS])
        o.step(6, 0.3)
        for a, b in zip(got, o.get_state()):
            assert np.array_equal(a[e], b.reshape(a[e].shape))
        tot_o = o.totals()
        tot_g = g.totals(event=e)
        assert np.allclose(tot_g, tot_o, rtol=1e-12, atol=1e-12)
