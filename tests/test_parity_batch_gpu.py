"""GPU parity of the batched-event launch (mf_create_batch; events are the paper's unit of work):
every event of a batch must evolve exactly as the oracle evolves it alone - own S_max, own dt sequence, own clock - while the kernels of
a step are launched once for all events."""
import numpy as np
import pytest

import parity
from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w
from paper_1510_06340_b200.binding import MustaForce, MustaForceError

pytestmark = pytest.mark.gpu

FIELDS = ("E", "Mx", "My", "Mz", "R")


def lumpy_events(n_events, shape, **kw):
    return [w.lumpy_event(shape=shape, event=ev, **kw) for ev in range(n_events)]


def stack(events):
    return [np.stack([ev[f] for ev in events]) for f in FIELDS]


@pytest.mark.parametrize("rk,limiter,k", [(2, "minmod", 2), (3, "superbee", 3)])
def test_batch_of_events_follows_the_oracle_event_by_event(rk, limiter, k):
    shape = (20, 28, 24)                                               # ragged against the 256-cell blocks, several blocks per event
    events = lumpy_events(3, shape, dx=0.1, n_gauss=8, radius=1.0, half_z=0.7)
    events[1]["E"] = events[1]["E"] * 3.0                              # different S_max histories: the events must not share a dt
    events[1]["R"] = events[1]["R"] * 2.0
    nz, ny, nx = shape
    kw = dict(dx=0.1, limiter=limiter, k_stages=k, rk=rk, bc="outflow")
    g = MustaForce(nx, ny, nz, batch=3, **kw)
    assert g.batch_size() == 3
    g.set_state(*stack(events))
    g.step(40, 0.3)
    got = g.get_state()
    assert g.last_status == 0
    times = []
    for ev, st in enumerate(events):
        o = Oracle(nx, ny, nz, omp=True, **kw)
        o.set_state(*[st[f] for f in FIELDS])
        o.step(40, 0.3)
        ref = o.get_state()
        parity.assert_parity([a[ev] for a in got], ref, what="event %d of a batch of 3" % ev)
        t, dt, steps = g.time(ev)
        to, dto, _ = o.time()
        assert steps == 40 and t == pytest.approx(to, rel=1e-12) and dt == pytest.approx(dto, rel=1e-12)
        times.append(t)
        np.testing.assert_allclose(g.totals(ev), o.totals(), rtol=1e-12, atol=1e-12 * abs(o.totals()[0]))
    assert abs(times[1] - times[0]) > 1e-6 * times[0]                  # the clocks really differ
    np.testing.assert_allclose(g.totals(), sum(g.totals(ev) for ev in range(3)), rtol=1e-12)


def test_config4_batch_of_8_full_size_events_against_their_oracles():
    """BASELINE.json config 4 at full size: the first eight of the 32 seeded 128^3 events in ONE batch (the launch configuration
    `bench.py --config 4 --batch 8` times), 25 steps, every event compared cell by cell with its own oracle run (own S_max, own dt)."""
    events = [w.lumpy_event(event=ev) for ev in range(8)]
    nz, ny, nx = events[0]["shape"]
    kw = dict(events[0]["scheme"])
    g = MustaForce(nx, ny, nz, dx=events[0]["dx"], batch=8, **kw)
    g.set_state(*stack(events))
    g.step(25, events[0]["cfl"])
    got = g.get_state()
    assert g.last_status == 0
    worst = 0.0
    for ev, st in enumerate(events):
        o = Oracle(nx, ny, nz, dx=st["dx"], omp=True, **kw)
        o.set_state(*[st[f] for f in FIELDS])
        o.step(25, st["cfl"])
        r = parity.assert_parity([a[ev] for a in got], o.get_state(), what="config 4 event %d of a batch of 8 at 128^3" % ev)
        worst = max(worst, max(r))
        t, dt, steps = g.time(ev)
        to, dto, _ = o.time()
        assert steps == 25 and t == pytest.approx(to, rel=1e-12) and dt == pytest.approx(dto, rel=1e-12)
    print("config 4, 8 events at 128^3, 25 steps: worst rel diff", worst)


def test_batch_equals_single_contexts_bit_for_bit():
    """Same kernels, same arithmetic: an event inside a batch gives the bits it gives in a context of its own (fixed dt and CFL mode)."""
    shape = (12, 16, 20)
    events = lumpy_events(4, shape, dx=0.1, n_gauss=5, radius=0.8, half_z=0.5)
    nz, ny, nx = shape
    kw = dict(dx=0.1, limiter="mc", k_stages=2, rk=3, bc="periodic")
    b = MustaForce(nx, ny, nz, batch=4, **kw)
    b.set_state(*stack(events))
    b.step(10, 0.3)
    b.step_dt(5, 0.01)
    got = b.get_state()
    prim = b.get_state_prim()
    for ev, st in enumerate(events):
        s = MustaForce(nx, ny, nz, **kw)
        s.set_state(*[st[f] for f in FIELDS])
        s.step(10, 0.3)
        s.step_dt(5, 0.01)
        for a, r in zip(got, s.get_state()):
            assert np.array_equal(a[ev], r)
        for a, r in zip(prim, s.get_state_prim()):
            assert np.array_equal(a[ev], r)
        assert b.time(ev) == s.time()


def test_batch_1d_and_prim_input():
    """1D events (one active axis: the k_combine route) set from rest-frame variables."""
    nx = 200
    x = w.centres(nx, 0.1)
    es = [np.where(x < 0, 10.0, 1.0), np.where(x < 1.0, 4.0, 2.0)]
    kw = dict(dx=0.1, limiter="minmod", k_stages=2, rk=2, bc="outflow")
    b = MustaForce(nx, batch=2, **kw)
    zeros = np.zeros((2, 1, 1, nx))
    e = np.stack(es).reshape(2, 1, 1, nx)
    b.set_state_prim(e, zeros + 0.1, zeros, zeros, e ** 0.75)
    b.step(60, 0.4)
    got = b.get_state()
    for ev in range(2):
        o = Oracle(nx, omp=False, **kw)
        z = np.zeros(nx)
        o.set_state_prim(es[ev], z + 0.1, z, z, es[ev] ** 0.75)
        o.step(60, 0.4)
        parity.assert_parity([a[ev] for a in got], o.get_state(), what="1D event %d" % ev)


def test_batch_argument_checks():
    with pytest.raises(MustaForceError):
        MustaForce(16, 16, 16, batch=0)
    with pytest.raises(MustaForceError):
        MustaForce(16, 16, 16, batch=70000)
    b = MustaForce(16, 16, 16, batch=2)
    with pytest.raises(MustaForceError):
        b.set_path("fused")                                            # the tile kernel is single-event
    with pytest.raises(MustaForceError):
        b.time(2)
    with pytest.raises(MustaForceError):
        b.totals(-1)
