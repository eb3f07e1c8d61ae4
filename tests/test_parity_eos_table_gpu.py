"""GPU parity for the tabulated equation of state with Newton con2prim (A18): the CUDA path through
the C ABI against the oracle on the same seeded inputs and the same table."""
import numpy as np
import pytest

import parity
from paper_1510_06340_b200 import workloads as w
from paper_1510_06340_b200.binding import MustaForce, MustaForceError

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def cross():
    return w.crossover_eos_table()


@pytest.mark.parametrize("case", ["diagonal_shock", "hot_spot", "lumpy"])
def test_crossover_table_100_steps(case, cross):
    if case == "diagonal_shock":
        st = w.diagonal_shock_3d(shape=(28, 24, 32))
    elif case == "hot_spot":
        st = w.gaussian_hot_spot(shape=(24, 28, 32), dx=0.2)
    else:
        st = w.lumpy_event(shape=(24, 32, 28), dx=0.1, n_gauss=8, radius=1.0, half_z=0.7)
    g, o = parity.make_pair(st, eos_table=cross)
    g.step(100, st["cfl"])
    o.step(100, st["cfl"])
    got, ref = g.get_state(), o.get_state()
    assert g.last_status == 0 and o.status() == 0
    r = parity.assert_parity(got, ref, what="table EOS, " + case)
    assert g.time()[0] == pytest.approx(o.time()[0], rel=1e-12)       # same dt sequence: S_max from the table's sound speed
    print(case, r)


def test_shock_tube_1d_with_table(cross):
    st = w.shock_tube_1d()
    g, o = parity.make_pair(st, eos_table=cross)
    g.step(100, 0.4)
    o.step(100, 0.4)
    parity.assert_parity(g.get_state(), o.get_state(), what="1D shock tube, table EOS")


def test_linear_table_reproduces_closed_form_on_the_gpu():
    st = w.diagonal_shock_3d(shape=(24, 20, 28))
    kw = dict(st["scheme"])
    a = MustaForce(28, 20, 24, dx=st["dx"], **kw)
    b = MustaForce(28, 20, 24, dx=st["dx"], eos_table=w.linear_eos_table(nn=3), **kw)
    for h in (a, b):
        h.set_state(st["E"], st["Mx"], st["My"], st["Mz"], st["R"])
        h.step(50, 0.3)
    parity.assert_parity(b.get_state(), a.get_state(), what="linear table vs closed form")


def test_prim_conversions_with_table(cross):
    rng = np.random.default_rng(8)
    shape = (6, 7, 8)
    e = 10 ** rng.uniform(-1, 1.5, size=shape)
    n = rng.uniform(0, 6, size=shape)
    v = [rng.uniform(-0.5, 0.5, size=shape) for _ in range(3)]
    from oracle.mfo import Oracle
    g = MustaForce(8, 7, 6, dx=0.1, eos_table=cross)
    o = Oracle(8, 7, 6, dx=0.1, eos_table=cross)
    g.set_state_prim(e, v[0], v[1], v[2], n)
    o.set_state_prim(e, v[0], v[1], v[2], n)
    for a, b in zip(g.get_state(), o.get_state()):
        assert np.allclose(a, b, rtol=1e-13, atol=0)
    for a, b, ref in zip(g.get_state_prim(), o.get_state_prim(), (e, v[0], v[1], v[2], n)):
        assert np.allclose(a, b, rtol=1e-12, atol=1e-13)
        assert np.allclose(a, ref, rtol=1e-11, atol=1e-12)                 # Eq.4 -> Eq.23 round trip
    assert g.max_signal_speed()[0] == pytest.approx(o.max_signal_speed()[0], rel=1e-12)


def test_tile_paths_refuse_the_table():
    with pytest.raises(MustaForceError):
        MustaForce(16, 16, 16, dx=0.1, eos_table=w.linear_eos_table(), path="fused")
