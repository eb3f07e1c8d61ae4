"""GPU parity on the paper's Hubble-like expansion into vacuum (Table 2 settings): true vacuum cells (E = 0 exactly,
guard A12(i)), a moving edge where states leave the admissible set, fixed dt as in the paper.  The closed-form check of this flow is done
on the oracle (tests/test_oracle_hubble.py); here the CUDA paths must follow the oracle."""
import numpy as np
import pytest

import parity
from test_oracle_hubble import hubble_state, T0
from oracle.mfo import Oracle
from paper_1510_06340_b200 import workloads as w
from paper_1510_06340_b200.binding import MustaForce

pytestmark = pytest.mark.gpu


@pytest.mark.parametrize("path", ["staged", "fused", "hybrid"])
def test_hubble_expansion_into_vacuum(path):
    n, dx = 44, 0.1
    x = w.centres(n, dx)
    X, Y, Z = x[None, None, :], x[None, :, None], x[:, None, None]
    e, v, nn = hubble_state([X, Y, Z], T0, 3)
    kw = dict(dx=dx, limiter="minmod", k_stages=4, rk=3, bc="outflow")
    g = MustaForce(n, n, n, path=path, **kw)
    o = Oracle(n, n, n, omp=True, **kw)
    for h in (g, o):
        h.set_state_prim(e, v[0], v[1], v[2], nn)
        h.step_dt(8, 0.03)
    got, ref = g.get_state(), o.get_state()
    assert np.count_nonzero(ref[0] == 0.0) > 1000                      # the far field is still exact vacuum ...
    assert np.count_nonzero((ref[0] > 0.0) & (ref[0] < 1e-12)) > 100   # ... with a shell of cells below the guard threshold around the matter
    parity.assert_parity(got, ref, what="Hubble expansion, 8 steps (%s)" % path)
    for a, b in zip(got, ref):
        assert np.array_equal(a == 0.0, b == 0.0)                      # vacuum cells are exactly vacuum on both sides
    for h in (g, o):
        h.step_dt(22, 0.03)
    got, ref = g.get_state(), o.get_state()
    r = parity.assert_parity(got, ref, what="Hubble expansion, 30 steps (%s)" % path)
    ee = g.get_state_prim()[0]
    ex = hubble_state([X, Y, Z], T0 + 0.9, 3)[0]
    core = np.sqrt(X * X + Y * Y + Z * Z) < 0.4
    assert np.abs(ee - ex)[core].max() < 0.08 * ex[core].max()          # and the GPU run sits on Eq.24 in the core
    print(path, r)
