"""mf_totals_static: the allocation-free entry point (scratch in a file-scope __device__ array instead of a cudaMalloc'ed buffer) against the
existing path, mf_conserved_totals.  Collected last on purpose (the suite runs with pytest -x).  Two calls in a row on different
states and sizes: the static array keeps the first call's contents, which must not leak into the second."""
import numpy as np
import pytest

from paper_1510_06340_b200 import binding, workloads as w
from paper_1510_06340_b200.binding import MustaForce, MustaForceError

pytestmark = pytest.mark.gpu

FIELDS = ("E", "Mx", "My", "Mz", "R")


def _moving(st, seed):
    """A state with non-zero momenta (the workloads start at rest)."""
    rng = np.random.default_rng(seed)
    out = dict(st)
    for k, a in (("Mx", 0.3), ("My", -0.2), ("Mz", 0.1)):
        out[k] = a * st["E"] * rng.uniform(0.5, 1.0, size=st["E"].shape)
    return out


def _existing_path(st):
    nz, ny, nx = st["shape"]
    g = MustaForce(nx, ny, nz, dx=st["dx"])
    g.set_state(*[st[f] for f in FIELDS])
    return g.totals()


def test_static_totals_match_the_existing_path_twice_in_a_row():
    import torch
    big = _moving(w.lumpy_event(shape=(40, 48, 56), dx=0.1, n_gauss=10, radius=1.5, half_z=1.0), 1)       # 7 blocks of 16384 cells, ragged tail
    small = _moving(w.gaussian_hot_spot(shape=(12, 10, 14), dx=0.2), 2)                                     # 1 block: slots 1..6 keep stale sums
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    for st in (big, small, big):
        dev = [torch.from_numpy(np.ascontiguousarray(st[f])).cuda() for f in FIELDS]
        torch.cuda.synchronize()
        n = dev[0].numel()
        binding.totals_static([t.data_ptr() for t in dev], n, st["dx"] ** 3, out.data_ptr(), stream=torch.cuda.current_stream().cuda_stream)
        got = out.cpu().numpy()
        want = _existing_path(st)
        exact = np.array([np.sum(st[f].astype(np.longdouble)) * st["dx"] ** 3 for f in FIELDS], dtype=np.float64)
        scale = abs(want[0])
        assert np.all(np.abs(got - want) <= 1e-12 * scale), (got, want)
        assert np.all(np.abs(got - exact) <= 1e-12 * scale), (got, exact)


def test_static_totals_reject_sizes_beyond_the_limit_and_null_pointers():
    import torch
    x = torch.ones(16, dtype=torch.float64, device="cuda")
    out = torch.zeros(5, dtype=torch.float64, device="cuda")
    p = [x.data_ptr()] * 5
    with pytest.raises(MustaForceError) as ei:
        binding.totals_static(p, (1 << 24) + 1, 1.0, out.data_ptr())
    assert "exceed" in str(ei.value) and "16777216" in str(ei.value)
    with pytest.raises(MustaForceError):
        binding.totals_static(p, 0, 1.0, out.data_ptr())
    with pytest.raises(MustaForceError):
        binding.totals_static([0] + p[1:], 16, 1.0, out.data_ptr())
    binding.totals_static(p, 16, 0.5, out.data_ptr())                  # still usable after the failures
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), np.full(5, 8.0))
