"""Pins for the pieces of the oracle: limiters (Q6), con2prim / flux (Q5), FORCE on linear advection (Q7),
the admissibility guard (A12).  CPU only."""
import math

import numpy as np
import pytest

from oracle import mfo
from oracle.mfo import Oracle

LIMS = ["minmod", "superbee", "vanalbada", "vanleer", "mc"]


# ---- the paper's xi(r), retyped from the print: Eq.18-21, PAPER.md:201-207 (MC: textbook form, A8) ----
def xi_paper(name, r):
    if name == "minmod":
        return max(0.0, min(1.0, r))
    if name == "superbee":
        return max(0.0, min(2 * r, 1.0), min(r, 2.0))
    if name == "vanalbada":
        return (r * r + r) / (r * r + 1)
    if name == "vanleer":
        return (r + abs(r)) / (1 + abs(r))
    if name == "mc":
        return max(0.0, min(2 * r, 0.5 * (1 + r), 2.0))
    raise ValueError(name)


@pytest.mark.parametrize("name", LIMS)
def test_slope_equals_xi_of_r_times_a(name):
    """Eq.15-16: Delta~ = xi(r)(U_i-U_{i-1}), r = b/a, on random (a,b) with a != 0."""
    rng = np.random.default_rng(1)
    for _ in range(4000):
        a = rng.normal() * 10 ** rng.uniform(-3, 3)
        b = rng.normal() * 10 ** rng.uniform(-3, 3)
        want = xi_paper(name, b / a) * a
        got = mfo.slope(name, a, b)
        assert got == pytest.approx(want, rel=4e-15, abs=2e-15 * (abs(a) + abs(b)))   # abs: cancellation in r^2+r near r=-1


@pytest.mark.parametrize("name", LIMS + ["none", "first"])
def test_slope_symmetry_eq22(name):
    """Eq.22: xi(1/r) = xi(r)/r  <=>  slope(a,b) == slope(b,a)."""
    rng = np.random.default_rng(2)
    for _ in range(2000):
        a, b = rng.normal(size=2)
        assert mfo.slope(name, a, b) == pytest.approx(mfo.slope(name, b, a), rel=1e-15, abs=0)


@pytest.mark.parametrize("name", LIMS + ["none"])
def test_slope_xi_of_one_is_one(name):
    for a in (1.0, -2.5, 3e-7, -4e9):
        assert mfo.slope(name, a, a) == pytest.approx(a, rel=2e-16)


def test_first_is_zero_and_none_is_central():
    assert mfo.slope("first", 1.3, 0.2) == 0.0
    assert mfo.slope("none", 1.0, 3.0) == 2.0           # Eq.14: (U_{i+1}-U_{i-1})/2


@pytest.mark.parametrize("name", ["minmod", "superbee", "vanleer", "mc"])
def test_tvd_limiters_vanish_at_extrema(name):
    for a, b in ((1.0, -1.0), (-0.3, 2.0), (0.0, 1.0), (1.0, 0.0), (0.0, 0.0)):
        assert mfo.slope(name, a, b) == 0.0


def test_vanalbada_as_printed_is_negative_between_minus_one_and_zero():
    """Reading A7: Eq.20 is printed without max(0,.), so xi<0 for -1<r<0."""
    assert mfo.slope("vanalbada", 1.0, -0.5) == pytest.approx((0.25 - 0.5) / (0.25 + 1.0))
    assert mfo.slope("vanalbada", 0.0, 0.0) == 0.0


def test_limiter_ordering():
    """Minbee is the lower, Superbee the upper edge of the TVD region."""
    rng = np.random.default_rng(3)
    for _ in range(2000):
        a, b = np.abs(rng.normal(size=2)) + 1e-3
        mm, sb = mfo.slope("minmod", a, b), mfo.slope("superbee", a, b)
        for mid in ("vanleer", "mc", "vanalbada"):
            m = mfo.slope(mid, a, b)
            assert mm <= m * (1 + 1e-15) and m <= sb * (1 + 1e-15)


# ---------------------------------------------------------------- con2prim / flux
@pytest.fixture(scope="module")
def orc():
    return Oracle(8, dx=1.0)


def test_con2prim_round_trip(orc):
    """Eq.4 -> Eq.23 returns (e, v, n); <= 1e-14*gamma^2 relative for |v| <= 0.999."""
    rng = np.random.default_rng(4)
    for _ in range(3000):
        e = 10 ** rng.uniform(-3, 3)
        n = 10 ** rng.uniform(-3, 3)
        vdir = rng.normal(size=3)
        vmag = rng.choice([0.0, 1e-8, rng.uniform(0, 0.9), rng.uniform(0.9, 0.999)])
        v = vdir / np.linalg.norm(vdir) * vmag
        prim = np.array([e, v[0], v[1], v[2], n])
        U = orc.prim2con(prim)
        back = orc.con2prim(U)
        g2 = 1.0 / (1.0 - vmag * vmag)
        tol = 1e-14 * g2
        assert back[0] == pytest.approx(e, rel=tol)
        assert np.allclose(back[1:4], v, rtol=0, atol=tol)
        assert back[4] == pytest.approx(n, rel=tol)


def test_prim2con_is_eq4_written_out(orc):
    """Eq.4 evaluated by hand for one boosted state, p = e/3."""
    e, v, n = 3.0, np.array([0.3, -0.2, 0.5]), 2.0
    g2 = 1.0 / (1.0 - v @ v)
    w = (e + e / 3.0) * g2
    U = orc.prim2con([e, *v, n])
    assert U[0] == pytest.approx(w - e / 3.0, rel=1e-15)
    assert np.allclose(U[1:4], w * v, rtol=1e-15)
    assert U[4] == pytest.approx(n * math.sqrt(g2), rel=1e-15)


def test_energy_density_identity_for_cs2_third(orc):
    """For cs2 = 1/3 Eq.23 has the closed form e = sqrt(4E^2 - 3M^2) - E."""
    rng = np.random.default_rng(5)
    for _ in range(500):
        E = 10 ** rng.uniform(-2, 2)
        M = rng.normal(size=3)
        M *= rng.uniform(0, 0.95) * E / np.linalg.norm(M)
        prim = orc.con2prim([E, *M, 1.0])
        assert prim[0] == pytest.approx(math.sqrt(4 * E * E - 3 * (M @ M)) - E, rel=2e-13)


@pytest.mark.parametrize("d", [0, 1, 2])
def test_flux_is_stress_tensor_column(orc, d):
    """Eq.3 equals T^{mu d} of a perfect fluid: ((e+p)g^2 v_d, (e+p)g^2 v_j v_d + p delta, n g v_d)."""
    rng = np.random.default_rng(6 + d)
    for _ in range(500):
        e, n = 10 ** rng.uniform(-2, 2), 10 ** rng.uniform(-2, 2)
        v = rng.normal(size=3)
        v *= rng.uniform(0, 0.99) / np.linalg.norm(v)
        p = e / 3.0
        g2 = 1 / (1 - v @ v)
        w = (e + p) * g2
        want = np.array([w * v[d], w * v[0] * v[d], w * v[1] * v[d], w * v[2] * v[d], n * math.sqrt(g2) * v[d]])
        want[1 + d] += p
        U = orc.prim2con([e, *v, n])
        F = orc.flux(d, U)
        assert np.allclose(F, want, rtol=1e-12 * g2, atol=1e-13 * w)
        assert F[0] == pytest.approx(U[1 + d], rel=1e-12 * g2, abs=1e-14 * w)     # A15: (E+p)v_d == M_d


def test_other_sound_speed():
    o = Oracle(8, dx=1.0, cs2=0.2)
    e, v = 2.0, np.array([0.1, 0.6, -0.3])
    back = o.con2prim(o.prim2con([e, *v, 1.0]))
    assert back[0] == pytest.approx(e, rel=1e-13)
    assert np.allclose(back[1:4], v, atol=1e-14)


def test_guard_vacuum_and_cap(orc):
    """Reading A12: E <= 1e-12 -> all fluxes 0; |M| > (1-1e-10)E -> speed capped, direction kept, M_j, R transported unscaled."""
    assert np.all(orc.flux(0, [1e-13, 1e-14, 0, 0, 5.0]) == 0.0)
    assert np.all(orc.flux(2, [0.0, 0.0, 0, 0, 0.0]) == 0.0)
    U = np.array([1.0, 0.8, 0.0, 0.6000001, 2.0])            # |M| > E
    prim = orc.con2prim(U)
    vmag = np.linalg.norm(prim[1:4])
    assert vmag < 1.0 and vmag > 0.99998
    assert prim[1] / prim[3] == pytest.approx(U[1] / U[3], rel=1e-12)
    F = orc.flux(0, U)
    assert F[4] == pytest.approx(U[4] * prim[1], rel=1e-15)
    assert F[3] == pytest.approx(U[3] * prim[1], rel=1e-15)


# ---------------------------------------------------------------- FORCE on linear advection (Q7)
@pytest.mark.parametrize("alpha", [1.0, 3.0])
def test_first_order_force_linear_stencil(alpha):
    """k=0, no slopes, no predictor: U + dt L(U) on the R-equation with uniform (E, M) is the 3-point stencil
    u_i - c/2 (u_{i+1}-u_{i-1}) + 1/4 (alpha c^2 + 1/alpha)(u_{i+1}-2u_i+u_{i-1}), c = v dt/dx
    (FORCE = 1/2 (Lax-Wendroff + Lax-Friedrichs), Eq.9-11, for the linear flux R v)."""
    nx, dx, dt = 32, 0.5, 0.2
    o = Oracle(nx, dx=dx, limiter="first", k_stages=0, predictor=False, bc="periodic", alpha=alpha)
    rng = np.random.default_rng(7)
    n = 1.0 + rng.uniform(size=nx)
    e0, v0 = 2.0, 0.4
    o.set_state_prim(np.full(nx, e0), np.full(nx, v0), np.zeros(nx), np.zeros(nx), n)
    R = o.get_state()[4].ravel()
    L = o.eval_L(dt)
    c = v0 * dt / dx
    got = R + dt * L[4].ravel()
    Rp, Rm = np.roll(R, -1), np.roll(R, 1)
    want = R - 0.5 * c * (Rp - Rm) + 0.25 * (alpha * c * c + 1 / alpha) * (Rp - 2 * R + Rm)
    assert np.allclose(got, want, rtol=0, atol=1e-14 * R.max())
    for q in range(4):                                           # uniform E, M stay put
        assert np.all(np.abs(L[q]) < 1e-14)


# ---------------------------------------------------------------- MUSCL-Hancock + FORCE on linear advection (pins Eq.12, Eq.13 and reading A3)
@pytest.mark.parametrize("shape,v", [((1, 1, 32), (0.4, 0.0, 0.0)), ((7, 5, 6), (0.3, -0.2, 0.25)), ((1, 9, 8), (-0.35, 0.3, 0.0))])
def test_muscl_hancock_force_closed_form_for_linear_advection(shape, v):
    """With uniform (e, v) the charge R is advected linearly, flux_d = v_d R, and every step of the reconstruction is linear for the central
    slope (Eq.14), so one evaluation of L has a closed form.  Written out here from the paper, not from the oracle:
      slopes       s_d = (u_{+d} - u_{-d})/2                                             Eq.12, Eq.14
      half step    delta = sum_d (lambda/2)(v_d u^{dL} - v_d u^{dR}) = -(1/2) sum_d c_d s_d,  c_d = v_d dt/dx
                   - ONE increment for all faces of the cell (reading A3)                Eq.13  :165-171
      faces        A_d = u + s_d/2 + delta (right face of the cell),  B_d = u_{+d} - s_d(+d)/2 + delta(+d)   :173
      FORCE, k=0   lambda F_d = (c_d/2)(A_d + B_d) - (1/4)(alpha c_d^2 + 1/alpha)(B_d - A_d)   Eq.9-11  :139-149
      L            = -(1/dt) sum_d (lambda F_d - lambda F_d(-d))                          Eq.1  :43
    A wrong factor or sign in the half step, an increment added to one face only, or a per-direction increment all change the result."""
    nz, ny, nx = shape
    dx, dt = 0.5, 0.15
    act = [nx > 1, ny > 1, nz > 1]
    alpha = float(sum(act))
    o = Oracle(nx, ny, nz, dx=dx, limiter="none", k_stages=0, predictor=True, bc="periodic")
    rng = np.random.default_rng(11)
    n = 1.0 + rng.uniform(size=shape)
    full = lambda c: np.full(shape, c)
    o.set_state_prim(full(2.0), full(v[0]), full(v[1]), full(v[2]), n)
    u = o.get_state()[4]
    L = o.eval_L(dt)
    axes = {0: 2, 1: 1, 2: 0}                                            # direction d lives on numpy axis axes[d] of (nz, ny, nx)
    plus = lambda a, d: np.roll(a, -1, axis=axes[d])
    minus = lambda a, d: np.roll(a, 1, axis=axes[d])
    c = [v[d] * dt / dx for d in range(3)]
    s = {d: 0.5 * (plus(u, d) - minus(u, d)) for d in range(3) if act[d]}
    delta = sum(-0.5 * c[d] * s[d] for d in s)
    want = np.zeros(shape)
    for d in s:
        A = u + 0.5 * s[d] + delta
        B = plus(u - 0.5 * s[d] + delta, d)
        lamF = 0.5 * c[d] * (A + B) - 0.25 * (alpha * c[d] ** 2 + 1.0 / alpha) * (B - A)
        want -= (lamF - minus(lamF, d)) / dt
    assert np.allclose(L[4], want, rtol=0, atol=2e-13 * np.abs(want).max())
    for q in range(4):                                                   # uniform E, M: nothing moves
        assert np.all(np.abs(L[q]) < 1e-13)
    # and the half step matters at the level this pin resolves: without it L differs by far more than the tolerance
    o2 = Oracle(nx, ny, nz, dx=dx, limiter="none", k_stages=0, predictor=False, bc="periodic")
    o2.set_state_prim(full(2.0), full(v[0]), full(v[1]), full(v[2]), n)
    assert np.abs(o2.eval_L(dt)[4] - want).max() > 1e-3 * np.abs(want).max()


def test_musta_flux_of_equal_states_is_the_physical_flux(orc):
    """Consistency: U_L = U_R = U gives F = F(U) for any k (Eq.8-11 reduce to the identity)."""
    U = orc.prim2con([2.0, 0.3, -0.2, 0.5, 1.5])
    for k in (0, 1, 4):
        o = Oracle(8, dx=1.0, k_stages=k)
        for d in range(3):
            assert np.allclose(o.musta_flux(d, 0.3, U, U), o.flux(d, U), rtol=1e-15, atol=1e-16)


def test_musta_flux_mirror_symmetry():
    """Mirror x -> -x: swapping the states and flipping M_x flips the sign of the E, M_y, M_z, R fluxes and keeps F_{Mx}."""
    o = Oracle(8, dx=1.0, k_stages=3)
    A = o.prim2con([5.0, 0.2, 0.1, -0.3, 2.0])
    B = o.prim2con([1.0, -0.4, 0.0, 0.2, 0.7])
    flip = np.array([1, -1, 1, 1, 1.0])
    F = o.musta_flux(0, 0.35, A, B)
    G = o.musta_flux(0, 0.35, B * flip, A * flip)
    assert np.allclose(G, F * np.array([-1, 1, -1, -1, -1.0]), rtol=1e-13, atol=1e-15)


# ---------------------------------------------------------------- MUSTA_k on a linear flux: closed form in k (pins Eq.8)
@pytest.mark.parametrize("alpha", [1.0, 3.0])
@pytest.mark.parametrize("d", [0, 1, 2])
def test_musta_linear_flux_closed_form(alpha, d):
    """Eq.8-11 for a LINEAR flux f = c u have a closed form in k, derived here from the paper's equations and
    not from any code: with s = u_L + u_R, j = u_R - u_L and D = (alpha lam c^2 + 1/(alpha lam))/2,
        Eq.10:  u_lw = s/2 - (alpha lam/2) c j          Eq.11:  f_lf = c s/2 - j/(2 alpha lam)
        Eq.9:   F    = c s/2 - D j/2
        Eq.8:   s'   = s - lam c j,   j' = j (1 - lam D)
    so j_l = j_0 q^l with q = 1 - lam D (a geometric sequence), s_l = s_0 - (c/D) j_0 (1 - q^l), and
        F^(k) = c s_0/2 - j_0 (c^2/(2D) (1 - q^k) + (D/2) q^k).
    The R equation of Eq.3 is exactly this when E and M are equal on both sides: they stay equal through every
    stage (their fluxes coincide), so v_d = c is one constant and F_R = c R.  A wrong factor, sign or index in Eq.8 changes q."""
    e0, v = 2.0, np.array([0.4, -0.3, 0.25])
    c = v[d]
    lam = 0.3
    for k in range(0, 6):
        o = Oracle(8, dx=1.0, k_stages=k, alpha=alpha)
        UL = o.prim2con([e0, *v, 1.7])
        UR = o.prim2con([e0, *v, 0.6])
        assert np.all(UL[:4] == UR[:4])
        F = o.musta_flux(d, lam, UL, UR)
        s0, j0 = UL[4] + UR[4], UR[4] - UL[4]
        D = 0.5 * (alpha * lam * c * c + 1.0 / (alpha * lam))
        q = 1.0 - lam * D
        want = 0.5 * c * s0 - j0 * (c * c / (2.0 * D) * (1.0 - q ** k) + 0.5 * D * q ** k)
        assert F[4] == pytest.approx(want, rel=1e-14, abs=1e-15), (k, F[4], want)
        assert np.allclose(F[:4], o.flux(d, UL)[:4], rtol=1e-14, atol=1e-15)        # E, M: the physical flux, untouched by the stages
    # the stages matter: k = 0 and k = 3 differ by far more than the tolerance above (so the test can see Eq.8)
    assert abs((1.0 - q ** 3) * (c * c / (2.0 * D) - 0.5 * D) * j0) > 1e-3


# ---------------------------------------------------------------- signal speed (A10): special cases and the velocity-addition identity
def test_max_signal_speed_special_cases():
    """S = (|v| + c_s)/(1 + |v| c_s) is the relativistic sum of |v| and c_s: equal to c_s for matter at rest, increasing in |v|,
    below 1 and tending to 1 as |v| -> 1, and tanh(artanh|v| + artanh c_s) (rapidities add)."""
    for cs2 in (1.0 / 3.0, 0.2):
        cs = math.sqrt(cs2)
        o = Oracle(4, dx=1.0, cs2=cs2)
        one = np.ones(4)
        o.set_state_prim(2.0 * one, 0 * one, 0 * one, 0 * one, one)
        assert o.max_signal_speed()[0] == pytest.approx(cs, rel=1e-15)
        last = cs
        for vmag in (0.1, 0.5, 0.9, 0.99, 0.9999, 0.999999):
            vx, vy, vz = vmag * 0.6, -vmag * 0.48, vmag * 0.64                         # |v| = vmag in a general direction
            o.set_state_prim(np.array([1.0, 2.0, 3.0, 0.5]), vx * one, vy * one, vz * one, one)
            s = o.max_signal_speed()[0]
            assert s == pytest.approx(math.tanh(math.atanh(vmag) + math.atanh(cs)), rel=1e-9 / (1 - vmag))
            assert last < s < 1.0
            last = s
        assert 1.0 - last < 1e-6


# ---------------------------------------------------------------- RK stage times of the source (A14): quadrature order on a single cell
@pytest.mark.parametrize("rk,order", [(2, 3), (3, 5)])
def test_source_stage_times_are_the_quadrature_nodes(rk, order):
    """On a grid of ONE cell nothing flows, so a step integrates dE/dt = S(t) alone and Eq.6 / Eq.7 become
    quadrature rules: RK2 with the source taken at t, t+dt is the trapezoidal rule, RK3 with t, t+dt, t+dt/2 is Simpson's rule.
    Against the exact integral (an error function) the one-step error must then fall as dt^3 and dt^5; any other stage time
    leaves an O(dt^2) error, and any other weight an O(dt) one."""
    dEdx, sig, x0 = 5.0, 0.5, -1.5                 # the pulse's leading flank: its derivatives keep their sign over [0, dt]
    amp = dEdx * (2 * math.pi * sig * sig) ** -1.5

    def exact(dt):                                  # integral of amp exp(-(x0+t)^2/(2 sig^2)) over [0, dt]; the cell centre sits at x = 0
        r = sig * math.sqrt(2.0)
        return amp * sig * math.sqrt(math.pi / 2) * (math.erf((x0 + dt) / r) - math.erf(x0 / r))

    errs = []
    for dt in (0.2, 0.1, 0.05):
        o = Oracle(1, 1, 1, dx=0.25, rk=rk)
        o.set_state([2.0], [0.0], [0.0], [0.0], [1.0])
        o.set_jet_source(dEdx, sig, x0, 0.0, 0.0)
        o.step_dt(1, dt)
        U = [u.ravel()[0] for u in o.get_state()]
        assert U[1] == pytest.approx(U[0] - 2.0, rel=1e-14)          # S_Mx = S_E
        assert U[2] == 0.0 and U[3] == 0.0 and U[4] == 1.0
        errs.append(abs((U[0] - 2.0) - exact(dt)))
        assert errs[-1] < 0.15 * exact(dt)
    for a, b in zip(errs, errs[1:]):
        assert 2 ** order * 0.7 < a / b < 2 ** order * 1.4, (errs, order)
