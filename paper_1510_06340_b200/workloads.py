"""Seeded synthetic inputs shaped like the five BASELINE.json configs.

This module serves BOTH the CUDA path and the CPU oracle and therefore holds none of the method's
arithmetic: no flux, no con2prim, no limiter, no Eq.4 — every config starts at rest (v = 0), where the
conserved state is simply E = e, M = 0, R = n.  numpy only; it imports neither the binding nor oracle/.

Configs 1-3 are analytic initial conditions.  Configs 4-5 are SYNTHETIC STAND-INS for the
event-by-event fluctuating initial states the paper only names (Monte-Carlo Glauber etc.,
PAPER.md:80-82): sums of Gaussians whose centres and amplitudes come from a counter-based generator.

Cell centres: x_i = (i + 1/2 - n/2) * dx on every axis.  Arrays have shape (nz, ny, nx), x fastest.
"""
import math

import numpy as np

_MASK = (1 << 64) - 1


def splitmix64(seed, count):
    """`count` uniform doubles in [0,1) from the splitmix64 sequence started at `seed` (pure integer recipe)."""
    out = np.empty(count, dtype=np.float64)
    s = seed & _MASK
    for i in range(count):
        s = (s + 0x9E3779B97F4A7C15) & _MASK
        z = s
        z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
        z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
        z = z ^ (z >> 31)
        out[i] = (z >> 11) * (1.0 / 9007199254740992.0)
    return out


def centres(n, dx):
    return (np.arange(n, dtype=np.float64) + 0.5 - n / 2.0) * dx


def _at_rest(e, n):
    z = np.zeros_like(e)
    return {"E": np.ascontiguousarray(e), "Mx": z, "My": z.copy(), "Mz": z.copy(), "R": np.ascontiguousarray(n)}


def _charge(e):
    """Charge density n = e^(3/4) (reading A13: proportional to the entropy density for p = e/3)."""
    return e ** 0.75


def shock_tube_1d(nx=400, length=40.0, e_left=10.0, e_right=1.0, n_left=10.0, n_right=1.0):
    """Config 1: 1D relativistic shock tube on x in [-length/2, length/2], membrane at x = 0, v = 0."""
    dx = length / nx
    x = centres(nx, dx).reshape(1, 1, nx)
    e = np.where(x < 0.0, e_left, e_right)
    n = np.where(x < 0.0, n_left, n_right)
    st = _at_rest(e, n)
    st.update(dx=dx, shape=(1, 1, nx), scheme=dict(limiter="minmod", k_stages=2, rk=2, bc="outflow"), cfl=0.4,
              t_end=12.0, name="cfg1_shock_tube_1d")
    return st


def diagonal_shock_3d(n=128, dx=0.1, e_in=10.0, e_out=1.0, shape=None):
    """Config 2: 3D shock tube along the grid diagonal; e = e_in where x+y+z < 0 else e_out, v = 0.

    With cell centres (i+1/2-n/2)dx the test x+y+z<0 is the integer test 2(i+j+k)+3 < nx+ny+nz."""
    nz, ny, nx = shape if shape is not None else (n, n, n)
    k, j, i = np.meshgrid(np.arange(nz), np.arange(ny), np.arange(nx), indexing="ij")
    inside = 2 * (i + j + k) + 3 < nx + ny + nz
    e = np.where(inside, e_in, e_out).astype(np.float64)
    st = _at_rest(e, _charge(e))
    st.update(dx=dx, shape=(nz, ny, nx), scheme=dict(limiter="mc", k_stages=2, rk=2, bc="outflow"), cfl=0.3,
              steps=200, name="cfg2_diagonal_shock_3d")
    return st


def gaussian_hot_spot(n=256, dx=0.05, e0=1.0, amp=20.0, width=1.0, shape=None):
    """Config 3: e = e0 + amp*exp(-r^2/(2 width^2)) centred in a periodic box, v = 0."""
    nz, ny, nx = shape if shape is not None else (n, n, n)
    gx = np.exp(-centres(nx, dx) ** 2 / (2.0 * width * width))
    gy = np.exp(-centres(ny, dx) ** 2 / (2.0 * width * width))
    gz = np.exp(-centres(nz, dx) ** 2 / (2.0 * width * width))
    e = e0 + amp * gz[:, None, None] * gy[None, :, None] * gx[None, None, :]
    st = _at_rest(e, _charge(e))
    st.update(dx=dx, shape=(nz, ny, nx), scheme=dict(limiter="superbee", k_stages=3, rk=3, bc="periodic"), cfl=0.3,
              steps=500, name="cfg3_gaussian_hot_spot")
    return st


def lumpy_event(event=0, n=128, dx=0.1, n_gauss=40, background=0.1, width=0.5, radius=6.0, half_z=3.0,
                mean_amp=5.0, seed_base=20151006, shape=None):
    """Configs 4/5: e = background + sum_m A_m exp(-|x-c_m|^2/(2 width^2)), v = 0.

    Per Gaussian four uniforms u1..u4: rho = radius*sqrt(u1), phi = 2 pi u2,
    c = (rho cos phi, rho sin phi, half_z (2 u3 - 1)), A = -mean_amp * ln(1 - u4)."""
    nz, ny, nx = shape if shape is not None else (n, n, n)
    u = splitmix64(seed_base + event, 4 * n_gauss).reshape(n_gauss, 4)
    rho = radius * np.sqrt(u[:, 0])
    phi = 2.0 * math.pi * u[:, 1]
    cx, cy, cz = rho * np.cos(phi), rho * np.sin(phi), half_z * (2.0 * u[:, 2] - 1.0)
    amp = -mean_amp * np.log(1.0 - u[:, 3])
    s2 = 2.0 * width * width
    gx = np.exp(-(centres(nx, dx)[None, :] - cx[:, None]) ** 2 / s2)          # (m, nx)
    gy = np.exp(-(centres(ny, dx)[None, :] - cy[:, None]) ** 2 / s2)          # (m, ny)
    gz = np.exp(-(centres(nz, dx)[None, :] - cz[:, None]) ** 2 / s2) * amp[:, None]
    gyx = (gy[:, :, None] * gx[:, None, :]).reshape(n_gauss, ny * nx)
    e = background + (gz.T @ gyx).reshape(nz, ny, nx)
    st = _at_rest(e, _charge(e))
    st.update(dx=dx, shape=(nz, ny, nx), scheme=dict(limiter="minmod", k_stages=2, rk=2, bc="outflow"), cfl=0.3,
              steps=300, name="cfg4_lumpy_event_%d" % event)
    return st


def jet_event(n=512, dx=0.04, shape=None):
    """Config 5: lumpy initial condition with 80 Gaussians (seed 20151006+1000) plus a jet source."""
    st = lumpy_event(event=1000, n=n, dx=dx, n_gauss=80, shape=shape)
    st.update(scheme=dict(limiter="mc", k_stages=3, rk=3, bc="outflow"), cfl=0.3, steps=400,
              jet=dict(dEdx=5.0, sigma=0.3, x0=-6.0, y0=0.0, z0=0.0), name="cfg5_jet_event")
    return st


def eos_table_from(p_of_e_n, e_min=1e-4, e_max=1e3, ne=257, n_max=12.0, nn=25):
    """Tabulate an equation of state p(e, n) the way the library wants it: ln p on a grid uniform in ln e and uniform in n
    (shape (nn, ne), e fastest).  nn = 1 gives a table without n dependence.  Pure data: the method's arithmetic is not here."""
    ln_e = np.linspace(math.log(e_min), math.log(e_max), ne)
    n = np.linspace(0.0, n_max, nn) if nn > 1 else np.zeros(1)
    e2, n2 = np.meshgrid(np.exp(ln_e), n, indexing="xy")               # (nn, ne)
    ln_p = np.log(p_of_e_n(e2, n2))
    return dict(ln_e0=float(ln_e[0]), dln_e=float(ln_e[1] - ln_e[0]), n0=0.0, dn=float(n[1] - n[0]) if nn > 1 else 1.0,
                ln_p=np.ascontiguousarray(ln_p))


def linear_eos_table(cs2=1.0 / 3.0, nn=1, **kw):
    """p = cs2*e as a table: ln p is linear in ln e, so the interpolation is exact and the run must reproduce the closed form."""
    return eos_table_from(lambda e, n: cs2 * e + 0.0 * n, nn=nn, **kw)


def crossover_eos_table(**kw):
    """A smooth synthetic crossover EOS of our own making (no lattice table is available offline): p/e rises from ~0.22 to 1/3
    around e ~ 2 and carries a mild charge dependence.  0 < dp/de < 1 everywhere."""
    def p(e, n):
        soft = 1.0 - 0.35 / (1.0 + (e / 2.0) ** 1.5)
        charge = 1.0 + 0.08 * n * n / ((1.0 + n * n) * (1.0 + e))
        return e / 3.0 * soft * charge
    return eos_table_from(p, **kw)


def config(index, scale=None):
    """BASELINE.json config `index` (1-based).  `scale` = (nz, ny, nx) replaces the grid, same dx, for parity sizes."""
    if index == 1:
        return shock_tube_1d() if scale is None else shock_tube_1d(nx=scale[2], length=scale[2] * 0.1)
    if index == 2:
        return diagonal_shock_3d(shape=scale)
    if index == 3:
        return gaussian_hot_spot(shape=scale)
    if index == 4:
        return lumpy_event(shape=scale)
    if index == 5:
        return jet_event(shape=scale)
    raise ValueError("config index must be 1..5")
