"""Independent numpy transcription of the scheme in SURVEY.md section 8(c) (pin Q9).

Written separately from oracle/mfo_oracle.cpp (array-at-once with np.pad and slicing instead of cell
loops, r-free limiters via np.where) so that a transcription slip in either shows up as a mismatch on
tiny inputs.  Test helper only; imports neither oracle/ nor the CUDA binding.
State U has shape (5, nz, ny, nx); axis d = 0,1,2 (x,y,z) is numpy axis 3-d.
"""
import numpy as np

E_VAC = 1e-12
V_CAP = 1.0 - 1e-10


def limiter(name, a, b):
    ab = a * b
    s = np.where(a > 0, 1.0, -1.0)
    fa, fb = np.abs(a), np.abs(b)
    if name == "none":
        return 0.5 * (a + b)
    if name == "first":
        return np.zeros_like(a)
    if name == "minmod":
        return np.where(ab > 0, s * np.minimum(fa, fb), 0.0)
    if name == "superbee":
        return np.where(ab > 0, s * np.maximum(np.minimum(2 * fb, fa), np.minimum(fb, 2 * fa)), 0.0)
    if name == "mc":
        return np.where(ab > 0, s * np.minimum(np.minimum(2 * fa, 2 * fb), 0.5 * np.abs(a + b)), 0.0)
    if name == "vanleer":
        return np.where(ab > 0, 2 * ab / np.where(ab > 0, a + b, 1.0), 0.0)
    if name == "vanalbada":
        den = a * a + b * b
        return np.where(den > 0, ab * (a + b) / np.where(den > 0, den, 1.0), 0.0)
    raise ValueError(name)


def vel_p(U, cs2):
    E, Mx, My, Mz = U[0], U[1], U[2], U[3]
    M2 = Mx * Mx + My * My + Mz * Mz
    cap = V_CAP * E
    over = M2 > cap * cap
    with np.errstate(all="ignore"):
        s = np.where(over, cap / np.sqrt(np.where(over, M2, 1.0)), 1.0)
        Mx, My, Mz = np.where(over, Mx * s, Mx), np.where(over, My * s, My), np.where(over, Mz * s, Mz)
        M2 = Mx * Mx + My * My + Mz * Mz
        c1 = 1.0 + cs2
        Q = np.sqrt(c1 * c1 * E * E - 4.0 * cs2 * M2)
        inv = 2.0 / (c1 * E + Q)
        v = [Mx * inv, My * inv, Mz * inv]
        e = E - (Mx * v[0] + My * v[1] + Mz * v[2])
        p = cs2 * e
    vac = ~(E > E_VAC)
    v = [np.where(vac, 0.0, c) for c in v]
    return v, np.where(vac, E, e), np.where(vac, 0.0, p)


def flux(U, d, cs2):
    v, _, p = vel_p(U, cs2)
    F = np.empty_like(U)
    F[0] = (U[0] + p) * v[d]
    for j in range(3):
        F[1 + j] = U[1 + j] * v[d]
    F[1 + d] = F[1 + d] + p
    F[4] = U[4] * v[d]
    return F


def _sl(axis, lo, hi, nd=4):
    s = [slice(None)] * nd
    s[axis] = slice(lo, hi)
    return tuple(s)


def L_op(U, dt, dx, k, lim, predictor, alpha, bc, cs2=1.0 / 3.0):
    shape = U.shape[1:]
    act = [shape[2 - d] > 1 for d in range(3)]          # d -> axis 3-d
    mode = "edge" if bc == "outflow" else "wrap"
    pad = [(0, 0)] + [(2, 2) if act[2 - (ax - 1)] else (0, 0) for ax in (1, 2, 3)]
    W = np.pad(U, pad, mode=mode)
    lam = dt / dx
    # region of cells interior + 1 layer on every active axis
    core = [slice(None)] + [slice(1, -1) if act[2 - (ax - 1)] else slice(None) for ax in (1, 2, 3)]
    C = W[tuple(core)]
    UL, UR = {}, {}
    for d in range(3):
        if not act[d]:
            continue
        ax = 3 - d
        lo = list(core)
        hi = list(core)
        lo[ax] = slice(0, -2)
        hi[ax] = slice(2, None)
        a = C - W[tuple(lo)]
        b = W[tuple(hi)] - C
        s = limiter(lim, a, b)
        UL[d] = C - 0.5 * s
        UR[d] = C + 0.5 * s
    if predictor:
        delta = None
        for d in UL:
            term = (0.5 * lam) * (flux(UL[d], d, cs2) - flux(UR[d], d, cs2))
            delta = term if delta is None else delta + term
        for d in UL:
            UL[d] = UL[d] + delta
            UR[d] = UR[d] + delta
    acc = None
    c_lw = 0.5 * alpha * lam
    c_lf = 0.5 / (alpha * lam)
    for d in UL:
        ax = 3 - d
        inner = [slice(None)] + [slice(1, -1) if (act[2 - (x - 1)] and x != ax) else slice(None) for x in (1, 2, 3)]
        A = UR[d][tuple(inner)][_sl(ax, 0, -1)].copy()
        B = UL[d][tuple(inner)][_sl(ax, 1, None)].copy()
        for l in range(k + 1):
            FA, FB = flux(A, d, cs2), flux(B, d, cs2)
            Flw = flux(0.5 * (A + B) - c_lw * (FB - FA), d, cs2)
            Flf = 0.5 * (FA + FB) - c_lf * (B - A)
            F = 0.5 * (Flw + Flf)
            if l == k:
                break
            A = A - lam * (F - FA)
            B = B - lam * (FB - F)
        diff = F[_sl(ax, 1, None)] - F[_sl(ax, 0, -1)]
        acc = diff if acc is None else acc + diff
    return -acc / dx


def jet(shape, dx, t, dEdx, sigma, x0):
    nz, ny, nx = shape
    x = (np.arange(nx) + 0.5 - nx / 2.0) * dx - (x0[0] + t)
    y = (np.arange(ny) + 0.5 - ny / 2.0) * dx - x0[1]
    z = (np.arange(nz) + 0.5 - nz / 2.0) * dx - x0[2]
    r2 = x[None, None, :] ** 2 + y[None, :, None] ** 2 + z[:, None, None] ** 2
    S = dEdx * (2 * np.pi * sigma ** 2) ** -1.5 * np.exp(-r2 / (2 * sigma ** 2))
    out = np.zeros((5,) + tuple(shape))
    out[0] = S
    out[1] = S
    return out


def smax(U, cs2=1.0 / 3.0):
    v, _, _ = vel_p(U, cs2)
    av = np.sqrt(v[0] ** 2 + v[1] ** 2 + v[2] ** 2)
    cs = np.sqrt(cs2)
    return np.max((av + cs) / (1 + av * cs))


def step(U, dt, dx, k, lim, rk, predictor, alpha, bc, t=0.0, src=None, cs2=1.0 / 3.0):
    def f(V, ts):
        out = L_op(V, dt, dx, k, lim, predictor, alpha, bc, cs2)
        if src is not None:
            out = out + jet(U.shape[1:], dx, ts, *src)
        return out
    if rk == 2:
        U1 = U + dt * f(U, t)
        return 0.5 * (U + U1 + dt * f(U1, t + dt))
    U1 = U + dt * f(U, t)
    U2 = 0.75 * U + 0.25 * U1 + 0.25 * dt * f(U1, t + dt)
    return (1.0 / 3.0) * U + (2.0 / 3.0) * U2 + (2.0 / 3.0) * dt * f(U2, t + 0.5 * dt)
