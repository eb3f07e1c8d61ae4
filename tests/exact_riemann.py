"""Exact solution of the 1D relativistic Riemann problem for p = cs2*e with cs2 = 1/3, v_L = v_R = 0.

A pin for the oracle; shares nothing with oracle/ or the CUDA path.

Left-going rarefaction: Riemann invariant  artanh(v) + (cs/(1+cs2)) ln e = const, and inside the fan
xi = x/t = (v - cs)/(1 - v cs).  Right-going shock into matter at rest: Taub adiabat for p = e/3.
Contact at xi = v*.  n follows n ~ e^(1/(1+cs2)) through the (isentropic) fan and the particle-flux
jump condition across the shock.
"""
import math

import numpy as np

CS2 = 1.0 / 3.0
CS = math.sqrt(CS2)
KAPPA = CS / (1.0 + CS2)          # = sqrt(3)/4


def _v_rarefaction(es, e_left):
    return math.tanh(KAPPA * math.log(e_left / es))


def _v_shock_side(es, e_right):
    return math.sqrt(3.0) * (es - e_right) / math.sqrt((3.0 * e_right + es) * (3.0 * es + e_right))


def star_state(e_left, e_right):
    """(e*, v*, v_shock) by bisection on v_rarefaction(e*) = v_shock_side(e*)."""
    lo, hi = e_right, e_left
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if _v_rarefaction(mid, e_left) - _v_shock_side(mid, e_right) > 0.0:
            lo = mid
        else:
            hi = mid
    es = 0.5 * (lo + hi)
    vs = _v_rarefaction(es, e_left)
    vsh = math.sqrt((3.0 * es + e_right) / (3.0 * (3.0 * e_right + es)))
    return es, vs, vsh


def landmarks(e_left, e_right):
    es, vs, vsh = star_state(e_left, e_right)
    tail = (vs - CS) / (1.0 - vs * CS)
    v1, v2 = vsh, CS2 / vsh                       # shock-frame inflow / outflow speeds

    def gam(u):
        return 1.0 / math.sqrt(1.0 - u * u)
    return dict(e_star=es, v_star=vs, v_shock=vsh, xi_tail=tail, xi_head=-CS,
                nR_star_over_nR=(gam(v1) * v1) / (gam(v2) * v2),
                nL_star_over_nL=(es / e_left) ** (1.0 / (1.0 + CS2)))


def exact(xi, e_left, e_right, n_left, n_right):
    """(e, v, n) at similarity coordinates xi = x/t."""
    lm = landmarks(e_left, e_right)
    es, vs, vsh, tail = lm["e_star"], lm["v_star"], lm["v_shock"], lm["xi_tail"]
    xi = np.asarray(xi, dtype=np.float64)
    e = np.empty_like(xi)
    v = np.empty_like(xi)
    n = np.empty_like(xi)
    for i, s in enumerate(xi.ravel()):
        if s <= -CS:
            ee, vv, nn = e_left, 0.0, n_left
        elif s < tail:
            vv = (s + CS) / (1.0 + s * CS)
            ee = e_left * math.exp(-math.atanh(vv) / KAPPA)
            nn = n_left * (ee / e_left) ** (1.0 / (1.0 + CS2))
        elif s < vs:
            ee, vv, nn = es, vs, n_left * lm["nL_star_over_nL"]
        elif s < vsh:
            ee, vv, nn = es, vs, n_right * lm["nR_star_over_nR"]
        else:
            ee, vv, nn = e_right, 0.0, n_right
        e.ravel()[i], v.ravel()[i], n.ravel()[i] = ee, vv, nn
    return e, v, n
