/*
 * mfo_oracle.cpp — plain, slow, obviously-correct CPU ORACLE of the MUSTA-FORCE time step of
 * ideal relativistic hydrodynamics (arXiv 1510.06340; text in /root/reference/PAPER.md).
 *
 * TEST INFRASTRUCTURE ONLY.  Loaded by tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs.  Shares NO code with the CUDA path; does not include its headers.
 *
 * It is the algorithm written out step by step in the paper's order and notation (the method is an
 * approximation scheme, so there is no closed-form definition to write instead):
 *     RK stages (Eq.5-7)  ->  L(V):
 *        ghost fill (reading A11)
 *        limited slopes and face values      (Eq.12, Eq.15-22)
 *        MUSCL-Hancock half step             (Eq.13)
 *        MUSTA_k with FORCE-alpha flux       (steps 1-5, Eq.8-11)
 *        flux function + con2prim            (Eq.3, Eq.23)
 *        flux divergence                     (Eq.1)
 * No blocking, fusion, SIMD or reordering.  double only.  Build: g++ -O2 -ffp-contract=off
 * (so the written order of operations is the executed one).  With -fopenmp the outer cell loops run in
 * parallel; every cell's arithmetic and order is unchanged, so results are bit-identical to 1 thread.
 *
 * Pins (tests/, -m "not gpu"): exact p=e/3 Riemann solution under refinement (Q1), conservation on a
 * periodic box (Q2), uniform-state fixed point (Q3), axis-permutation symmetry (Q4), Eq.4<->Eq.23 round
 * trip (Q5), limiter identities vs Eq.18-22 (Q6), first-order FORCE closed-form stencil on linear
 * advection (Q7), limiter/k ordering (Q8), numpy transcription on tiny inputs (Q9), source budget (Q10),
 * the MUSTA_k predictor-corrector update Eq.8 against its closed form in k for a linear flux (a geometric
 * sequence; tests/test_oracle_pieces.py::test_musta_linear_flux_closed_form), the signal speed at rest / at
 * |v| -> 1 / as a sum of rapidities, and the source's RK stage times as the nodes of the trapezoidal and
 * Simpson rules on a one-cell grid (error orders dt^3, dt^5 against the exact erf integral), and the MUSCL-Hancock
 * half step with its face values (Eq.12-14, reading A3: ONE increment for all faces of a cell) through FORCE against the
 * closed form of L for linear advection of the charge in 1D, 2D and 3D
 * (tests/test_oracle_pieces.py::test_muscl_hancock_force_closed_form_for_linear_advection: a half-step factor of lam instead of
 * lam/2, or its sign flipped, fails it), and the Runge-Kutta steps Eq.6 / Eq.7 against their stability polynomials 1 + z + z^2/2 (+ z^3/6)
 * for the linear operator of charge advection (tests/test_oracle_scheme.py::test_runge_kutta_step_is_the_taylor_polynomial_of_a_linear_operator).
 * Ghost cells (reading A11): cyclic translation invariance on a periodic box (bit for bit) and mirror symmetry under outflow, per axis.
 * Single-precision state mode (mfo_set_state_precision, reading A19): tests/test_oracle_state32.py - stored values are
 * floats, one step equals Eq.6 / Eq.7 composed in numpy with float32 rounding of every stage around the 64-bit mfo_eval_L, uniform
 * state fixed, conservation and distance to the 64-bit run at single-precision round-off.
 * PARITY UNPINNED by the paper (definitions of ours): accuracy effect of running the
 * Hancock half step inside every RK stage (A4), admissibility-guard constants (A12), jet source
 * definition (A14), charge profile (A13).
 */
#include "mfo_oracle.h"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>
#ifdef _OPENMP
#include <omp.h>
#endif

namespace {

const double E_VACUUM = 1e-12;          /* A12(i)  */
const double V_CAP    = 1.0 - 1e-10;    /* A12(ii) */

/* Equation of state p = p(e, n), Eq.2 PAPER.md:47.  kind 0: p = cs2*e (the only one the paper gives concretely, :312).
 * kind 1: tabulated.  ln p is stored on a grid that is uniform in ln e (ne points from ln_e0, step dln_e) and uniform in n
 * (nn points from n0, step dn; nn = 1 means no n dependence) and interpolated bilinearly; below/above the e range the end
 * cells extrapolate linearly in (ln e, ln p), outside the n range the value is held.  DESIGN.md reading A18. */
struct Params {
    double cs2;
    int kind;
    int ne, nn;
    double ln_e0, dln_e, n0, dn;
    const double* lnp;          /* [nn][ne], e fastest */
};

struct EosValue {
    double p, p_e, p_n;         /* p, dp/de at fixed n, dp/dn at fixed e */
};

EosValue eos_eval(const Params& P, double e, double n)
{
    EosValue r;
    if (P.kind == 0) { r.p = P.cs2 * e; r.p_e = P.cs2; r.p_n = 0.0; return r; }
    double x = (std::log(e) - P.ln_e0) / P.dln_e;
    int i = (int)std::floor(x);
    if (i < 0) i = 0;
    if (i > P.ne - 2) i = P.ne - 2;
    double fx = x - (double)i;                          /* may leave [0,1]: linear extrapolation in (ln e, ln p) */
    int j = 0;
    double fy = 0.0;
    bool n_inside = false;
    if (P.nn > 1) {
        double y = (n - P.n0) / P.dn;
        j = (int)std::floor(y);
        if (j < 0) j = 0;
        if (j > P.nn - 2) j = P.nn - 2;
        fy = y - (double)j;
        n_inside = fy >= 0.0 && fy <= 1.0;
        if (fy < 0.0) fy = 0.0;
        if (fy > 1.0) fy = 1.0;
    }
    const double* row0 = P.lnp + (long)j * P.ne;
    const double* row1 = P.nn > 1 ? row0 + P.ne : row0;
    double d0 = row0[i + 1] - row0[i], d1 = row1[i + 1] - row1[i];
    double l0 = row0[i] + fx * d0, l1 = row1[i] + fx * d1;
    double lp = l0 + fy * (l1 - l0);
    r.p = std::exp(lp);
    double dlnp_dlne = ((1.0 - fy) * d0 + fy * d1) / P.dln_e;
    r.p_e = r.p * dlnp_dlne / e;
    r.p_n = n_inside ? r.p * ((l1 - l0) / P.dn) : 0.0;
    return r;
}

/* ---------- Eq.14-21 in two-argument form (reading A6/A7/A8): a = U_i-U_{i-1}, b = U_{i+1}-U_i ---------- */
double slope2(int lim, double a, double b)
{
    switch (lim) {
    case MFO_LIM_NONE:                                   /* Eq.14 */
        return 0.5 * (a + b);
    case MFO_LIM_FIRST:
        return 0.0;
    case MFO_LIM_MINMOD: {                               /* Eq.18 Minbee: xi = max(0,min(1,r)) */
        if (a * b > 0.0) {
            double s = (a > 0.0) ? 1.0 : -1.0;
            return s * std::fmin(std::fabs(a), std::fabs(b));
        }
        return 0.0;
    }
    case MFO_LIM_SUPERBEE: {                             /* Eq.19: xi = max(0,min(2r,1),min(r,2)) */
        if (a * b > 0.0) {
            double s = (a > 0.0) ? 1.0 : -1.0;
            double fa = std::fabs(a), fb = std::fabs(b);
            return s * std::fmax(std::fmin(2.0 * fb, fa), std::fmin(fb, 2.0 * fa));
        }
        return 0.0;
    }
    case MFO_LIM_VANALBADA: {                            /* Eq.20, as printed (no max(0,.)), A7 */
        double den = a * a + b * b;
        if (den > 0.0) return (a * b) * (a + b) / den;
        return 0.0;
    }
    case MFO_LIM_VANLEER: {                              /* Eq.21: xi = (r+|r|)/(1+|r|) */
        if (a * b > 0.0) return 2.0 * (a * b) / (a + b);
        return 0.0;
    }
    case MFO_LIM_MC: {                                   /* monotonized central (BASELINE.json cfg 2,5), A8 */
        if (a * b > 0.0) {
            double s = (a > 0.0) ? 1.0 : -1.0;
            return s * std::fmin(std::fmin(2.0 * std::fabs(a), 2.0 * std::fabs(b)), 0.5 * std::fabs(a + b));
        }
        return 0.0;
    }
    }
    return 0.0;
}

/* ---------- Eq.23 for p = cs2*e in closed form, with the admissibility guard A12 ----------
 * v = M/(E+p), e = E - M.v, p = cs2*e  =>  |v| = 2|M| / ((1+cs2)E + sqrt((1+cs2)^2 E^2 - 4 cs2 |M|^2)).
 * Returns v (3), e, p.  PAPER.md:227-234. */
/* Eq.23 for a general p(e, n): the last line is a scalar equation for the speed v = |v|,
 *     f(v) = v (E + p(E - |M| v, R sqrt(1 - v^2))) - |M| = 0,
 * solved by Newton's method from v = |M|/E (where f >= 0), kept inside a bracket [lo, hi] by bisection whenever a Newton step
 * leaves it; at most 60 iterations, stop when |dv| <= 1e-15.  The paper says "solved numerically ... as the fixed point
 * equation for v" (:236); BASELINE.json's north_star names Newton.  DESIGN.md reading A18.  Returns the speed. */
double solve_speed(const Params& P, double E, double M, double R, double* e_out, double* p_out)
{
    double lo = 0.0, hi = M / E, v = hi;
    for (int it = 0; it < 60; ++it) {
        double e = E - M * v;
        double g = std::sqrt(1.0 - v * v);
        EosValue q = eos_eval(P, e, R * g);
        double f = v * (E + q.p) - M;
        if (f == 0.0) break;
        if (f > 0.0) hi = v; else lo = v;
        double df = E + q.p + v * (-M * q.p_e - R * (v / g) * q.p_n);
        double vn = v - f / df;
        if (!(vn > lo && vn < hi)) vn = 0.5 * (lo + hi);
        double dv = std::fabs(vn - v);
        v = vn;
        if (dv <= 1e-15) break;
    }
    double e = E - M * v;
    *e_out = e;
    *p_out = eos_eval(P, e, R * std::sqrt(1.0 - v * v)).p;
    return v;
}

void velocity_pressure(const Params& P, double E, double Mx, double My, double Mz, double R,
                       double v[3], double* e_out, double* p_out)
{
    const double cs2 = P.cs2;
    if (!(E > E_VACUUM)) {                               /* A12(i): vacuum -> v = 0, p = 0 (NaN E also lands here) */
        if (E != E) { v[0] = v[1] = v[2] = E; *e_out = E; *p_out = E; return; }
        v[0] = v[1] = v[2] = 0.0; *e_out = E; *p_out = 0.0;
        return;
    }
    double M2 = Mx * Mx + My * My + Mz * Mz;
    double cap = V_CAP * E;
    if (M2 > cap * cap) {                                /* A12(ii): rescale M to |M| = V_CAP*E, direction kept */
        double s = cap / std::sqrt(M2);
        Mx *= s; My *= s; Mz *= s;
        M2 = Mx * Mx + My * My + Mz * Mz;
    }
    if (P.kind != 0) {                                   /* tabulated EOS: Newton on the speed, then v_j = M_j v/|M| */
        double M = std::sqrt(M2);
        if (M == 0.0) {
            v[0] = v[1] = v[2] = 0.0; *e_out = E; *p_out = eos_eval(P, E, R).p;
            return;
        }
        double e, p;
        double sp = solve_speed(P, E, M, R, &e, &p);
        double s = sp / M;
        v[0] = Mx * s; v[1] = My * s; v[2] = Mz * s;
        *e_out = e; *p_out = p;
        return;
    }
    double c1 = 1.0 + cs2;
    double Q = std::sqrt(c1 * c1 * E * E - 4.0 * cs2 * M2);
    double inv = 2.0 / (c1 * E + Q);
    v[0] = Mx * inv; v[1] = My * inv; v[2] = Mz * inv;
    double e = E - (Mx * v[0] + My * v[1] + Mz * v[2]);  /* e = E - M.v, Eq.23 first line */
    *e_out = e;
    *p_out = cs2 * e;
}

/* ---------- Eq.3: F_d(U) = ((E+p)v_d, M_j v_d + p delta_jd, R v_d) ---------- */
void flux_d(const Params& P, int d, const double U[5], double F[5])
{
    double v[3], e, p;
    velocity_pressure(P, U[0], U[1], U[2], U[3], U[4], v, &e, &p);
    double vd = v[d];
    F[0] = (U[0] + p) * vd;
    F[1] = U[1] * vd;
    F[2] = U[2] * vd;
    F[3] = U[3] * vd;
    F[1 + d] += p;
    F[4] = U[4] * vd;
}

/* ---------- MUSTA_k with FORCE-alpha, steps 1-5 PAPER.md:123-135, Eq.8-11 PAPER.md:130-149 ----------
 * A = U_L^(0), B = U_R^(0).  c_lw = 0.5*alpha*lam, c_lf = 0.5/(alpha*lam) (computed once per step, A16).
 * Reading A1: the Lax-Wendroff state of Eq.10 uses the FLUX difference (Richtmyer), not U_R-U_L as printed.
 * Reading A5: k = number of Eq.8 updates; FORCE is evaluated k+1 times. */
void musta_flux(const Params& cs2, int d, int k, double lam, double c_lw, double c_lf,
                const double A0[5], const double B0[5], double F[5])
{
    double A[5], B[5], FA[5], FB[5], Ulw[5], Flw[5], Flf[5];
    for (int c = 0; c < 5; ++c) { A[c] = A0[c]; B[c] = B0[c]; }
    for (int l = 0;; ++l) {
        flux_d(cs2, d, A, FA);
        flux_d(cs2, d, B, FB);
        for (int c = 0; c < 5; ++c) Ulw[c] = 0.5 * (A[c] + B[c]) - c_lw * (FB[c] - FA[c]);   /* Eq.10 (A1) */
        flux_d(cs2, d, Ulw, Flw);
        for (int c = 0; c < 5; ++c) Flf[c] = 0.5 * (FA[c] + FB[c]) - c_lf * (B[c] - A[c]);   /* Eq.11 */
        for (int c = 0; c < 5; ++c) F[c] = 0.5 * (Flw[c] + Flf[c]);                          /* Eq.9  */
        if (l == k) break;                                                                   /* step 3 */
        for (int c = 0; c < 5; ++c) {                                                        /* Eq.8  */
            A[c] = A[c] - lam * (F[c] - FA[c]);
            B[c] = B[c] - lam * (FB[c] - F[c]);
        }
    }
}

} // namespace

struct mfo_ctx {
    int n[3];            /* interior extents */
    int act[3];          /* extent > 1 */
    int g[3];            /* ghost layers per side: 2 on active axes */
    int tot[3];          /* n + 2g */
    long ncell, ntot;
    int nact;
    double dx;
    int eos, limiter, k, rk, bc, predictor;
    Params P;
    std::vector<double> table;   /* owned copy of ln p for the tabulated EOS */
    double alpha;
    double jet_dEdx, jet_sigma, jet_x0[3];
    int state_bits;      /* 64 (default) or 32: every STORED state value is rounded to float (reading A19) */
    double t, last_dt;
    long long steps;
    int status;
    std::string err;
    /* states in interior layout */
    std::vector<double> U[5], U1[5], U2[5], Lbuf[5];
    /* work arrays in ghost layout */
    std::vector<double> W[5];
    std::vector<double> FL[3][5], FR[3][5];   /* face states U^{dL}, U^{dR} of each cell */
    std::vector<double> FX[3][5];             /* interface flux between c and c+e_d, stored at c */

    long gi(int i, int j, int k_) const {
        return (long)(i + g[0]) + (long)tot[0] * ((long)(j + g[1]) + (long)tot[1] * (long)(k_ + g[2]));
    }
    long ci(int i, int j, int k_) const { return (long)i + (long)n[0] * ((long)j + (long)n[1] * (long)k_); }
};

namespace {

int fail(mfo_ctx* c, int code, const char* msg) { if (c) c->err = msg; return code; }

int bc_index(int i, int n, int bc)
{
    if (bc == MFO_BC_PERIODIC) { int m = i % n; return m < 0 ? m + n : m; }
    return i < 0 ? 0 : (i >= n ? n - 1 : i);               /* outflow = clamp, A11 */
}

/* a1: copy V (interior layout) into W (ghost layout); 2 ghost layers per active axis, per-axis clamp/modulo */
void fill_with_ghosts(mfo_ctx* c, const std::vector<double> V[5])
{
    const int* n = c->n; const int* g = c->g;
#pragma omp parallel for collapse(2)
    for (int k = -g[2]; k < n[2] + g[2]; ++k)
        for (int j = -g[1]; j < n[1] + g[1]; ++j)
            for (int i = -g[0]; i < n[0] + g[0]; ++i) {
                long src = c->ci(bc_index(i, n[0], c->bc), bc_index(j, n[1], c->bc), bc_index(k, n[2], c->bc));
                long dst = c->gi(i, j, k);
                for (int q = 0; q < 5; ++q) c->W[q][dst] = V[q][src];
            }
}

/* L(V) -> c->Lbuf (interior layout).  dt is the step's global dt in every RK stage (A4). */
void eval_L(mfo_ctx* c, const std::vector<double> V[5], double dt)
{
    const int* n = c->n;
    const int h[3] = { c->act[0] ? 1 : 0, c->act[1] ? 1 : 0, c->act[2] ? 1 : 0 };
    const long stride[3] = { 1, (long)c->tot[0], (long)c->tot[0] * (long)c->tot[1] };
    const double lam = dt / c->dx;
    const double hl = 0.5 * lam;
    const double c_lw = 0.5 * c->alpha * lam;
    const double c_lf = 0.5 / (c->alpha * lam);
    const Params& cs2 = c->P;

    fill_with_ghosts(c, V);

    /* a3 + a4: every cell of interior + 1 ghost layer */
#pragma omp parallel for collapse(2)
    for (int k = -h[2]; k < n[2] + h[2]; ++k)
        for (int j = -h[1]; j < n[1] + h[1]; ++j)
            for (int i = -h[0]; i < n[0] + h[0]; ++i) {
                long p = c->gi(i, j, k);
                double UL[3][5], UR[3][5];
                for (int d = 0; d < 3; ++d) {
                    if (!c->act[d]) continue;
                    for (int q = 0; q < 5; ++q) {
                        double um = c->W[q][p - stride[d]], u0 = c->W[q][p], up = c->W[q][p + stride[d]];
                        double a = u0 - um, b = up - u0;
                        double s = slope2(c->limiter, a, b);                   /* Eq.15-17 (A6) */
                        UL[d][q] = u0 - 0.5 * s;                               /* Eq.12 */
                        UR[d][q] = u0 + 0.5 * s;
                    }
                }
                if (c->predictor) {                                            /* Eq.13 (A3): one delta for all faces */
                    double delta[5] = { 0, 0, 0, 0, 0 };
                    bool first = true;
                    for (int d = 0; d < 3; ++d) {
                        if (!c->act[d]) continue;
                        double Fl[5], Fr[5];
                        flux_d(cs2, d, UL[d], Fl);
                        flux_d(cs2, d, UR[d], Fr);
                        for (int q = 0; q < 5; ++q) {
                            double term = hl * (Fl[q] - Fr[q]);
                            delta[q] = first ? term : delta[q] + term;
                        }
                        first = false;
                    }
                    for (int d = 0; d < 3; ++d) {
                        if (!c->act[d]) continue;
                        for (int q = 0; q < 5; ++q) { UL[d][q] += delta[q]; UR[d][q] += delta[q]; }
                    }
                }
                for (int d = 0; d < 3; ++d) {
                    if (!c->act[d]) continue;
                    for (int q = 0; q < 5; ++q) { c->FL[d][q][p] = UL[d][q]; c->FR[d][q][p] = UR[d][q]; }
                }
            }

    /* a5: interface between c and c+e_d: U_L^0 = U~^{dR}_c, U_R^0 = U~^{dL}_{c+e_d} (A2) */
    for (int d = 0; d < 3; ++d) {
        if (!c->act[d]) continue;
        int lo[3] = { 0, 0, 0 };
        lo[d] = -1;
#pragma omp parallel for collapse(2)
        for (int k = lo[2]; k < n[2]; ++k)
            for (int j = lo[1]; j < n[1]; ++j)
                for (int i = lo[0]; i < n[0]; ++i) {
                    long p = c->gi(i, j, k);
                    double A[5], B[5], F[5];
                    for (int q = 0; q < 5; ++q) { A[q] = c->FR[d][q][p]; B[q] = c->FL[d][q][p + stride[d]]; }
                    musta_flux(cs2, d, c->k, lam, c_lw, c_lf, A, B, F);
                    for (int q = 0; q < 5; ++q) c->FX[d][q][p] = F[q];
                }
    }

    /* a7 (first half): L = -(sum_d (F_{+1/2} - F_{-1/2}))/dx, d ascending.  Eq.1 */
#pragma omp parallel for collapse(2)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                long p = c->gi(i, j, k);
                long o = c->ci(i, j, k);
                for (int q = 0; q < 5; ++q) {
                    double acc = 0.0;
                    bool first = true;
                    for (int d = 0; d < 3; ++d) {
                        if (!c->act[d]) continue;
                        double diff = c->FX[d][q][p] - c->FX[d][q][p - stride[d]];
                        acc = first ? diff : acc + diff;
                        first = false;
                    }
                    c->Lbuf[q][o] = -acc / c->dx;
                }
            }
}

/* a8: S_E = S_Mx = dEdx * G_sigma(x - x_jet(t)), x_jet = (x0+t, y0, z0).  Not in the paper; reading A14. */
double jet_source(const mfo_ctx* c, int i, int j, int k, double t)
{
    const double PI = 3.14159265358979323846;
    double s2 = c->jet_sigma * c->jet_sigma;
    double x = (i + 0.5 - c->n[0] / 2.0) * c->dx - (c->jet_x0[0] + t);
    double y = (j + 0.5 - c->n[1] / 2.0) * c->dx - c->jet_x0[1];
    double z = (k + 0.5 - c->n[2] / 2.0) * c->dx - c->jet_x0[2];
    double r2 = x * x + y * y + z * z;
    double norm = 1.0 / std::pow(2.0 * PI * s2, 1.5);
    return c->jet_dEdx * norm * std::exp(-r2 / (2.0 * s2));
}

/* out = ca*Ua + cb*Ub + cdt*(L + S(ts))   (one RK stage of Eq.6/Eq.7; Ub may be null) */
void rk_combine(mfo_ctx* c, std::vector<double> out[5], double ca, const std::vector<double> Ua[5],
                double cb, const std::vector<double>* Ub, double cdt, double ts, int form)
{
    const int* n = c->n;
    const bool src = c->jet_dEdx != 0.0;
#pragma omp parallel for collapse(2)
    for (int k = 0; k < n[2]; ++k)
        for (int j = 0; j < n[1]; ++j)
            for (int i = 0; i < n[0]; ++i) {
                long o = c->ci(i, j, k);
                double S = src ? jet_source(c, i, j, k, ts) : 0.0;
                for (int q = 0; q < 5; ++q) {
                    double Lq = c->Lbuf[q][o];
                    if (src && (q == 0 || q == 1)) Lq = Lq + S;
                    double r;
                    if (form == 0)      r = Ua[q][o] + cdt * Lq;                                   /* U + dt L          */
                    else if (form == 1) r = 0.5 * (Ua[q][o] + Ub[q][o] + cdt * Lq);               /* Eq.6 second line  */
                    else                r = ca * Ua[q][o] + cb * Ub[q][o] + cdt * Lq;             /* Eq.7 lines 2, 3   */
                    out[q][o] = c->state_bits == 32 ? (double)(float)r : r;                        /* A19: the stored state is single precision */
                }
            }
}

/* a2: S_max = max_cells (|v|+cs)/(1+|v|cs), |v| from Eq.23.  Not in the paper (fixed dt there); reading A10. */
double max_signal_speed(mfo_ctx* c, int* bad)
{
    double smax = 0.0;
    int nbad = 0;
    for (long o = 0; o < c->ncell; ++o) {
        double E = c->U[0][o], Mx = c->U[1][o], My = c->U[2][o], Mz = c->U[3][o], R = c->U[4][o];
        if (!std::isfinite(E) || !std::isfinite(Mx) || !std::isfinite(My) || !std::isfinite(Mz) || !std::isfinite(R)) { ++nbad; continue; }
        if (E > E_VACUUM && Mx * Mx + My * My + Mz * Mz > E * E) ++nbad;   /* superluminal stored state (guard still applies) */
        double v[3], e, p;
        velocity_pressure(c->P, E, Mx, My, Mz, R, v, &e, &p);
        double av = std::sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        double cs = std::sqrt(c->P.cs2);
        if (c->P.kind != 0) {                               /* adiabatic sound speed of the table: cs^2 = p_e + n p_n/(e+p) */
            double cs2t = 0.0;
            if (e > 0.0) {
                double nn = R * std::sqrt(1.0 - av * av);
                EosValue q = eos_eval(c->P, e, nn);
                cs2t = q.p_e + nn * q.p_n / (e + q.p);
            }
            cs = cs2t > 0.0 ? std::sqrt(cs2t) : 0.0;
        }
        double s = (av + cs) / (1.0 + av * cs);
        if (s > smax) smax = s;
    }
    if (bad) *bad = nbad;
    return smax;
}

/* A19 ("The state of the system is saved as 5 single precision floating-point numbers per lattice cell"): in 32-bit state
 * mode every value that is STORED as a state - the state handed in, and the result of every Runge-Kutta stage - is rounded to float
 * (round to nearest even); all arithmetic between a load and the next store stays double. */
void round_stored_state(mfo_ctx* c)
{
    if (c->state_bits != 32) return;
    for (int q = 0; q < 5; ++q)
        for (long o = 0; o < c->ncell; ++o) c->U[q][o] = (double)(float)c->U[q][o];
}

void one_step(mfo_ctx* c, double dt)
{
    const double t = c->t;
    if (c->rk == 2) {                                       /* Eq.6 */
        eval_L(c, c->U, dt);
        rk_combine(c, c->U1, 1.0, c->U, 0.0, nullptr, dt, t, 0);
        eval_L(c, c->U1, dt);
        rk_combine(c, c->U2, 0.5, c->U, 0.5, c->U1, dt, t + dt, 1);
        for (int q = 0; q < 5; ++q) c->U[q].swap(c->U2[q]);
    } else {                                                /* Eq.7 */
        eval_L(c, c->U, dt);
        rk_combine(c, c->U1, 1.0, c->U, 0.0, nullptr, dt, t, 0);
        eval_L(c, c->U1, dt);
        rk_combine(c, c->U2, 0.75, c->U, 0.25, c->U1, 0.25 * dt, t + dt, 2);
        eval_L(c, c->U2, dt);
        rk_combine(c, c->U1, 1.0 / 3.0, c->U, 2.0 / 3.0, c->U2, (2.0 / 3.0) * dt, t + 0.5 * dt, 2);
        for (int q = 0; q < 5; ++q) c->U[q].swap(c->U1[q]);
    }
    c->t = t + dt;
    c->last_dt = dt;
    c->steps += 1;
}

} // namespace

extern "C" {

mfo_ctx* mfo_create(int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages)
{
    const int n[3] = { nx, ny, nz };
    for (int a = 0; a < 3; ++a) if (n[a] < 1 || (n[a] > 1 && n[a] < 4)) return nullptr;
    if (!(dx > 0.0) || (eos != MFO_EOS_CS2 && eos != MFO_EOS_TABLE) || limiter < 0 || limiter > MFO_LIM_FIRST || k_stages < 0 || k_stages > 8) return nullptr;
    mfo_ctx* c = new (std::nothrow) mfo_ctx();
    if (!c) return nullptr;
    c->nact = 0;
    for (int a = 0; a < 3; ++a) {
        c->n[a] = n[a]; c->act[a] = n[a] > 1; c->g[a] = c->act[a] ? 2 : 0; c->tot[a] = n[a] + 2 * c->g[a];
        c->nact += c->act[a];
    }
    c->ncell = (long)nx * ny * nz;
    c->ntot = (long)c->tot[0] * c->tot[1] * c->tot[2];
    c->dx = dx; c->eos = eos; c->limiter = limiter; c->k = k_stages;
    c->rk = 2; c->bc = MFO_BC_OUTFLOW; c->predictor = 1;
    c->P.cs2 = 1.0 / 3.0; c->P.kind = 0; c->P.ne = c->P.nn = 0; c->P.ln_e0 = c->P.dln_e = c->P.n0 = c->P.dn = 0.0; c->P.lnp = nullptr;
    c->alpha = c->nact > 0 ? (double)c->nact : 1.0;         /* A9: alpha = number of active directions */
    c->state_bits = 64;
    c->jet_dEdx = 0.0; c->jet_sigma = 1.0; c->jet_x0[0] = c->jet_x0[1] = c->jet_x0[2] = 0.0;
    c->t = 0.0; c->last_dt = 0.0; c->steps = 0; c->status = MFO_OK;
    try {
        for (int q = 0; q < 5; ++q) {
            c->U[q].assign(c->ncell, 0.0); c->U1[q].assign(c->ncell, 0.0); c->U2[q].assign(c->ncell, 0.0);
            c->Lbuf[q].assign(c->ncell, 0.0); c->W[q].assign(c->ntot, 0.0);
            for (int d = 0; d < 3; ++d) if (c->act[d]) {
                c->FL[d][q].assign(c->ntot, 0.0); c->FR[d][q].assign(c->ntot, 0.0); c->FX[d][q].assign(c->ntot, 0.0);
            }
        }
    } catch (...) { delete c; return nullptr; }
    return c;
}

void mfo_destroy(mfo_ctx* c) { delete c; }

int mfo_set_state(mfo_ctx* c, const double* E, const double* Mx, const double* My, const double* Mz, const double* R)
{
    if (!c) return MFO_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MFO_EINVAL, "null pointer");
    const double* src[5] = { E, Mx, My, Mz, R };
    for (int q = 0; q < 5; ++q) std::memcpy(c->U[q].data(), src[q], sizeof(double) * c->ncell);
    round_stored_state(c);
    c->t = 0.0; c->last_dt = 0.0; c->steps = 0; c->status = MFO_OK;
    return MFO_OK;
}

int mfo_get_state(mfo_ctx* c, double* E, double* Mx, double* My, double* Mz, double* R)
{
    if (!c) return MFO_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MFO_EINVAL, "null pointer");
    double* dst[5] = { E, Mx, My, Mz, R };
    for (int q = 0; q < 5; ++q) std::memcpy(dst[q], c->U[q].data(), sizeof(double) * c->ncell);
    return c->status;
}

int mfo_prim2con(mfo_ctx* c, const double prim[5], double U[5])
{
    if (!c || !prim || !U) return MFO_EINVAL;
    /* Eq.4: E=(eps+p)g^2-p, M_i=(eps+p)g^2 v_i, R=n g, g=1/sqrt(1-v^2) */
    double e = prim[0], vx = prim[1], vy = prim[2], vz = prim[3], nn = prim[4];
    double p = eos_eval(c->P, e, nn).p;
    double g2 = 1.0 / (1.0 - (vx * vx + vy * vy + vz * vz));
    double w = (e + p) * g2;
    U[0] = w - p; U[1] = w * vx; U[2] = w * vy; U[3] = w * vz; U[4] = nn * std::sqrt(g2);
    return MFO_OK;
}

int mfo_con2prim(mfo_ctx* c, const double U[5], double prim[5])
{
    if (!c || !prim || !U) return MFO_EINVAL;
    double v[3], e, p;
    velocity_pressure(c->P, U[0], U[1], U[2], U[3], U[4], v, &e, &p);
    prim[0] = e; prim[1] = v[0]; prim[2] = v[1]; prim[3] = v[2];
    prim[4] = U[4] * std::sqrt(1.0 - (v[0] * v[0] + v[1] * v[1] + v[2] * v[2]));   /* n = R sqrt(1-v^2), Eq.23 */
    return MFO_OK;
}

int mfo_set_state_prim(mfo_ctx* c, const double* e, const double* vx, const double* vy, const double* vz, const double* n)
{
    if (!c) return MFO_EINVAL;
    if (!e || !vx || !vy || !vz || !n) return fail(c, MFO_EINVAL, "null pointer");
    for (long o = 0; o < c->ncell; ++o) {
        double prim[5] = { e[o], vx[o], vy[o], vz[o], n[o] }, U[5];
        mfo_prim2con(c, prim, U);
        for (int q = 0; q < 5; ++q) c->U[q][o] = U[q];
    }
    round_stored_state(c);
    c->t = 0.0; c->last_dt = 0.0; c->steps = 0; c->status = MFO_OK;
    return MFO_OK;
}

int mfo_get_state_prim(mfo_ctx* c, double* e, double* vx, double* vy, double* vz, double* n)
{
    if (!c) return MFO_EINVAL;
    if (!e || !vx || !vy || !vz || !n) return fail(c, MFO_EINVAL, "null pointer");
    for (long o = 0; o < c->ncell; ++o) {
        double U[5] = { c->U[0][o], c->U[1][o], c->U[2][o], c->U[3][o], c->U[4][o] }, prim[5];
        mfo_con2prim(c, U, prim);
        e[o] = prim[0]; vx[o] = prim[1]; vy[o] = prim[2]; vz[o] = prim[3]; n[o] = prim[4];
    }
    return c->status;
}

int mfo_max_signal_speed(mfo_ctx* c, double* smax)
{
    if (!c || !smax) return MFO_EINVAL;
    int bad = 0;
    *smax = max_signal_speed(c, &bad);
    if (bad) { c->status = MFO_ESTATE; c->err = "non-finite or superluminal state"; }
    return c->status;
}

int mfo_step(mfo_ctx* c, int n, double cfl)
{
    if (!c) return MFO_EINVAL;
    if (n < 0 || !(cfl > 0.0)) return fail(c, MFO_EINVAL, "bad n or cfl");
    for (int s = 0; s < n; ++s) {
        int bad = 0;
        double smax = max_signal_speed(c, &bad);            /* from U^n, once per step (A10) */
        if (bad) { c->status = MFO_ESTATE; c->err = "non-finite or superluminal state"; }
        double dt = cfl * c->dx / smax;
        one_step(c, dt);
    }
    return c->status;
}

int mfo_step_dt(mfo_ctx* c, int n, double dt)
{
    if (!c) return MFO_EINVAL;
    if (n < 0 || !(dt > 0.0)) return fail(c, MFO_EINVAL, "bad n or dt");
    for (int s = 0; s < n; ++s) one_step(c, dt);
    return c->status;
}

int mfo_conserved_totals(mfo_ctx* c, double out[5])
{
    if (!c || !out) return MFO_EINVAL;
    double vol = 1.0;
    for (int a = 0; a < 3; ++a) if (c->act[a]) vol *= c->dx;   /* dx^D */
    for (int q = 0; q < 5; ++q) {
        long double acc = 0.0L;                              /* 80-bit accumulation */
        for (long o = 0; o < c->ncell; ++o) acc += (long double)c->U[q][o];
        out[q] = (double)(acc * (long double)vol);
    }
    return c->status;
}

int mfo_get_time(mfo_ctx* c, double* t, double* last_dt, long long* steps)
{
    if (!c) return MFO_EINVAL;
    if (t) *t = c->t;
    if (last_dt) *last_dt = c->last_dt;
    if (steps) *steps = c->steps;
    return c->status;
}

int mfo_set_rk(mfo_ctx* c, int order) { if (!c) return MFO_EINVAL; if (order != 2 && order != 3) return fail(c, MFO_EINVAL, "rk order must be 2 or 3"); c->rk = order; return MFO_OK; }
int mfo_set_boundary(mfo_ctx* c, int bc) { if (!c) return MFO_EINVAL; if (bc != MFO_BC_OUTFLOW && bc != MFO_BC_PERIODIC) return fail(c, MFO_EINVAL, "unknown bc"); c->bc = bc; return MFO_OK; }
int mfo_set_cs2(mfo_ctx* c, double cs2) { if (!c) return MFO_EINVAL; if (!(cs2 > 0.0) || !(cs2 < 1.0)) return fail(c, MFO_EINVAL, "cs2 must be in (0,1)"); c->P.cs2 = cs2; return MFO_OK; }
int mfo_set_state_precision(mfo_ctx* c, int bits)
{
    if (!c) return MFO_EINVAL;
    if (bits != 32 && bits != 64) return fail(c, MFO_EINVAL, "state precision must be 32 or 64 bits");
    c->state_bits = bits;
    round_stored_state(c);
    return MFO_OK;
}
int mfo_set_predictor(mfo_ctx* c, int on) { if (!c) return MFO_EINVAL; c->predictor = on ? 1 : 0; return MFO_OK; }
int mfo_set_alpha(mfo_ctx* c, double alpha) { if (!c) return MFO_EINVAL; if (!(alpha > 0.0)) return fail(c, MFO_EINVAL, "alpha must be > 0"); c->alpha = alpha; return MFO_OK; }
int mfo_set_jet_source(mfo_ctx* c, double dEdx, double sigma, double x0, double y0, double z0)
{
    if (!c) return MFO_EINVAL;
    if (dEdx != 0.0 && !(sigma > 0.0)) return fail(c, MFO_EINVAL, "sigma must be > 0");
    c->jet_dEdx = dEdx; c->jet_sigma = sigma > 0.0 ? sigma : 1.0; c->jet_x0[0] = x0; c->jet_x0[1] = y0; c->jet_x0[2] = z0;
    return MFO_OK;
}
int mfo_set_eos_table(mfo_ctx* c, int ne, int nn, double ln_e0, double dln_e, double n0, double dn, const double* ln_p)
{
    if (!c) return MFO_EINVAL;
    if (c->eos != MFO_EOS_TABLE) return fail(c, MFO_EINVAL, "context was not created with MFO_EOS_TABLE");
    if (ne < 2 || nn < 1 || !(dln_e > 0.0) || (nn > 1 && !(dn > 0.0)) || !ln_p) return fail(c, MFO_EINVAL, "bad table");
    c->table.assign(ln_p, ln_p + (long)ne * nn);
    c->P.kind = 1; c->P.ne = ne; c->P.nn = nn; c->P.ln_e0 = ln_e0; c->P.dln_e = dln_e; c->P.n0 = n0; c->P.dn = nn > 1 ? dn : 1.0;
    c->P.lnp = c->table.data();
    return MFO_OK;
}
int mfo_eos(mfo_ctx* c, double e, double n, double out[3])
{
    if (!c || !out) return MFO_EINVAL;
    EosValue q = eos_eval(c->P, e, n);
    out[0] = q.p; out[1] = q.p_e; out[2] = q.p_n;
    return MFO_OK;
}
int mfo_sync(mfo_ctx* c) { return c ? c->status : MFO_EINVAL; }
const char* mfo_last_error(mfo_ctx* c) { return c ? c->err.c_str() : "null context"; }

double mfo_slope(int limiter, double a, double b) { return slope2(limiter, a, b); }

int mfo_flux(mfo_ctx* c, int d, const double U[5], double F[5])
{
    if (!c || !U || !F || d < 0 || d > 2) return MFO_EINVAL;
    flux_d(c->P, d, U, F);
    return MFO_OK;
}

int mfo_musta_flux(mfo_ctx* c, int d, double lam, const double UL[5], const double UR[5], double F[5])
{
    if (!c || !UL || !UR || !F || d < 0 || d > 2 || !(lam > 0.0)) return MFO_EINVAL;
    musta_flux(c->P, d, c->k, lam, 0.5 * c->alpha * lam, 0.5 / (c->alpha * lam), UL, UR, F);
    return MFO_OK;
}

int mfo_eval_L(mfo_ctx* c, double dt, double* L_E, double* L_Mx, double* L_My, double* L_Mz, double* L_R)
{
    if (!c || !(dt > 0.0) || !L_E || !L_Mx || !L_My || !L_Mz || !L_R) return MFO_EINVAL;
    eval_L(c, c->U, dt);
    double* dst[5] = { L_E, L_Mx, L_My, L_Mz, L_R };
    for (int q = 0; q < 5; ++q) std::memcpy(dst[q], c->Lbuf[q].data(), sizeof(double) * c->ncell);
    return MFO_OK;
}

int mfo_eval_faces(mfo_ctx* c, double dt, int d, int side, double* out5)
{
    if (!c || !(dt > 0.0) || d < 0 || d > 2 || !c->act[d] || !out5) return MFO_EINVAL;
    eval_L(c, c->U, dt);
    for (int q = 0; q < 5; ++q)
        for (int k = 0; k < c->n[2]; ++k)
            for (int j = 0; j < c->n[1]; ++j)
                for (int i = 0; i < c->n[0]; ++i)
                    out5[q * c->ncell + c->ci(i, j, k)] = (side ? c->FR : c->FL)[d][q][c->gi(i, j, k)];
    return MFO_OK;
}

int mfo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

} // extern "C"
