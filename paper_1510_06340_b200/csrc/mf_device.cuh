// mf_device.cuh — per-cell / per-interface device arithmetic of the MUSTA-FORCE step (fp64, sm_100a).
// Everything here lives in registers; the kernels in mf_kernels.cu decide where operands come from.
// Citations are PAPER.md lines; readings A1..A19 are listed in DESIGN.md.
#pragma once
#include <cuda_runtime.h>

namespace mf {

constexpr double E_VACUUM = 1e-12;        // A12(i)
constexpr double V_CAP    = 1.0 - 1e-10;  // A12(ii)

enum Limiter { LIM_NONE = 0, LIM_MINMOD = 1, LIM_SUPERBEE = 2, LIM_VANALBADA = 3, LIM_VANLEER = 4, LIM_MC = 5, LIM_FIRST = 6 };

// p = cs2*e constants, computed once on the host in the order of reading A16
struct Eos {
    double cs2;
    double c1;      // 1 + cs2
    double c1sq;    // c1*c1
    double four_cs2;
    double cs;      // sqrt(cs2)
    // derived constants of the product build's fast flux (not used by the strict build)
    double qc1sq;   // c1*c1/4
    double hc1;     // c1/2
    double vcap2;   // V_CAP^2
    // tabulated EOS (kind 1, reading A18): ln p on a grid uniform in ln e (ne points) and in n (nn points), e fastest, device memory
    int kind, ne, nn, pad;
    double ln_e0, dln_e, n0, dn;
    const double* lnp;
    // product build: reciprocal spacings and a float copy of ln p for the fp32 seed of the speed solve
    double inv_dln_e, inv_dn;
    const float* lnpf;
};

struct EosValue {
    double p, p_e, p_n;   // p, dp/de at fixed n, dp/dn at fixed e
};

// The table part of the EOS lives in NON-inlined device functions that take the table by value, so that the p = cs2*e kernels keep their
// register allocation: all they carry is a predicate on q.kind and a call on the cold path.
struct TableRef {
    const double* lnp;
    int ne, nn;
    double ln_e0, dln_e, n0, dn;
    double inv_dln_e, inv_dn;
    const float* lnpf;
};
__device__ __forceinline__ TableRef table_of(const Eos& q)
{
    TableRef t; t.lnp = q.lnp; t.ne = q.ne; t.nn = q.nn; t.ln_e0 = q.ln_e0; t.dln_e = q.dln_e; t.n0 = q.n0; t.dn = q.dn;
    t.inv_dln_e = q.inv_dln_e; t.inv_dn = q.inv_dn; t.lnpf = q.lnpf;
    return t;
}

// Eq.2 :47, p = p(e, n) from the table: bilinear interpolation of ln p in (ln e, n); the end cells extrapolate linearly in (ln e, ln p),
// outside the n range the value is held.
static __device__ __noinline__ EosValue eos_table_eval(TableRef q, double e, double n)
{
    EosValue r;
    const double x = (log(e) - q.ln_e0) / q.dln_e;
    int i = (int)floor(x);
    i = max(0, min(i, q.ne - 2));
    const double fx = x - (double)i;
    int j = 0;
    double fy = 0.0;
    bool n_inside = false;
    if (q.nn > 1) {
        const double y = (n - q.n0) / q.dn;
        j = (int)floor(y);
        j = max(0, min(j, q.nn - 2));
        fy = y - (double)j;
        n_inside = fy >= 0.0 && fy <= 1.0;
        fy = fmin(fmax(fy, 0.0), 1.0);
    }
    const double* row0 = q.lnp + (long long)j * q.ne;
    const double* row1 = q.nn > 1 ? row0 + q.ne : row0;
    const double d0 = __ldg(row0 + i + 1) - __ldg(row0 + i), d1 = __ldg(row1 + i + 1) - __ldg(row1 + i);
    const double l0 = __ldg(row0 + i) + fx * d0, l1 = __ldg(row1 + i) + fx * d1;
    const double lp = l0 + fy * (l1 - l0);
    r.p = exp(lp);
    const double dlnp_dlne = ((1.0 - fy) * d0 + fy * d1) / q.dln_e;
    r.p_e = r.p * dlnp_dlne / e;
    r.p_n = n_inside ? r.p * ((l1 - l0) / q.dn) : 0.0;
    return r;
}

// EK is a COMPILE-TIME switch (0: p = cs2*e, 1: table): the kernels are instantiated twice and the launchers pick by q.kind, so that
// the closed-form instantiations do not carry a single instruction or register of the table path.
template <int EK = 0>
__device__ __forceinline__ EosValue eos_eval(const Eos& q, double e, double n)
{
    if (EK == 0) { EosValue r; r.p = q.cs2 * e; r.p_e = q.cs2; r.p_n = 0.0; return r; }
    return eos_table_eval(table_of(q), e, n);
}

// Eq.23 :231-236 for a tabulated p(e, n): Newton on f(v) = v (E + p(E - |M| v, R sqrt(1 - v^2))) - |M| from v = |M|/E, bisection whenever
// a step leaves the bracket, at most 60 iterations, stop at |dv| <= 1e-15.  Data-dependent trip count: lanes of a warp wait for the
// slowest.  out = (speed, e, p).
struct SpeedEP {
    double v, e, p;
};
// Measurement build only (-DMF_COUNT_EVALS, never the product): how many speed solves run and how many table evaluations they take,
// printed by k_end_step; bench.py's roofline for the tabulated EOS is built on these means (DESIGN.md section 10 row 1).
#ifdef MF_COUNT_EVALS
static __device__ unsigned long long g_eval_count[4];      // solves, full evaluations (log + exp), incremental evaluations, fallback solves
#define MF_COUNT(i) atomicAdd(&g_eval_count[i], 1ull)
#else
#define MF_COUNT(i) ((void)0)
#endif
#ifndef MF_STRICT
// ---- product build: the same root in far fewer FP64 instructions.
//  1. fp32 seed: the p = e/3 closed form, then two Newton steps on the float copy of the table (MUFU log/exp): |dv|/v ~ 1e-5.
//  2. fp64 Newton from the seed.  The first evaluation pays log() and exp(); every later one moves e and ln p by a tiny
//     relative amount, so ln e' = ln e + log1p(d) and p' = p exp(d') are three-term series (|d| < 1e-4, error < 3e-17).
//  3. Quadratic convergence: once |dv| <= 3e-8 the step just taken is the last (error ~ dv^2) provided p is smooth between the two
//     speeds, i.e. both lie in one table cell (ln p has kinks at the cell edges, across which Newton converges only linearly);
//     p at the new speed is then the first-order update with the derivative Newton already has.
// Anything unusual (seed or step outside (0, |M|/E), no convergence in 6 steps, non-finite) falls back to the bracketed loop below.
// The solve stays a non-inlined call: inlined into the kernels it measured 15% slower (B200, 128^3), at 80 and at 128 registers.
struct TableEvalState {
    double e, inv_e, lne, lp, p, p_e, p_n;
    int i, j;                                                  // table cell of the evaluation
};

__device__ __forceinline__ double rcp_pos(double x)            // 1/x, x normal and positive; 3 FP64 instructions, < 1 ulp
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    const double e1 = fma(-x, y, 1.0);
    return fma(y, fma(e1, e1, e1), y);
}
__device__ __forceinline__ double sqrt_newton(double x)        // sqrt(x), x normal and positive; 7 FP64 instructions
{
    double r;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    double g = x * r, h = 0.5 * r;
    const double e1 = fma(-g, h, 0.5);
    g = fma(g, e1, g); h = fma(h, e1, h);
    return fma(h, fma(-g, g, x), g);
}

template <bool INCR>
__device__ __forceinline__ void table_eval_step(const TableRef& q, double e, double n, TableEvalState& s)
{
    double lne;
    if (INCR) {
        const double d = (e - s.e) * s.inv_e;
        lne = fabs(d) < 1e-4 ? fma(d, fma(d, fma(d, 1.0 / 3.0, -0.5), 1.0), s.lne) : log(e);
    } else lne = log(e);
    const double x = (lne - q.ln_e0) * q.inv_dln_e;
    const int i = max(0, min(__double2int_rd(x), q.ne - 2));
    const double fx = x - (double)i;
    int j = 0;
    double fy = 0.0;
    bool n_inside = false;
    if (q.nn > 1) {
        const double y = (n - q.n0) * q.inv_dn;
        j = max(0, min(__double2int_rd(y), q.nn - 2));
        fy = y - (double)j;
        n_inside = fy >= 0.0 && fy <= 1.0;
        fy = fmin(fmax(fy, 0.0), 1.0);
    }
    const double* row0 = q.lnp + (unsigned int)(j * q.ne + i);
    const double* row1 = q.nn > 1 ? row0 + q.ne : row0;
    const double l00 = __ldg(row0), l10 = __ldg(row1);
    const double d0 = __ldg(row0 + 1) - l00, d1 = __ldg(row1 + 1) - l10;
    const double l0 = fma(fx, d0, l00), l1 = fma(fx, d1, l10);
    const double lp = fma(fy, l1 - l0, l0);
    double p;
    if (INCR) {
        const double d = lp - s.lp;
        p = fabs(d) < 1e-4 ? s.p * fma(d, fma(d, fma(d, 1.0 / 6.0, 0.5), 1.0), 1.0) : exp(lp);
    } else p = exp(lp);
    const double inv_e = rcp_pos(e);
    s.e = e; s.inv_e = inv_e; s.lne = lne; s.lp = lp; s.p = p; s.i = i; s.j = j;
    s.p_e = p * (fma(fy, d1 - d0, d0) * q.inv_dln_e) * inv_e;
    s.p_n = n_inside ? p * ((l1 - l0) * q.inv_dn) : 0.0;
}

// fp32 seed of the speed: p = e/3 closed form, then two Newton steps on the float table.  Any float in [0, hi] is a valid seed.
__device__ __forceinline__ float seed_speed_f32(const TableRef& q, float E, float M, float R, float hi)
{
    const float c1 = 4.0f / 3.0f;
    float v = __fdividef(2.0f * M, fmaf(c1, E, sqrtf(fmaxf(fmaf(c1 * c1 * E, E, -c1 * M * M), 0.0f))));
    const float ln_e0 = (float)q.ln_e0, inv_dln_e = (float)q.inv_dln_e, n0 = (float)q.n0, inv_dn = (float)q.inv_dn;
#pragma unroll
    for (int it = 0; it < 2; ++it) {
        const float e = fmaf(-M, v, E);
        const float g2 = fmaf(-v, v, 1.0f);
        if (!(e > 0.0f) || !(g2 > 0.0f)) break;
        const float rg = rsqrtf(g2), g = g2 * rg;
        const float x = (__logf(e) - ln_e0) * inv_dln_e;
        const int i = max(0, min(__float2int_rd(x), q.ne - 2));
        const float fx = x - (float)i;
        int j = 0;
        float fy = 0.0f;
        bool n_inside = false;
        if (q.nn > 1) {
            const float y = (R * g - n0) * inv_dn;
            j = max(0, min(__float2int_rd(y), q.nn - 2));
            fy = y - (float)j;
            n_inside = fy >= 0.0f && fy <= 1.0f;
            fy = fminf(fmaxf(fy, 0.0f), 1.0f);
        }
        const float* row0 = q.lnpf + (unsigned int)(j * q.ne + i);
        const float* row1 = q.nn > 1 ? row0 + q.ne : row0;
        const float l00 = __ldg(row0), l10 = __ldg(row1);
        const float d0 = __ldg(row0 + 1) - l00, d1 = __ldg(row1 + 1) - l10;
        const float l0 = fmaf(fx, d0, l00), l1 = fmaf(fx, d1, l10);
        const float p = __expf(fmaf(fy, l1 - l0, l0));
        const float p_e = __fdividef(p * fmaf(fy, d1 - d0, d0) * inv_dln_e, e);
        const float p_n = n_inside ? p * (l1 - l0) * inv_dn : 0.0f;
        const float f = fmaf(v, E + p, -M);
        const float df = E + p - v * fmaf(M, p_e, R * v * rg * p_n);
        const float vn = v - __fdividef(f, df);
        if (!(vn >= 0.0f && vn <= hi)) break;
        v = vn;
    }
    return v;
}

__device__ __forceinline__ bool solve_speed_fast(const TableRef& q, double E, double M, double R, double& v_out, double& e_out, double& p_out)
{
    const double hi = M * rcp_pos(E);
    double v = (double)seed_speed_f32(q, (float)E, (float)M, (float)R, (float)hi);
    if (!(v > 0.0 && v < hi)) return false;
    TableEvalState s;
#pragma unroll 1
    for (int it = 0; it < 6; ++it) {
        const double e = fma(-M, v, E);
        const double g = sqrt_newton(fma(-v, v, 1.0));
        if (it == 0) { MF_COUNT(1); table_eval_step<false>(q, e, R * g, s); } else { MF_COUNT(2); table_eval_step<true>(q, e, R * g, s); }
        const double f = fma(v, E + s.p, -M);
        const double dpdv = -fma(M, s.p_e, R * (v * rcp_pos(g)) * s.p_n);
        const double df = fma(v, dpdv, E + s.p);
        const double dv = -f * rcp_pos(df);
        const double vn = v + dv;
        if (!(df > 0.0) || !(vn > 0.0 && vn < hi)) return false;
        if (fabs(dv) <= 3e-8) {
            // the step is the last one if p is smooth between v and vn, i.e. both lie in one table cell (ln p has kinks at the cell
            // edges, across which Newton converges only linearly), or if it is as small as the bracketed loop's own stopping step
            const double en = fma(-M, vn, E);
            const double d = (en - s.e) * s.inv_e;
            bool last = fabs(dv) <= 1e-15;
            if (!last && fabs(d) < 1e-4) {
                const double lne = fma(d, fma(d, fma(d, 1.0 / 3.0, -0.5), 1.0), s.lne);
                last = max(0, min(__double2int_rd((lne - q.ln_e0) * q.inv_dln_e), q.ne - 2)) == s.i;
                if (last && q.nn > 1) {
                    const double gn = sqrt_newton(fma(-vn, vn, 1.0));
                    last = max(0, min(__double2int_rd((R * gn - q.n0) * q.inv_dn), q.nn - 2)) == s.j;
                }
            }
            if (last) { v_out = vn; e_out = en; p_out = fma(dpdv, dv, s.p); return true; }
        }
        v = vn;
    }
    return false;
}
#endif

static __device__ __noinline__ SpeedEP solve_speed(TableRef q, double E, double M, double R)
{
    MF_COUNT(0);
#ifndef MF_STRICT
    {
        SpeedEP r;
        if (solve_speed_fast(q, E, M, R, r.v, r.e, r.p)) return r;
    }
#endif
    MF_COUNT(3);
    double lo = 0.0, hi = M / E, v = hi;
    for (int it = 0; it < 60; ++it) {
        const double e = E - M * v;
        const double g = sqrt(1.0 - v * v);
        const EosValue w = eos_table_eval(q, e, R * g);
        const double f = v * (E + w.p) - M;
        if (f == 0.0) break;
        if (f > 0.0) hi = v; else lo = v;
        const double df = E + w.p + v * (-M * w.p_e - R * (v / g) * w.p_n);
        double vn = v - f / df;
        if (!(vn > lo && vn < hi)) vn = 0.5 * (lo + hi);
        const double dv = fabs(vn - v);
        v = vn;
        if (dv <= 1e-15) break;
    }
    SpeedEP r;
    r.v = v;
    r.e = E - M * v;
    r.p = eos_table_eval(q, r.e, R * sqrt(1.0 - v * v)).p;
    return r;
}

// ---- Eq.14-21 in two-argument form (A6): a = U_i - U_{i-1}, b = U_{i+1} - U_i; returns the limited slope
template <int LIM>
__device__ __forceinline__ double slope2(double a, double b)
{
    if (LIM == LIM_NONE) return 0.5 * (a + b);                                     // Eq.14 :177
    if (LIM == LIM_FIRST) return 0.0;
    if (LIM == LIM_VANALBADA) {                                                    // Eq.20 :205 as printed (A7)
        double den = a * a + b * b;
        return den > 0.0 ? (a * b) * (a + b) / den : 0.0;
    }
    double ab = a * b;
    if (LIM == LIM_VANLEER) return ab > 0.0 ? 2.0 * ab / (a + b) : 0.0;            // Eq.21 :207
    double fa = fabs(a), fb = fabs(b), m;
    if (LIM == LIM_MINMOD) m = fmin(fa, fb);                                       // Eq.18 :201
    else if (LIM == LIM_SUPERBEE) m = fmin(fmax(fa, fb), 2.0 * fmin(fa, fb));      // Eq.19 :203: max(min(2|b|,|a|), min(|b|,2|a|)) = min(hi, 2 lo), exactly
    else m = fmin(2.0 * fmin(fa, fb), 0.5 * fabs(a + b));                          // MC (A8): min(2|a|, 2|b|) = 2 min(|a|,|b|), exactly
    m = copysign(m, a);
    return ab > 0.0 ? m : 0.0;
}

// Half the limited slope, 0.5 * slope2(a, b), for the product build.  For minmod, superbee and MC the magnitude comparisons are single
// DSETPs with |.| operand modifiers and the selects act on the SIGNED operands (lo, hi, a+b all carry the sign of a wherever the result is
// used), so no fmin/fmax (a DSETP, two selects, a NaN fix-up and register moves each on this target), no copysign: 14 instructions for
// superbee.  An earlier form took min/max on the integer pipe from the bit patterns (~20 instructions, none on the FP64 pipe); measured on
// B200 the shorter sequence wins even in the FP64-bound sweep kernels (cell stage 0.73 -> 0.67 ms, sweep path 7.19 -> 6.97 ms per step).
// Equal to 0.5 * slope2 bit for bit: every operation is exact except a + b, which slope2 forms too; "same sign" is a*b > 0 (A6, A16).
template <int LIM>
__device__ __forceinline__ double half_slope2(double a, double b)
{
    if (LIM != LIM_MINMOD && LIM != LIM_SUPERBEE && LIM != LIM_MC) return 0.5 * slope2<LIM>(a, b);
    const bool a_less = fabs(a) < fabs(b);
    const double lo = a_less ? a : b, hi = a_less ? b : a;
    double r;
    if (LIM == LIM_MINMOD) r = 0.5 * lo;
    else if (LIM == LIM_SUPERBEE) { const double lo2 = lo + lo; r = 0.5 * (fabs(hi) < fabs(lo2) ? hi : lo2); }      // min(hi, 2 lo)/2
    else { const double q = 0.25 * (a + b); r = fabs(q) < fabs(lo) ? q : lo; }                                     // min(2 lo, |a+b|/2)/2
    return a * b > 0.0 ? r : 0.0;
}

// ---- fp64 reciprocal and square root for the flux core.
// The product build uses branch-free Newton sequences seeded by the MUFU approximations (rcp/rsqrt.approx.ftz.f64,
// ~20 good bits): 3 and 6 FP64-pipe instructions instead of the 9 and 14.5 issue slots that the IEEE-rounded '/' and
// sqrt() cost on B200 (mf_probe_fp64), and no slow-path branch, so independent flux evaluations interleave.
// Results are within 1 ulp of the correctly rounded value.  The strict build (MF_STRICT)
// keeps IEEE division and sqrt so that it can be compared with the oracle bit for bit.
#ifdef MF_STRICT
__device__ __forceinline__ double two_over(double x) { return 2.0 / x; }
__device__ __forceinline__ double sqrt_pos(double x) { return sqrt(x); }
#else
__device__ __forceinline__ double two_over(double x)          // 2/x for normal, positive x
{
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double e = fma(-x, y, 1.0);
    double t = fma(e, e, e);
    y = fma(y, t, y);                                           // relative error eps^3 + rounding
    return y + y;
}
__device__ __forceinline__ double sqrt_pos(double x)          // sqrt(x) for normal, positive x: 6 FP64 instructions
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));    // y = (1 + eps)/sqrt(x), |eps| ~ 2^-20
    double g = x * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);                                 // -eps - eps^2/2
    g = fma(g, r, g);                                           // sqrt(x) (1 - 1.5 eps^2)
    double d = fma(-g, g, x);                                   // 3 eps^2 x
    return fma(d, h, g);                                        // the seed's h is good enough for the correction: error 1.5 eps^3 + rounding
}
#endif

// ---- Eq.23 for p = cs2*e in closed form with the admissibility guard A12.  :227-234
// Returns the three velocity components and the pressure.
template <int EK = 0>
__device__ __forceinline__ void velocity_pressure(const Eos& q, double E, double Mx, double My, double Mz, double R,
                                                  double& vx, double& vy, double& vz, double& e, double& p)
{
    double M2 = Mx * Mx + My * My + Mz * Mz;
    double cap = V_CAP * E;
    if (!(E > E_VACUUM)) {                        // vacuum (or NaN): v = 0, p = 0
        bool nan = E != E;
        vx = vy = vz = nan ? E : 0.0; e = E; p = nan ? E : 0.0;
        return;
    }
    if (M2 > cap * cap) {                         // superluminal: rescale M to |M| = V_CAP*E, keep direction
        double s = cap / sqrt(M2);
        Mx *= s; My *= s; Mz *= s;
        M2 = Mx * Mx + My * My + Mz * Mz;
    }
    if (EK != 0) {                                // tabulated EOS: Newton on the speed, then v_j = M_j v/|M|
#ifdef MF_STRICT
        const double M = sqrt(M2);
#else
        const double M = M2 > 1e-280 ? sqrt_pos(M2) : sqrt(M2);            // (Newton root: normal, positive arguments only)
#endif
        if (M == 0.0) { vx = vy = vz = 0.0; e = E; p = eos_table_eval(table_of(q), E, R).p; return; }
        const SpeedEP r = solve_speed(table_of(q), E, M, R);
#ifdef MF_STRICT
        const double s = r.v / M;
#else
        const double s = M > 1e-140 ? r.v * rcp_pos(M) : r.v / M;
#endif
        vx = Mx * s; vy = My * s; vz = Mz * s; e = r.e; p = r.p;
        return;
    }
    double Q = sqrt_pos(q.c1sq * E * E - q.four_cs2 * M2);
    double inv = two_over(q.c1 * E + Q);
    vx = Mx * inv; vy = My * inv; vz = Mz * inv;
#ifdef MF_STRICT
    e = E - (Mx * vx + My * vy + Mz * vz);        // the oracle's order
#else
    e = fma(-M2, inv, E);                         // M.v = |M|^2 inv
#endif
    p = q.cs2 * e;
}

// ---- Eq.3 :53-59: F_d(U) = ((E+p)v_d, M_j v_d + p delta_jd, R v_d)
template <int D, int EK = 0>
__device__ __forceinline__ void flux_d(const Eos& q, const double (&U)[5], double (&F)[5])
{
    double vx, vy, vz, e, p;
    velocity_pressure<EK>(q, U[0], U[1], U[2], U[3], U[4], vx, vy, vz, e, p);
    double vd = D == 0 ? vx : (D == 1 ? vy : vz);
    F[0] = (U[0] + p) * vd;
    F[1] = U[1] * vd;
    F[2] = U[2] * vd;
    F[3] = U[3] * vd;
    F[1 + D] += p;
    F[4] = U[4] * vd;
}

#ifndef MF_STRICT
// Product build: the same flux on the admissible fast path with the minimum number of FP64-pipe instructions (24):
//   Q/2 = sqrt(c1^2/4 E^2 - cs2 |M|^2),  inv = 1/(c1/2 E + Q/2) = 2/(c1 E + Q),  v_d = M_d inv,  p = cs2 (E - |M|^2 inv),
//   F_E = M_d  (reading A15: (E+p) v_d == M_d identically when the guard is inactive).
// Returns false when the state needs the guarded general path (vacuum, NaN, |M| > V_CAP E); the caller then calls flux_d.
// The vacuum test compares the high word of E as an integer (conservative: borderline values take the general path).
template <int D>
__device__ __forceinline__ bool flux_fast(const Eos& q, const double (&U)[5], double (&F)[5])
{
    const double E = U[0];
    const double M2 = fma(U[3], U[3], fma(U[2], U[2], U[1] * U[1]));
    const double EE = E * E;
    // admissible and not vacuum, decided on the integer pipe: E > ~1e-12 (high word) and |M|^2 < E^2 by at least one unit of the
    // high word (2^-21 relative, so |M| <= V_CAP E holds with room to spare); anything closer takes the guarded general path
    // The words are compared as UNSIGNED numbers with one unit of room (the high word of |M|^2 at least TWO below that of E^2): a NaN of
    // either sign in M (CUDA's canonical NaN has the sign bit set) is larger than every finite E^2 and fails the test.
    const bool ok = (__double2hiint(E) > 0x3D719799) && ((unsigned int)__double2hiint(M2) + 1u < (unsigned int)__double2hiint(EE));
    const double Qh = sqrt_pos(fma(q.cs2, -M2, q.qc1sq * EE));      // (the sign on the register operand: cs2 stays a uniform-register operand)
    double y;
    {
        const double x = fma(q.hc1, E, Qh);
        asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
        const double e1 = fma(-x, y, 1.0);
        y = fma(y, fma(e1, e1, e1), y);
    }
    const double vd = U[1 + D] * y;
    const double p = q.cs2 * fma(-M2, y, E);
    F[0] = U[1 + D];
    F[1] = U[1] * vd;
    F[2] = U[2] * vd;
    F[3] = U[3] * vd;
    F[1 + D] += p;
    F[4] = U[4] * vd;
    return ok;
}
#endif

// flux evaluation used outside MUSTA (Hancock predictor): fast path with the guarded fallback
template <int D, int EK = 0>
__device__ __forceinline__ void flux_eval(const Eos& q, const double (&U)[5], double (&F)[5])
{
#ifdef MF_STRICT
    flux_d<D, EK>(q, U, F);
#else
    if (EK != 0) { flux_d<D, EK>(q, U, F); return; }
    if (!flux_fast<D>(q, U, F)) flux_d<D>(q, U, F);
#endif
}

// ---- MUSTA_k with FORCE-alpha, steps 1-5 :123-135, Eq.8-11 :130-149 (A1: Richtmyer state uses the flux difference)
// A, B are U_L^(0), U_R^(0) on entry and are overwritten.
// The stage coefficients: lam, c_lw = alpha lam/2, c_lf = 1/(2 alpha lam) as the step computed them (A16), and the negated multiples the
// product form multiplies with.  Taken from constant memory they are uniform-register operands (mf_stepconst.cuh).
struct MustaCoef {
    double lam, c_lw, c_lf;
    double nc_lw, nc2_lf, nhlam;      // -c_lw, -2 c_lf, -lam/2
};

template <int D, int EK = 0>
__device__ __forceinline__ void musta_flux(const Eos& q, int k, const MustaCoef& mc, double (&A)[5], double (&B)[5], double (&F)[5])
{
    const double lam = mc.lam, c_lw = mc.c_lw, c_lf = mc.c_lf;
    (void)lam; (void)c_lw; (void)c_lf;
#ifndef MF_STRICT
    if (EK == 0) {
    // The same stages on the mean s = (A+B)/2 and the half jump d = (B-A)/2 of the two states, with the constant factors folded:
    //   Eq.10  U^lw = s - c_lw (F_B - F_A)
    //   Eq.9,11  2F = F^lw + (F_A + F_B)/2 - 2 c_lf d
    //   Eq.8   s' = s - (lam/2)(F_B - F_A),   d' = d - (lam/2)(F_A + F_B - 2F)
    // 10 FP64 instructions per component and stage (6 in the last) instead of 13 (9), and the 24-instruction flux.
    // Every multiplier below is one of mc's scalars, so that each DFMA reads at most two registers (a DFMA with three distinct register
    // operands holds the FP64 pipe for 3 cycles instead of 2).
    const double nc_lw = mc.nc_lw, nc2_lf = mc.nc2_lf, nhlam = mc.nhlam;
    double s[5], d[5];
#pragma unroll
    for (int c = 0; c < 5; ++c) { s[c] = 0.5 * (A[c] + B[c]); d[c] = 0.5 * (B[c] - A[c]); }
    for (int l = 0;; ++l) {
        double FA[5], FB[5], W[5];
        const bool okA = flux_fast<D>(q, A, FA);
        const bool okB = flux_fast<D>(q, B, FB);
        if (!(okA && okB)) { flux_d<D>(q, A, FA); flux_d<D>(q, B, FB); }                     // rare: guarded general path
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            const double FD = FB[c] - FA[c];
            FA[c] = FA[c] + FB[c];                                                            // F_A + F_B from here on
            FB[c] = FD;                                                                       // F_B - F_A from here on
            W[c] = fma(nc_lw, FD, s[c]);                                                      // Eq.10
        }
        if (!flux_fast<D>(q, W, F)) flux_d<D>(q, W, F);                                       // F^lw
#pragma unroll
        for (int c = 0; c < 5; ++c) F[c] = fma(nc2_lf, d[c], fma(0.5, FA[c], F[c]));          // 2F: Eq.9 with Eq.11 inside
        if (l == k) break;
#pragma unroll
        for (int c = 0; c < 5; ++c) {                                                         // Eq.8
            s[c] = fma(nhlam, FB[c], s[c]);
            d[c] = fma(nhlam, FA[c] - F[c], d[c]);
            A[c] = s[c] - d[c];
            B[c] = s[c] + d[c];
        }
    }
#pragma unroll
    for (int c = 0; c < 5; ++c) F[c] = 0.5 * F[c];
    } else
#endif
    for (int l = 0;; ++l) {
        double FA[5], FB[5], W[5];
        flux_d<D, EK>(q, A, FA);
        flux_d<D, EK>(q, B, FB);
#pragma unroll
        for (int c = 0; c < 5; ++c) W[c] = 0.5 * (A[c] + B[c]) - c_lw * (FB[c] - FA[c]);      // Eq.10
        flux_d<D, EK>(q, W, F);                                                               // F^lw
#pragma unroll
        for (int c = 0; c < 5; ++c) {
            double Flf = 0.5 * (FA[c] + FB[c]) - c_lf * (B[c] - A[c]);                        // Eq.11
            F[c] = 0.5 * (F[c] + Flf);                                                        // Eq.9
        }
        if (l == k) break;
#pragma unroll
        for (int c = 0; c < 5; ++c) {                                                         // Eq.8
            A[c] = A[c] - lam * (F[c] - FA[c]);
            B[c] = B[c] - lam * (FB[c] - F[c]);
        }
    }
}

// ---- a2: local signal speed (|v|+cs)/(1+|v|cs) (A10) and the state check behind MF_ESTATE
template <int EK = 0>
__device__ __forceinline__ double signal_speed(const Eos& q, double E, double Mx, double My, double Mz, double R, int& bad)
{
#ifndef MF_STRICT
    if (EK == 0) {
        // Product build, p = cs2*e: the common case - a finite, admissible, non-vacuum state - is recognised on the high words (E in (1e-12,
        // 1e154), |M|^2 below E^2 by a unit of the high word, R finite) and costs ~35 FP64 instructions: |v| = |M| y with the fast flux's
        // root and reciprocal, one more Newton root, one more Newton reciprocal.  Everything else takes the general path below.
        const double M2 = fma(Mz, Mz, fma(My, My, Mx * Mx)), EE = E * E;
        const int hEE = __double2hiint(EE);
        // (unsigned compare with a unit of room: a NaN of either sign in M compares above every finite E^2 and takes the general path)
        if (__double2hiint(E) > 0x3D719799 && hEE < 0x7ff00000 && (unsigned int)__double2hiint(M2) + 1u < (unsigned int)hEE &&
            (__double2hiint(R) & 0x7fffffff) < 0x7ff00000) {
            const double Qh = sqrt_pos(fma(-q.cs2, M2, q.qc1sq * EE));
            const double y = rcp_pos(fma(q.hc1, E, Qh));
            const double av2 = M2 * (y * y);
            const double av = av2 > 1e-280 ? sqrt_pos(av2) : 0.0;
            return (av + q.cs) * rcp_pos(fma(av, q.cs, 1.0));
        }
    }
#endif
    bool finite = isfinite(E) && isfinite(Mx) && isfinite(My) && isfinite(Mz) && isfinite(R);
    if (!finite) { bad = 1; return 0.0; }
    if (E > E_VACUUM && Mx * Mx + My * My + Mz * Mz > E * E) bad = 1;
    double vx, vy, vz, e, p;
    velocity_pressure<EK>(q, E, Mx, My, Mz, R, vx, vy, vz, e, p);
    double av = sqrt(vx * vx + vy * vy + vz * vz);
    double cs = q.cs;
    if (EK != 0) {                            // adiabatic sound speed of the table: cs^2 = p_e + n p_n/(e+p)
        double cs2t = 0.0;
        if (e > 0.0) {
            const double nn = R * sqrt(1.0 - av * av);
            const EosValue w = eos_table_eval(table_of(q), e, nn);
            cs2t = w.p_e + nn * w.p_n / (e + w.p);
        }
        cs = cs2t > 0.0 ? sqrt(cs2t) : 0.0;
    }
    return (av + cs) / (1.0 + av * cs);
}

// ---- reading A19 ("saved as 5 single precision floating-point numbers per lattice cell"): the state registers hold elements
// of type ST (double, or float in 32-bit state mode).  The structs carry double pointers whatever ST is (the host computes them with the
// element size of the mode); a load widens to double, a store rounds to nearest even, and every operation in between is fp64.
template <class ST>
__device__ __forceinline__ double ld_state(const double* base, unsigned int o) { return (double)reinterpret_cast<const ST*>(base)[o]; }
template <class ST>
__device__ __forceinline__ void st_state(double* base, unsigned int o, double x) { reinterpret_cast<ST*>(base)[o] = (ST)x; }
template <class ST>
__device__ __forceinline__ double as_stored(double x) { return (double)(ST)x; }      // the value a later load of the stored element returns

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

// idx -> (a, b, c) with idx = a + d0*(b + d1*c), idx < 2^32 (mf_create refuses larger grids), by two multiply-shift divisions.
template <class FD>
__device__ __forceinline__ unsigned int fastdiv(unsigned int n, const FD& f)
{
    const unsigned int t = __umulhi(f.mul, n);
    return (t + ((n - t) >> f.sh1)) >> f.sh2;
}
template <class FD>
__device__ __forceinline__ void unflatten3(unsigned int idx, const FD& d0, const FD& d1, int& a, int& b, int& c)
{
    const unsigned int r = fastdiv(idx, d0), q2 = fastdiv(r, d1);
    a = (int)(idx - r * d0.d); b = (int)(r - q2 * d1.d); c = (int)q2;
}

__device__ __forceinline__ int bc_index(int i, int n, int periodic)
{
    if (periodic) { i = i < 0 ? i + n : i; return i >= n ? i - n : i; }     // |offset| <= 2 < n
    return min(max(i, 0), n - 1);
}

} // namespace mf
