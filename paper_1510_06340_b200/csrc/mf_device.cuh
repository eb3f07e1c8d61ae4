// mf_device.cuh — per-cell / per-interface device arithmetic of the MUSTA-FORCE step (fp64, sm_100a).
// Everything here lives in registers; the kernels in mf_kernels.cu decide where operands come from.
// Citations are PAPER.md lines; readings A1..A17 are listed in DESIGN.md.
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
};

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
    else if (LIM == LIM_SUPERBEE) m = fmax(fmin(2.0 * fb, fa), fmin(fb, 2.0 * fa));// Eq.19 :203
    else m = fmin(fmin(2.0 * fa, 2.0 * fb), 0.5 * fabs(a + b));                    // MC (A8)
    m = copysign(m, a);
    return ab > 0.0 ? m : 0.0;
}

// ---- fp64 reciprocal and square root for the flux core.
// The product build uses branch-free Newton sequences seeded by the MUFU approximations (rcp/rsqrt.approx.ftz.f64,
// ~20 good bits): 3 and 7 FP64-pipe instructions instead of the 9 and 14.5 issue slots that the IEEE-rounded '/' and
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
__device__ __forceinline__ double sqrt_pos(double x)          // sqrt(x) for normal, positive x
{
    double y;
    asm("rsqrt.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(x));
    double g = x * y, h = 0.5 * y;
    double r = fma(-g, h, 0.5);
    g = fma(g, r, g);
    h = fma(h, r, h);
    double d = fma(-g, g, x);
    return fma(d, h, g);
}
#endif

// ---- Eq.23 for p = cs2*e in closed form with the admissibility guard A12.  :227-234
// Returns the three velocity components and the pressure.
__device__ __forceinline__ void velocity_pressure(const Eos& q, double E, double Mx, double My, double Mz,
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
template <int D>
__device__ __forceinline__ void flux_d(const Eos& q, const double (&U)[5], double (&F)[5])
{
    double vx, vy, vz, e, p;
    velocity_pressure(q, U[0], U[1], U[2], U[3], vx, vy, vz, e, p);
    double vd = D == 0 ? vx : (D == 1 ? vy : vz);
    F[0] = (U[0] + p) * vd;
    F[1] = U[1] * vd;
    F[2] = U[2] * vd;
    F[3] = U[3] * vd;
    F[1 + D] += p;
    F[4] = U[4] * vd;
}

#ifndef MF_STRICT
// Product build: the same flux on the admissible fast path with the minimum number of FP64-pipe instructions (26):
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
    const bool ok = (__double2hiint(E) > 0x3D719799) && (M2 <= q.vcap2 * EE);
    const double Qh = sqrt_pos(fma(-q.cs2, M2, q.qc1sq * EE));
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
template <int D>
__device__ __forceinline__ void flux_eval(const Eos& q, const double (&U)[5], double (&F)[5])
{
#ifdef MF_STRICT
    flux_d<D>(q, U, F);
#else
    if (!flux_fast<D>(q, U, F)) flux_d<D>(q, U, F);
#endif
}

// ---- MUSTA_k with FORCE-alpha, steps 1-5 :123-135, Eq.8-11 :130-149 (A1: Richtmyer state uses the flux difference)
// A, B are U_L^(0), U_R^(0) on entry and are overwritten.
template <int D>
__device__ __forceinline__ void musta_flux(const Eos& q, int k, double lam, double c_lw, double c_lf,
                                           double (&A)[5], double (&B)[5], double (&F)[5])
{
#ifdef MF_STRICT
    for (int l = 0;; ++l) {
        double FA[5], FB[5], W[5];
        flux_d<D>(q, A, FA);
        flux_d<D>(q, B, FB);
#pragma unroll
        for (int c = 0; c < 5; ++c) W[c] = 0.5 * (A[c] + B[c]) - c_lw * (FB[c] - FA[c]);      // Eq.10
        flux_d<D>(q, W, F);                                                                   // F^lw
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
#else
    // same formulas with the constant factors folded so that every line is one FP64 instruction
    const double hc_lf = 0.5 * c_lf;
    for (int l = 0;; ++l) {
        double FA[5], FB[5], W[5];
        const bool okA = flux_fast<D>(q, A, FA);
        const bool okB = flux_fast<D>(q, B, FB);
        if (!(okA && okB)) { flux_d<D>(q, A, FA); flux_d<D>(q, B, FB); }                     // rare: guarded general path
#pragma unroll
        for (int c = 0; c < 5; ++c) W[c] = fma(0.5, A[c] + B[c], -(c_lw * (FB[c] - FA[c])));  // Eq.10
        if (!flux_fast<D>(q, W, F)) flux_d<D>(q, W, F);                                       // F^lw
#pragma unroll
        for (int c = 0; c < 5; ++c)                                                           // Eq.9 with Eq.11 inside
            F[c] = fma(-hc_lf, B[c] - A[c], fma(0.25, FA[c] + FB[c], 0.5 * F[c]));
        if (l == k) break;
#pragma unroll
        for (int c = 0; c < 5; ++c) {                                                         // Eq.8
            A[c] = fma(-lam, F[c] - FA[c], A[c]);
            B[c] = fma(-lam, FB[c] - F[c], B[c]);
        }
    }
#endif
}

// ---- a2: local signal speed (|v|+cs)/(1+|v|cs) (A10) and the state check behind MF_ESTATE
__device__ __forceinline__ double signal_speed(const Eos& q, double E, double Mx, double My, double Mz, double R, int& bad)
{
    bool finite = isfinite(E) && isfinite(Mx) && isfinite(My) && isfinite(Mz) && isfinite(R);
    if (!finite) { bad = 1; return 0.0; }
    if (E > E_VACUUM && Mx * Mx + My * My + Mz * Mz > E * E) bad = 1;
    double vx, vy, vz, e, p;
    velocity_pressure(q, E, Mx, My, Mz, vx, vy, vz, e, p);
    double av = sqrt(vx * vx + vy * vy + vz * vz);
    return (av + q.cs) / (1.0 + av * q.cs);
}

__device__ __forceinline__ void prefetch_l2(const void* p) { asm volatile("prefetch.global.L2 [%0];" :: "l"(p)); }

__device__ __forceinline__ int bc_index(int i, int n, int periodic)
{
    if (periodic) { i = i < 0 ? i + n : i; return i >= n ? i - n : i; }     // |offset| <= 2 < n
    return min(max(i, 0), n - 1);
}

} // namespace mf
