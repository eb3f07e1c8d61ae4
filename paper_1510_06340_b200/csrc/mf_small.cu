// mf_small.cu — small 1D grids (MF_PATH_SMALL): the whole step loop in ONE launch of ONE CTA.
//
// Config 1 (400 cells) is launch bound on every other path: a step is six launches of a few microseconds of work each (55 us eagerly, 16-18
// us when mf_step replays a captured CUDA graph).  Here a single block owns the whole grid - thread t is extended cell t, interface t and
// cell t in turn - keeps the face data and the interface fluxes of a stage in shared memory, synchronises with __syncthreads between the
// cell stage (a1+a3+a4), the interface fluxes (a5+a6) and the combine (a7+a8), takes S_max and dt at the start of every step with a block
// reduction (a2), and runs all n steps of an mf_step / mf_step_dt call before it returns: one launch per call, nothing else.
// The state registers stay in global memory (they fit L1) and rotate exactly as run_step rotates them, so every other call of the ABI sees
// what it would see after the staged path.  Per cell and per interface the arithmetic is the staged kernels' in the same order (the same
// device functions): the strict build is bit-identical to the oracle, dt included.
// 1D grids with an active x axis, nx + 2 <= 768 (80 registers per thread), p = cs2*e, one event, fp64 state, three state registers.
#include "mf_kernels.h"
#include "mf_blocks.cuh"

namespace mf {

namespace {

struct SmallArgs {
    int limiter, predictor, k, rk;
    int mode;            // 0: dt = value*dx/S_max (cfl), 1: dt = value
    int nsteps, cur;     // steps to run; register that holds U^n at entry
    double value, alpha;
};

// block-wide max of a non-negative double and OR of a flag (every thread calls)
__device__ __forceinline__ void block_max_or(double& x, int& flag, double* s_max, int* s_flag)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        x = fmax(x, __shfl_xor_sync(0xffffffffu, x, off));
        flag |= __shfl_xor_sync(0xffffffffu, flag, off);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5, nw = (blockDim.x + 31) >> 5;
    if (lane == 0) { s_max[warp] = x; s_flag[warp] = flag; }
    __syncthreads();
    double m = 0.0;
    int f = 0;
    for (int w = 0; w < nw; ++w) { m = fmax(m, s_max[w]); f |= s_flag[w]; }
    x = m; flag = f;
    __syncthreads();
}

// cell stage of extended cell ie (interior cell ie - 1, may be a ghost): the 1D case of k_cell_stage
template <int LIM>
__device__ __forceinline__ void small_cell(const Grid& g, const Eos& q, int predictor, double hl, const double* const (&V)[5], int ie,
                                           double (*s_lo)[5], double (*s_hi)[5])
{
    const int n = g.n[0];
    const int c = ie - 1, cc = bc_index(c, n, g.periodic), cm = bc_index(c - 1, n, g.periodic), cp = bc_index(c + 1, n, g.periodic);
    double U0[5], Um[5], Up[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { U0[v] = V[v][cc]; Um[v] = V[v][cm]; Up[v] = V[v][cp]; }
#ifdef MF_STRICT
    double UL[5], UR[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double a = U0[v] - Um[v], b = Up[v] - U0[v];
        const double s = slope2<LIM>(a, b);                                // Eq.15-17
        UL[v] = U0[v] - 0.5 * s;                                           // Eq.12 :161
        UR[v] = U0[v] + 0.5 * s;
    }
    if (predictor) {                                                        // Eq.13, one direction
        double Fl[5], Fr[5];
        flux_eval<0>(q, UL, Fl); flux_eval<0>(q, UR, Fr);
#pragma unroll
        for (int v = 0; v < 5; ++v) { const double delta = hl * (Fl[v] - Fr[v]); UL[v] += delta; UR[v] += delta; }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) { s_lo[ie][v] = UL[v]; s_hi[ie][v] = UR[v]; }          // lo = U~L, hi = U~R
#else
    double H[5], W[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) { H[v] = half_slope2<LIM>(U0[v] - Um[v], Up[v] - U0[v]); W[v] = U0[v]; }
    if (predictor) {
        double UL[5], UR[5], Fl[5], Fr[5], acc[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
#pragma unroll
        for (int v = 0; v < 5; ++v) { UL[v] = U0[v] - H[v]; UR[v] = U0[v] + H[v]; }
        flux_eval<0>(q, UL, Fl); flux_eval<0>(q, UR, Fr);
#pragma unroll
        for (int v = 0; v < 5; ++v) { acc[v] += Fl[v] - Fr[v]; W[v] = fma(hl, acc[v], U0[v]); }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) { s_lo[ie][v] = H[v]; s_hi[ie][v] = W[v]; }            // lo = H_x, hi = W
#endif
}

__device__ __forceinline__ void small_cell_rt(int lim, const Grid& g, const Eos& q, int predictor, double hl, const double* const (&V)[5], int ie,
                                              double (*s_lo)[5], double (*s_hi)[5])
{
    switch (lim) {
    case LIM_NONE:      small_cell<LIM_NONE>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    case LIM_MINMOD:    small_cell<LIM_MINMOD>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    case LIM_SUPERBEE:  small_cell<LIM_SUPERBEE>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    case LIM_VANALBADA: small_cell<LIM_VANALBADA>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    case LIM_VANLEER:   small_cell<LIM_VANLEER>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    case LIM_MC:        small_cell<LIM_MC>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    default:            small_cell<LIM_FIRST>(g, q, predictor, hl, V, ie, s_lo, s_hi); break;
    }
}

// MAXT: the largest block this instantiation is launched with (512: up to 128 registers per thread, no spills; 768: 80)
template <int MAXT>
__global__ void __launch_bounds__(MAXT, 1)
k_small1d(Grid g, Eos q, SmallArgs a, double* U0p, double* U1p, double* U2p, Source src, StepState* ds)
{
    extern __shared__ double sm[];                       // [n+2][5] lo, [n+2][5] hi, [n+1][5] F
    const int n = g.n[0], t = threadIdx.x;
    double (*s_lo)[5] = reinterpret_cast<double (*)[5]>(sm);
    double (*s_hi)[5] = reinterpret_cast<double (*)[5]>(sm + 5 * (n + 2));
    double (*s_F)[5] = reinterpret_cast<double (*)[5]>(sm + 10 * (n + 2));
    __shared__ double s_max[24];
    __shared__ int s_flag[24];
    double* const regs[3] = { U0p, U1p, U2p };
    int cur = a.cur;
    double tnow = ds->t;
    long long steps = ds->steps;
    double dt = 0.0, lam = 0.0, hl = 0.0, c_lw = 0.0, c_lf = 0.0;

    for (int step = 0; step < a.nsteps; ++step) {
        const double* Un = regs[cur];
        // ------------------------------------------------------------ a2: S_max of U^n, status, dt (the arithmetic of k_cfl / k_begin_step)
        {
            double s = 0.0;
            int bad = 0;
            if (t < n) s = signal_speed<0>(q, Un[t], Un[n + t], Un[2 * n + t], Un[3 * n + t], Un[4 * n + t], bad);
            block_max_or(s, bad, s_max, s_flag);           // (with a fixed dt too: the state check behind MF_ESTATE runs on every U^n)
            if (bad && t == 0) atomicOr(&ds->status, 1);
            dt = a.mode == 0 ? a.value * g.dx / s : a.value;                   // A10
            lam = dt / g.dx;
            hl = 0.5 * lam;
            c_lw = 0.5 * a.alpha * lam;                                        // A16: in this order
            c_lf = 0.5 / (a.alpha * lam);
        }
        MustaCoef mc;
        mc.lam = lam; mc.c_lw = c_lw; mc.c_lf = c_lf; mc.nc_lw = -c_lw; mc.nc2_lf = -2.0 * c_lf; mc.nhlam = -0.5 * lam;
        const int nstage = a.rk == 2 ? 2 : 3;
        double* Ra = regs[(cur + 1) % 3];
        double* Rb = regs[(cur + 2) % 3];
        for (int st = 0; st < nstage; ++st) {
            // the stages of run_step: (input state, RK form, output register)
            Stage sg;
            const double* Vp; double* outp;
            if (a.rk == 2) {
                if (st == 0) { sg = Stage{ 0, 1.0, 0.0, 1.0, 0.0, 0 }; Vp = Un; outp = Ra; }
                else         { sg = Stage{ 1, 0.5, 0.5, 1.0, 1.0, 0 }; Vp = Ra; outp = Rb; }
            } else {
                if (st == 0)      { sg = Stage{ 0, 1.0, 0.0, 1.0, 0.0, 0 }; Vp = Un; outp = Ra; }
                else if (st == 1) { sg = Stage{ 2, 0.75, 0.25, 0.25, 1.0, 0 }; Vp = Ra; outp = Rb; }
                else              { sg = Stage{ 2, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 0.5, 0 }; Vp = Rb; outp = Ra; }
            }
            const double* const V[5] = { Vp, Vp + n, Vp + 2 * n, Vp + 3 * n, Vp + 4 * n };
            // ---------------------------------------------------- a1 + a3 + a4: extended cells 0 .. n+1
            if (t < n + 2) small_cell_rt(a.limiter, g, q, a.predictor, hl, V, t, s_lo, s_hi);
            __syncthreads();
            // ---------------------------------------------------- a5 + a6: interfaces 0 .. n (between extended cells t and t+1)
            if (t < n + 1) {
                double A[5], B[5], F[5];
#ifdef MF_STRICT
#pragma unroll
                for (int v = 0; v < 5; ++v) { A[v] = s_hi[t][v]; B[v] = s_lo[t + 1][v]; }
#else
#pragma unroll
                for (int v = 0; v < 5; ++v) { A[v] = s_hi[t][v] + s_lo[t][v]; B[v] = s_hi[t + 1][v] - s_lo[t + 1][v]; }
#endif
                musta_flux<0, 0>(q, a.k, mc, A, B, F);
#pragma unroll
                for (int v = 0; v < 5; ++v) s_F[t][v] = F[v];
            }
            __syncthreads();
            // ---------------------------------------------------- a7 + a8: cells 0 .. n-1
            if (t < n) {
                double S = 0.0;
                if (src.on) S = jet_source(g, src, t, 0, 0, tnow + sg.ts * dt);
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    const double acc = s_F[t + 1][v] - s_F[t][v];
#ifdef MF_STRICT
                    double L = -acc / g.dx;                                    // Eq.1 :43
#else
                    double L = -acc * g.inv_dx;
#endif
                    if (src.on && v < 2) L = L + S;
                    const double ua = Un[v * n + t], ub = Vp[v * n + t];
                    outp[v * n + t] = rk_form(sg, ua, ub, dt, L);
                }
            }
            __syncthreads();                                                    // the new stage state is complete (global memory, one block)
        }
        cur = a.rk == 2 ? (cur + 2) % 3 : (cur + 1) % 3;
        tnow = tnow + dt;
        steps += 1;
    }
    {                                                     // the last state is checked as well (the staged path does it in its last combine)
        const double* Un = regs[cur];
        double s = 0.0;
        int bad = 0;
        if (t < n) s = signal_speed<0>(q, Un[t], Un[n + t], Un[2 * n + t], Un[3 * n + t], Un[4 * n + t], bad);
        block_max_or(s, bad, s_max, s_flag);
        if (bad && t == 0) atomicOr(&ds->status, 1);
    }
    if (t == 0) {
        ds->t = tnow; ds->dt = dt; ds->lam = lam; ds->hl = hl; ds->c_lw = c_lw; ds->c_lf = c_lf; ds->steps = steps;
        ds->smax_bits = 0ull;                                                   // the accumulator stays empty: the next reduction starts clean
    }
}

} // namespace

bool small_supported(const Grid& g, int eos_kind)
{
    return g.act[0] && !g.act[1] && !g.act[2] && g.n[0] + 2 <= 768 && g.nev == 1 && eos_kind == 0 && !g.state32;
}

// n steps in one launch; `cur` is the register holding U^n; returns the number of launches (1) or 0 on a launch configuration error
int launch_small_steps(const Grid& g, const Eos& q, int limiter, int predictor, int k, int rk, double alpha, int mode, double value, int nsteps,
                       int cur, double* const U[3], Source src, StepState* ds, cudaStream_t st)
{
    SmallArgs a;
    a.limiter = limiter; a.predictor = predictor; a.k = k; a.rk = rk; a.mode = mode; a.nsteps = nsteps; a.cur = cur; a.value = value; a.alpha = alpha;
    const int n = g.n[0];
    const int threads = ((n + 2 + 31) / 32) * 32;
    const size_t smem = sizeof(double) * (size_t)(15 * (n + 2));
    static DeviceOnce once;
    if (once.first()) {
        cudaFuncSetAttribute(k_small1d<512>, cudaFuncAttributeMaxDynamicSharedMemorySize, 15 * 512 * (int)sizeof(double));
        cudaFuncSetAttribute(k_small1d<768>, cudaFuncAttributeMaxDynamicSharedMemorySize, 15 * 768 * (int)sizeof(double));
    }
    if (threads <= 512) k_small1d<512><<<1, threads, smem, st>>>(g, q, a, U[0], U[1], U[2], src, ds);
    else k_small1d<768><<<1, threads, smem, st>>>(g, q, a, U[0], U[1], U[2], src, ds);
    return 1;
}

} // namespace mf
