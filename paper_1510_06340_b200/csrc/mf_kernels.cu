// mf_kernels.cu — staged path (MF_PATH_STAGED) and the small kernels every path shares:
// CFL reduction (a2), per-step scalars, cell stage (a3+a4), interface flux stage (a5+a6), combine (a7+a8),
// prim<->con conversions, totals.  Boundary handling (a1) is index mapping in the loads: no stored ghosts.
#include "mf_kernels.h"
#include <cstdio>
#include "mf_blocks.cuh"
#include "mf_stepconst.cuh"

namespace mf {

// threads per block / resident blocks per SM of the three hot kernels of the staged path (24 warps per SM at 80 registers)
#ifndef MF_CELL_TPB
#define MF_CELL_TPB 128
#endif
#ifndef MF_FLUX_TPB
#define MF_FLUX_TPB 256
#endif
#ifndef MF_XC_TPB
#define MF_XC_TPB 128
#endif
#ifndef MF_XC_MINB
#define MF_XC_MINB 5        // x kernel: 5 blocks of 128 threads (96 registers): the combine holds its 30 operands in registers at once
#endif
#ifndef MF_CELL_PF
#define MF_CELL_PF (148 * 768)   // cells ahead (in the plane above) whose lines a cell-stage thread prefetches to L2: one wave of resident threads; 0 = off
#endif
#ifndef MF_YZ_INTERLEAVE
#define MF_YZ_INTERLEAVE 1       // y and z flux blocks alternate in the merged launch (W is read from HBM once for both)
#endif
#ifndef MF_CELL_MINB
#define MF_CELL_MINB (768 / MF_CELL_TPB)
#endif
#ifndef MF_FLUX_MINB
#define MF_FLUX_MINB (768 / MF_FLUX_TPB)
#endif
constexpr int CT = MF_CELL_TPB, FT = MF_FLUX_TPB, XT = MF_XC_TPB;

static inline unsigned int blocks_for(long long n, int tpb) { return (unsigned int)((n + tpb - 1) / tpb); }


// =========================================================================== a2: CFL reduction
template <int EK, class ST>
__global__ void __launch_bounds__(TPB) k_cfl(Grid g, Eos q, CState5 U, StepState* ds)
{
    double smax = 0.0;
    int bad = 0;
    const unsigned int eo = blockIdx.y * (unsigned int)g.ncell;       // this block's event
    const unsigned int stride = gridDim.x * blockDim.x;
    for (unsigned int i = blockIdx.x * blockDim.x + threadIdx.x; i < (unsigned int)g.ncell; i += stride) {
        const unsigned int o = eo + i;
        double s = signal_speed<EK>(q, ld_state<ST>(U.q[0], o), ld_state<ST>(U.q[1], o), ld_state<ST>(U.q[2], o), ld_state<ST>(U.q[3], o),
                                    ld_state<ST>(U.q[4], o), bad);
        smax = fmax(smax, s);
    }
    block_reduce_smax(smax, bad, ds + blockIdx.y);
}

int launch_cfl(const Grid& g, const Eos& q, CState5 U, StepState* ds, int num_sms, cudaStream_t st)
{
    unsigned int nb = blocks_for(g.ncell, TPB);
    unsigned int cap = (unsigned int)num_sms * 8u / (unsigned int)g.nev;
    if (cap < 1u) cap = 1u;
    if (nb > cap) nb = cap;
    const dim3 grid(nb, g.nev);
    if (g.state32) { if (q.kind) k_cfl<1, float><<<grid, TPB, 0, st>>>(g, q, U, ds); else k_cfl<0, float><<<grid, TPB, 0, st>>>(g, q, U, ds); }
    else { if (q.kind) k_cfl<1, double><<<grid, TPB, 0, st>>>(g, q, U, ds); else k_cfl<0, double><<<grid, TPB, 0, st>>>(g, q, U, ds); }
    return 1;
}

// =========================================================================== per-step scalars
// one thread per event of the batch
__global__ void k_begin_step(StepState* ds, StepConst* dsc, int nev, int mode, double value, double dx, double alpha)
{
    const int ev = blockIdx.x * blockDim.x + threadIdx.x;
    if (ev >= nev) return;
    ds += ev;
    dsc += ev;
    double dt;
    if (mode == 0) {
        double smax = __longlong_as_double((long long)ds->smax_bits);
        dt = value * dx / smax;                                   // A10
    } else {
        dt = value;
    }
    double lam = dt / dx;
    ds->dt = dt;
    ds->lam = lam;
    ds->hl = 0.5 * lam;
    ds->c_lw = 0.5 * alpha * lam;                                 // A16: computed once per step, in this order
    ds->c_lf = 0.5 / (alpha * lam);
    ds->smax_bits = 0ull;
    // the same scalars, with the negated multiples of the product build's MUSTA, for the constant-memory copy (mf_stepconst.cuh)
    dsc->dt = dt; dsc->lam = lam; dsc->hl = ds->hl; dsc->c_lw = ds->c_lw; dsc->c_lf = ds->c_lf;
    dsc->nc_lw = -ds->c_lw; dsc->nc2_lf = -2.0 * ds->c_lf; dsc->nhlam = -0.5 * lam;
}

__global__ void k_end_step(StepState* ds, int nev)
{
    const int ev = blockIdx.x * blockDim.x + threadIdx.x;
    if (ev >= nev) return;
    ds += ev;
    ds->t = ds->t + ds->dt;
    ds->steps += 1;
#ifdef MF_COUNT_EVALS
    if (ev == 0) printf("MF_COUNT_EVALS step %lld: solves %llu full %llu incremental %llu fallback %llu\n", ds->steps, g_eval_count[0], g_eval_count[1],
                        g_eval_count[2], g_eval_count[3]);
#endif
}

__global__ void k_reset(StepState* ds, int nev)
{
    const int ev = blockIdx.x * blockDim.x + threadIdx.x;
    if (ev >= nev) return;
    ds += ev;
    ds->t = 0.0; ds->dt = 0.0; ds->lam = 0.0; ds->hl = 0.0; ds->c_lw = 0.0; ds->c_lf = 0.0;
    ds->smax_bits = 0ull; ds->status = 0; ds->pad = 0; ds->steps = 0;
}

int launch_begin_step(StepState* ds, StepConst* dsc, int nev, int mode, double value, double dx, double alpha, cudaStream_t st)
{
    k_begin_step<<<(nev + 63) / 64, nev < 64 ? nev : 64, 0, st>>>(ds, dsc, nev, mode, value, dx, alpha);
    return 1;
}
int upload_step_const_staged(const StepConst* dsc, int slot, int nev, cudaStream_t st) { return upload_step_const(dsc, slot, nev, st); }
int launch_end_step(StepState* ds, int nev, cudaStream_t st) { k_end_step<<<(nev + 63) / 64, nev < 64 ? nev : 64, 0, st>>>(ds, nev); return 1; }
int launch_reset(StepState* ds, int nev, cudaStream_t st) { k_reset<<<(nev + 63) / 64, nev < 64 ? nev : 64, 0, st>>>(ds, nev); return 1; }

// =========================================================================== a3 + a4: cell stage
// One thread per cell of the extended region (interior + 1 layer on every active axis).
template <int LIM, int EK, bool UC, class ST>
__global__ void __launch_bounds__(CT, MF_CELL_MINB) k_cell_stage(Grid g, Eos q, int predictor, CState5 V, Faces fc, State5 Wout, const StepState* ds)
{
    // linear index over the extended region, x fastest: 256 consecutive cells per block (measured on B200: 32 x 8 tiles, which
    // reuse the y neighbours through L1, are 10-15% slower because the DRAM bursts get shorter)
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.next) return;
    int ie, je, ke;
    unflatten3((unsigned int)p, g.dv[0][2 * g.h[0]], g.dv[1][2 * g.h[1]], ie, je, ke);
    const int c[3] = { ie - g.h[0], je - g.h[1], ke - g.h[2] };             // interior coordinates, may be -1 or n
    int cc[3];
#pragma unroll
    for (int a = 0; a < 3; ++a) cc[a] = g.act[a] ? bc_index(c[a], g.n[a], g.periodic) : 0;
    // every offset fits 32 bits (mf_create refuses grids of 2^32 cells or more - 400 B/cell of HBM is the tighter limit); unsigned
    // 32-bit offsets make each address one IMAD.WIDE.U32 instead of a 64-bit add pair
    const unsigned int ns[3] = { (unsigned int)g.ns[0], (unsigned int)g.ns[1], (unsigned int)g.ns[2] };
    const unsigned int o0 = blockIdx.y * (unsigned int)g.ncell + cc[0] * ns[0] + cc[1] * ns[1] + cc[2] * ns[2];
    const unsigned int pu = blockIdx.y * (unsigned int)g.next + (unsigned int)p;
    double U0[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) U0[v] = ld_state<ST>(V.q[v], o0);
#if MF_CELL_PF
    // The kernel is latency bound, and the only lines a block meets for the first time are those of the plane above (z+1): everything else
    // was touched by the blocks before it.  Pull that plane's lines for the cells one wave of blocks ahead towards L2.
    if (g.act[2]) {
        const unsigned int opf = o0 + ns[2] + (unsigned int)MF_CELL_PF;
        if (opf < (blockIdx.y + 1u) * (unsigned int)g.ncell) {
#pragma unroll
            for (int v = 0; v < 5; ++v) prefetch_l2(reinterpret_cast<const ST*>(V.q[v]) + opf);
        }
    }
#endif

#ifdef MF_STRICT
    double UL[3][5], UR[3][5];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if (!g.act[d]) continue;
        const unsigned int om = o0 + (unsigned int)(bc_index(c[d] - 1, g.n[d], g.periodic) - cc[d]) * ns[d];
        const unsigned int op = o0 + (unsigned int)(bc_index(c[d] + 1, g.n[d], g.periodic) - cc[d]) * ns[d];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            double a = U0[v] - ld_state<ST>(V.q[v], om);
            double b = ld_state<ST>(V.q[v], op) - U0[v];
            double s = slope2<LIM>(a, b);                                  // Eq.15-17
            UL[d][v] = U0[v] - 0.5 * s;                                    // Eq.12 :161
            UR[d][v] = U0[v] + 0.5 * s;
        }
    }
    if (predictor) {                                                        // Eq.13 (A3)
        const double hl = step_scalars<UC>(g, ds).hl;
        double delta[5];
        bool first = true;
        double Fl[5], Fr[5];
        if (g.act[0]) {
            flux_eval<0, EK>(q, UL[0], Fl); flux_eval<0, EK>(q, UR[0], Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) delta[v] = hl * (Fl[v] - Fr[v]);
            first = false;
        }
        if (g.act[1]) {
            flux_eval<1, EK>(q, UL[1], Fl); flux_eval<1, EK>(q, UR[1], Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) { double t = hl * (Fl[v] - Fr[v]); delta[v] = first ? t : delta[v] + t; }
            first = false;
        }
        if (g.act[2]) {
            flux_eval<2, EK>(q, UL[2], Fl); flux_eval<2, EK>(q, UR[2], Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) { double t = hl * (Fl[v] - Fr[v]); delta[v] = first ? t : delta[v] + t; }
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (!g.act[d]) continue;
#pragma unroll
            for (int v = 0; v < 5; ++v) { UL[d][v] += delta[v]; UR[d][v] += delta[v]; }
        }
    }
#pragma unroll
    for (int d = 0; d < 3; ++d) {
        if (!g.act[d]) continue;
#pragma unroll
        for (int v = 0; v < 5; ++v) { fc.f[d][0][v][pu] = UL[d][v]; fc.f[d][1][v][pu] = UR[d][v]; }
    }
#else
    // Product build, compact scratch (160 instead of 240 B/cell in 3D): the half slopes H_d = slope_d/2 per direction and
    // W = U + delta once; the flux kernel rebuilds U~dR = W + H_d, U~dL = W - H_d.
    double H[3][5];
    {
        // all neighbour loads are issued before the first use: the kernel is latency bound, memory-level parallelism is what counts
        double Um[3][5], Up[3][5];
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (!g.act[d]) continue;
            const unsigned int om = o0 + (unsigned int)(bc_index(c[d] - 1, g.n[d], g.periodic) - cc[d]) * ns[d];
            const unsigned int op = o0 + (unsigned int)(bc_index(c[d] + 1, g.n[d], g.periodic) - cc[d]) * ns[d];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                Um[d][v] = (double)__ldg(reinterpret_cast<const ST*>(V.q[v]) + om); Up[d][v] = (double)__ldg(reinterpret_cast<const ST*>(V.q[v]) + op);
            }
        }
#pragma unroll
        for (int d = 0; d < 3; ++d) {
            if (!g.act[d]) continue;
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                double a = U0[v] - Um[d][v];
                double b = Up[d][v] - U0[v];
                H[d][v] = half_slope2<LIM>(a, b);                           // Eq.15-17, Eq.12
                fc.f[d][0][v][pu] = H[d][v];
            }
        }
    }
    double W[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) W[v] = U0[v];
    if (predictor) {                                                        // Eq.13 (A3)
        const double hl = step_scalars<UC>(g, ds).hl;
        double acc[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
        double UL[5], UR[5], Fl[5], Fr[5];
        if (g.act[0]) {
#pragma unroll
            for (int v = 0; v < 5; ++v) { UL[v] = U0[v] - H[0][v]; UR[v] = U0[v] + H[0][v]; }
            flux_eval<0, EK>(q, UL, Fl); flux_eval<0, EK>(q, UR, Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) acc[v] += Fl[v] - Fr[v];
        }
        if (g.act[1]) {
#pragma unroll
            for (int v = 0; v < 5; ++v) { UL[v] = U0[v] - H[1][v]; UR[v] = U0[v] + H[1][v]; }
            flux_eval<1, EK>(q, UL, Fl); flux_eval<1, EK>(q, UR, Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) acc[v] += Fl[v] - Fr[v];
        }
        if (g.act[2]) {
#pragma unroll
            for (int v = 0; v < 5; ++v) { UL[v] = U0[v] - H[2][v]; UR[v] = U0[v] + H[2][v]; }
            flux_eval<2, EK>(q, UL, Fl); flux_eval<2, EK>(q, UR, Fr);
#pragma unroll
            for (int v = 0; v < 5; ++v) acc[v] += Fl[v] - Fr[v];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) W[v] = fma(hl, acc[v], U0[v]);
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) Wout.q[v][pu] = W[v];                        // = fc.f[first active axis][1]
#endif
}

int launch_cell_stage(const Grid& g, const Eos& q, int limiter, int predictor, CState5 V, Faces fc, const StepState* ds, cudaStream_t st)
{
    const dim3 nb(blocks_for(g.next, CT), g.nev);
    State5 Wout;
    for (int v = 0; v < 5; ++v) Wout.q[v] = fc.f[g.act[0] ? 0 : (g.act[1] ? 1 : 2)][1][v];
    switch (limiter) {
#define MF_CASE_ST(L, ST_) if (q.kind) k_cell_stage<L, 1, false, ST_><<<nb, CT, 0, st>>>(g, q, predictor, V, fc, Wout, ds); \
                           else if (g.cslot >= 0) k_cell_stage<L, 0, true, ST_><<<nb, CT, 0, st>>>(g, q, predictor, V, fc, Wout, ds); \
                           else k_cell_stage<L, 0, false, ST_><<<nb, CT, 0, st>>>(g, q, predictor, V, fc, Wout, ds);
#define MF_CASE(L) case L: if (g.state32) { MF_CASE_ST(L, float) } else { MF_CASE_ST(L, double) } break;
        MF_CASE(LIM_NONE) MF_CASE(LIM_MINMOD) MF_CASE(LIM_SUPERBEE) MF_CASE(LIM_VANALBADA) MF_CASE(LIM_VANLEER) MF_CASE(LIM_MC) MF_CASE(LIM_FIRST)
#undef MF_CASE
#undef MF_CASE_ST
    default: return 0;
    }
    return 1;
}

// =========================================================================== a5 + a6: interface fluxes
// One thread per interface between cell c and c+e_D; c runs over -1..n_D-1 along D and the interior on the other axes.
template <int D, int EK, bool UC>
__device__ __forceinline__ void flux_stage_body(const Grid& g, const Eos& q, int k, const CState5& Wc, const Faces& fc, const Fluxes& fx,
                                                const StepState* ds, unsigned int block)
{
    int m[3] = { g.n[0], g.n[1], g.n[2] };
    m[D] += 1;
    const long long total = (long long)m[0] * m[1] * m[2];
    const long long t = (long long)block * blockDim.x + threadIdx.x;
    if (t >= total) return;
    int c[3];
    unflatten3((unsigned int)t, g.dv[0][D == 0], g.dv[1][D == 1], c[0], c[1], c[2]);
    c[D] -= 1;
    const unsigned int es[3] = { (unsigned int)g.es[0], (unsigned int)g.es[1], (unsigned int)g.es[2] };
    const unsigned int p = blockIdx.y * (unsigned int)g.next + (c[0] + g.h[0]) * es[0] + (c[1] + g.h[1]) * es[1] + (c[2] + g.h[2]) * es[2];   // < 2^32 (mf_create)
    double A[5], B[5], F[5];
#ifdef MF_STRICT
#pragma unroll
    for (int v = 0; v < 5; ++v) { A[v] = fc.f[D][1][v][p]; B[v] = fc.f[D][0][v][p + es[D]]; }   // A2 :173
#else
    {                                                                                             // compact scratch: W and H_D
        const unsigned int pn = p + es[D];                          // (W's arrays come as an argument of their own: picking them out of fc
#pragma unroll                                                      //  with a runtime index costs indexed constant loads the loads then wait for)
        for (int v = 0; v < 5; ++v) { A[v] = Wc.q[v][p] + fc.f[D][0][v][p]; B[v] = Wc.q[v][pn] - fc.f[D][0][v][pn]; }
    }
#endif
    musta_flux<D, EK>(q, k, musta_coef(step_scalars<UC>(g, ds)), A, B, F);
#pragma unroll
    for (int v = 0; v < 5; ++v) fx.f[D][v][p] = F[v];
}

template <int D, int EK, bool UC>
__global__ void __launch_bounds__(FT, MF_FLUX_MINB) k_flux_stage(Grid g, Eos q, int k, CState5 Wc, Faces fc, Fluxes fx, const StepState* ds)
{
    flux_stage_body<D, EK, UC>(g, q, k, Wc, fc, fx, ds, blockIdx.x);
}

// The y and the z interfaces of a stage are independent of each other: ONE launch runs both (blocks [0, nby) take y, the rest z), so that the
// z blocks fill the SMs while the last y blocks drain - one kernel boundary less per RK stage.
template <int EK, bool UC>
__global__ void __launch_bounds__(FT, MF_FLUX_MINB) k_flux_stage_yz(Grid g, Eos q, int k, CState5 Wc, Faces fc, Fluxes fx, const StepState* ds, unsigned int nby)
{
#if MF_YZ_INTERLEAVE
    // even blocks take y, odd blocks z, of the same stretch of cells: the W lines a y block reads are read again by the z block next to it
    // while they are still in L2 (W(k) is the y block's plane and the z block's upper plane), so W crosses HBM once for the two directions
    const unsigned int b = blockIdx.x >> 1;
    if ((blockIdx.x & 1u) == 0) { if (b < nby) flux_stage_body<1, EK, UC>(g, q, k, Wc, fc, fx, ds, b); }
    else flux_stage_body<2, EK, UC>(g, q, k, Wc, fc, fx, ds, b);
#else
    if (blockIdx.x < nby) flux_stage_body<1, EK, UC>(g, q, k, Wc, fc, fx, ds, blockIdx.x);
    else flux_stage_body<2, EK, UC>(g, q, k, Wc, fc, fx, ds, blockIdx.x - nby);
#endif
}

int launch_flux_stage(const Grid& g, const Eos& q, int k, int dmask, Faces fc, Fluxes fx, const StepState* ds, cudaStream_t st)
{
    int launches = 0;
    CState5 Wc;
    for (int v = 0; v < 5; ++v) Wc.q[v] = fc.f[g.act[0] ? 0 : (g.act[1] ? 1 : 2)][1][v];
#ifndef MF_NO_YZ_MERGE
    if (dmask == 6 && g.act[1] && g.act[2]) {
        const unsigned int nby = blocks_for((long long)g.n[0] * (g.n[1] + 1) * g.n[2], FT), nbz = blocks_for((long long)g.n[0] * g.n[1] * (g.n[2] + 1), FT);
#if MF_YZ_INTERLEAVE
        const dim3 nb(2 * (nby > nbz ? nby : nbz), g.nev);
#else
        const dim3 nb(nby + nbz, g.nev);
#endif
        if (q.kind) k_flux_stage_yz<1, false><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds, nby);
        else if (g.cslot >= 0) k_flux_stage_yz<0, true><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds, nby);
        else k_flux_stage_yz<0, false><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds, nby);
        return 1;
    }
#endif
    for (int d = 0; d < 3; ++d) {
        if (!g.act[d] || !(dmask & (1 << d))) continue;
        long long total = 1;
        for (int a = 0; a < 3; ++a) total *= (a == d) ? g.n[a] + 1 : g.n[a];
        const dim3 nb(blocks_for(total, FT), g.nev);
#define MF_FLUX(D_) do { if (q.kind) k_flux_stage<D_, 1, false><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds); \
                         else if (g.cslot >= 0) k_flux_stage<D_, 0, true><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds); \
                         else k_flux_stage<D_, 0, false><<<nb, FT, 0, st>>>(g, q, k, Wc, fc, fx, ds); } while (0)
        if (d == 0) MF_FLUX(0);
        if (d == 1) MF_FLUX(1);
        if (d == 2) MF_FLUX(2);
#undef MF_FLUX
        ++launches;
    }
    return launches;
}

// =========================================================================== a7 + a8: divergence, source, RK combine
template <int EK, class ST>
__global__ void __launch_bounds__(TPB) k_combine(Grid g, Eos q, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out, Source src, StepState* ds)
{
    const long long ol = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    double smax = 0.0;
    int bad = 0;
    ds += blockIdx.y;
    if (ol < g.ncell) {
        int i, j, k;
        unflatten3((unsigned int)ol, g.dv[0][0], g.dv[1][0], i, j, k);
        const unsigned int o = blockIdx.y * (unsigned int)g.ncell + (unsigned int)ol;
        const unsigned int p = blockIdx.y * (unsigned int)g.next + (i + g.h[0]) * (unsigned int)g.es[0] + (j + g.h[1]) * (unsigned int)g.es[1]
                               + (k + g.h[2]) * (unsigned int)g.es[2];
        const double dt = ds->dt;
        double S = 0.0;
        if (src.on) S = jet_source(g, src, i, j, k, ds->t + sg.ts * dt);
        double fhi[3][5], flo[3][5], ua5[5], ub5[5];                   // all loads before the first store (see k_xflux_combine)
#pragma unroll
        for (int v = 0; v < 5; ++v) {
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (!g.act[d]) continue;
                fhi[d][v] = fx.f[d][v][p]; flo[d][v] = fx.f[d][v][p - (unsigned int)g.es[d]];
            }
            ua5[v] = sg.form == 3 ? 0.0 : ld_state<ST>(Ua.q[v], o);
            ub5[v] = (sg.form == 1 || sg.form == 2) ? ld_state<ST>(Ub.q[v], o) : 0.0;
        }
        double W[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            double acc = 0.0;
            bool first = true;
#pragma unroll
            for (int d = 0; d < 3; ++d) {
                if (!g.act[d]) continue;
                double diff = fhi[d][v] - flo[d][v];
                acc = first ? diff : acc + diff;
                first = false;
            }
#ifdef MF_STRICT
            double L = -acc / g.dx;                                    // Eq.1 :43
#else
            double L = -acc * g.inv_dx;
#endif
            if (src.on && v < 2) L = L + S;
            W[v] = rk_form(sg, ua5[v], ub5[v], dt, L);
            if (sg.form == 3) out.q[v][o] = W[v];                      // L itself (mf_eval_L): double whatever the state precision
            else { st_state<ST>(out.q[v], o, W[v]); W[v] = as_stored<ST>(W[v]); }
        }
        if (sg.cfl) smax = signal_speed<EK>(q, W[0], W[1], W[2], W[3], W[4], bad);   // a2 for the next step, while U^{n+1} is in registers
    }
    if (sg.cfl) block_reduce_smax(smax, bad, ds);
}

int launch_combine(const Grid& g, const Eos& q, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out, Source src, StepState* ds, cudaStream_t st)
{
    const dim3 nb(blocks_for(g.ncell, TPB), g.nev);
    if (g.state32) {
        if (q.kind) k_combine<1, float><<<nb, TPB, 0, st>>>(g, q, fx, sg, Ua, Ub, out, src, ds);
        else k_combine<0, float><<<nb, TPB, 0, st>>>(g, q, fx, sg, Ua, Ub, out, src, ds);
    } else {
        if (q.kind) k_combine<1, double><<<nb, TPB, 0, st>>>(g, q, fx, sg, Ua, Ub, out, src, ds);
        else k_combine<0, double><<<nb, TPB, 0, st>>>(g, q, fx, sg, Ua, Ub, out, src, ds);
    }
    return 1;
}

// =========================================================================== a5 (x) + a7 + a8 (+ a2) in one kernel
// The x fluxes are the last ones of a stage.  Thread t of a block of XT threads owns x interface I = (XT-1)*block + t (linear over all rows,
// nx+1 per row), runs MUSTA on it and leaves the flux in shared memory; the cell to the right of the interface then has both of its x
// fluxes on chip (its own and thread t+1's), reads F_y, F_z of its four other faces, and is finished: divergence, source, RK combine, one
// store.  Blocks overlap by one interface, so XT-1 of XT threads finish a cell.  F_x is never written, and the 30 loads of the combine hide
// under the FP64 work of a compute-bound kernel instead of making a memory-bound pass of their own.
// Measured on B200 (256^3): 128-thread blocks, 5 per SM at 96 registers (the combine's 30 operands are all in flight at once, issued before
// the barrier; an extra L2 prefetch of them before MUSTA stopped paying once they were); staging them with cp.async in shared memory
// instead was 40% slower (the 35 KB per block cost the L1 hits of the x-neighbour loads).  History of this kernel: 1.56 -> 1.37 -> 1.03 -> 0.95 ms per launch.
// FORM (the RK form of the stage) and CFL (last stage of a step) are compile-time: the stage loop has no form branches, and the
// signal-speed code with its block reduction exists only in the instantiations that need it.
template <int EK, int FORM, bool CFL, bool UC, class ST>
__global__ void __launch_bounds__(XT, MF_XC_MINB) k_xflux_combine(Grid g, Eos q, int k, Faces fc, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out,
                                                          Source src, StepState* ds)
{
    __shared__ double sF[5][XT];
    const int t = threadIdx.x;
    const int nf = g.n[0] + 1;                                              // x interfaces per row
    const long long nrows = (long long)g.n[1] * g.n[2];
    const long long I = (long long)blockIdx.x * (XT - 1) + t;
    const bool live = I < nrows * nf;
    int f = 0, j = 0, kz = 0;
    unsigned int p = 0;                                                      // cell offsets fit 32 bits (mf_create)
    double F[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    const unsigned int eo = blockIdx.y * (unsigned int)g.ncell, ep = blockIdx.y * (unsigned int)g.next;   // this block's event
    const StepConst sc = step_scalars<UC>(g, ds);
    ds += blockIdx.y;
    if (live) {
        unflatten3((unsigned int)I, g.dv[0][1], g.dv[1][0], f, j, kz);                       // f: interface between cells f-1 and f of row (j, kz)
        p = ep + f + (unsigned int)(j + g.h[1]) * (unsigned int)g.es[1] + (unsigned int)(kz + g.h[2]) * (unsigned int)g.es[2];   // extended index of cell f-1
        double A[5], B[5];
#ifdef MF_STRICT
#pragma unroll
        for (int v = 0; v < 5; ++v) { A[v] = fc.f[0][1][v][p]; B[v] = fc.f[0][0][v][p + 1]; }
#else
#pragma unroll
        for (int v = 0; v < 5; ++v) { A[v] = fc.f[0][1][v][p] + fc.f[0][0][v][p]; B[v] = fc.f[0][1][v][p + 1] - fc.f[0][0][v][p + 1]; }
#endif
        musta_flux<0, EK>(q, k, musta_coef(sc), A, B, F);
    }
    // The combine's operands.  Every one is loaded before the first store: `out` may alias the inputs as far as the compiler knows (and does
    // alias U_(s) in low-storage mode), so loads written after a store would wait for it - five dependent round trips to memory instead of
    // one.  And they are issued BEFORE the barrier, so that their latency runs while the block's other warps finish MUSTA.
    const bool owns_cell = live && t < XT - 1 && f < g.n[0];                // cell (f, j, kz): lower x face = this interface, upper = thread t+1's
    const unsigned int pc = p + 1;
    const unsigned int o = eo + f + (unsigned int)j * (unsigned int)g.ns[1] + (unsigned int)kz * (unsigned int)g.ns[2];
    double fy1[5], fy0[5], fz1[5], fz0[5], ua5[5], ub5[5];
    if (owns_cell) {
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            if (g.act[1]) { fy1[v] = fx.f[1][v][pc]; fy0[v] = fx.f[1][v][pc - (unsigned int)g.es[1]]; }
            if (g.act[2]) { fz1[v] = fx.f[2][v][pc]; fz0[v] = fx.f[2][v][pc - (unsigned int)g.es[2]]; }
            ua5[v] = FORM == 3 ? 0.0 : ld_state<ST>(Ua.q[v], o);
            ub5[v] = (FORM == 1 || FORM == 2) ? ld_state<ST>(Ub.q[v], o) : 0.0;
        }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) sF[v][t] = F[v];
    __syncthreads();
    double smax = 0.0;
    int bad = 0;
    if (owns_cell) {
        const double dt = sc.dt;
        double S = 0.0;
        if (src.on) S = jet_source(g, src, f, j, kz, ds->t + sg.ts * dt);
        double W[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            double acc = sF[v][t + 1] - F[v];
            if (g.act[1]) acc = acc + (fy1[v] - fy0[v]);
            if (g.act[2]) acc = acc + (fz1[v] - fz0[v]);
#ifdef MF_STRICT
            double L = -acc / g.dx;                                        // Eq.1 :43
#else
            double L = -acc * g.inv_dx;
#endif
            if (src.on && v < 2) L = L + S;
            const double ua = ua5[v], ub = ub5[v];
            W[v] = FORM == 0 ? ua + dt * L : (FORM == 1 ? 0.5 * (ua + ub + dt * L) : (FORM == 2 ? sg.ca * ua + sg.cb * ub + (sg.cdt * dt) * L : L));
            if (FORM == 3) out.q[v][o] = W[v];                             // L itself (mf_eval_L): double whatever the state precision
            else st_state<ST>(out.q[v], o, W[v]);
        }
        if (CFL) {                                                         // S_max of the STORED (rounded, reading A19) new state
#pragma unroll
            for (int v = 0; v < 5; ++v) W[v] = as_stored<ST>(W[v]);
            smax = signal_speed<EK>(q, W[0], W[1], W[2], W[3], W[4], bad);
        }
    }
    if (CFL) block_reduce_smax<XT>(smax, bad, ds);
}

int launch_xflux_combine(const Grid& g, const Eos& q, int k, Faces fc, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out, Source src,
                         StepState* ds, cudaStream_t st)
{
    const long long total = (long long)(g.n[0] + 1) * g.n[1] * g.n[2];
    const dim3 nb(blocks_for(total, XT - 1), g.nev);
#define MF_XFC_ST(EK_, FORM_, CFL_, ST_) do { if (EK_ == 0 && g.cslot >= 0) k_xflux_combine<EK_, FORM_, CFL_, EK_ == 0, ST_><<<nb, XT, 0, st>>>(g, q, k, fc, fx, sg, Ua, Ub, out, src, ds); \
                                      else k_xflux_combine<EK_, FORM_, CFL_, false, ST_><<<nb, XT, 0, st>>>(g, q, k, fc, fx, sg, Ua, Ub, out, src, ds); } while (0)
#define MF_XFC(EK_, FORM_, CFL_) do { if (g.state32) MF_XFC_ST(EK_, FORM_, CFL_, float); else MF_XFC_ST(EK_, FORM_, CFL_, double); } while (0)
#define MF_XFC_FORMS(EK_) \
    if (sg.form == 0) { if (sg.cfl) MF_XFC(EK_, 0, true); else MF_XFC(EK_, 0, false); } \
    else if (sg.form == 1) { if (sg.cfl) MF_XFC(EK_, 1, true); else MF_XFC(EK_, 1, false); } \
    else if (sg.form == 2) { if (sg.cfl) MF_XFC(EK_, 2, true); else MF_XFC(EK_, 2, false); } \
    else MF_XFC(EK_, 3, false);
    if (q.kind) { MF_XFC_FORMS(1) } else { MF_XFC_FORMS(0) }
#undef MF_XFC_FORMS
#undef MF_XFC
#undef MF_XFC_ST
    return 1;
}

// =========================================================================== conversions
template <int EK>
__global__ void __launch_bounds__(TPB) k_prim2con(Grid g, Eos q, State5 U)
{
    const long long ol = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ol >= g.ncell) return;
    const unsigned int o = blockIdx.y * (unsigned int)g.ncell + (unsigned int)ol;
    double e = U.q[0][o], vx = U.q[1][o], vy = U.q[2][o], vz = U.q[3][o], n = U.q[4][o];
    double p = eos_eval<EK>(q, e, n).p;                                // Eq.4 :63-67
    double g2 = 1.0 / (1.0 - (vx * vx + vy * vy + vz * vz));
    double w = (e + p) * g2;
    U.q[0][o] = w - p; U.q[1][o] = w * vx; U.q[2][o] = w * vy; U.q[3][o] = w * vz; U.q[4][o] = n * sqrt(g2);
}

template <int EK, class ST>
__global__ void __launch_bounds__(TPB) k_con2prim(Grid g, Eos q, CState5 U, State5 P)
{
    const long long ol = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (ol >= g.ncell) return;
    const unsigned int o = blockIdx.y * (unsigned int)g.ncell + (unsigned int)ol;
    double vx, vy, vz, e, p;
    const double R = ld_state<ST>(U.q[4], o);
    velocity_pressure<EK>(q, ld_state<ST>(U.q[0], o), ld_state<ST>(U.q[1], o), ld_state<ST>(U.q[2], o), ld_state<ST>(U.q[3], o), R, vx, vy, vz, e, p);
    P.q[0][o] = e; P.q[1][o] = vx; P.q[2][o] = vy; P.q[3][o] = vz;
    P.q[4][o] = R * sqrt(1.0 - (vx * vx + vy * vy + vz * vz));           // n = R sqrt(1-v^2), Eq.23
}

int launch_prim2con(const Grid& g, const Eos& q, State5 U, cudaStream_t st)
{
    const dim3 nb(blocks_for(g.ncell, TPB), g.nev);
    if (q.kind) k_prim2con<1><<<nb, TPB, 0, st>>>(g, q, U); else k_prim2con<0><<<nb, TPB, 0, st>>>(g, q, U);
    return 1;
}
int launch_con2prim(const Grid& g, const Eos& q, CState5 U, State5 P, cudaStream_t st)
{
    const dim3 nb(blocks_for(g.ncell, TPB), g.nev);
    if (g.state32) { if (q.kind) k_con2prim<1, float><<<nb, TPB, 0, st>>>(g, q, U, P); else k_con2prim<0, float><<<nb, TPB, 0, st>>>(g, q, U, P); }
    else { if (q.kind) k_con2prim<1, double><<<nb, TPB, 0, st>>>(g, q, U, P); else k_con2prim<0, double><<<nb, TPB, 0, st>>>(g, q, U, P); }
    return 1;
}

// =========================================================================== totals: per-block partial sums (host adds them in long double)
template <class ST>
__global__ void __launch_bounds__(TPB) k_totals(Grid g, CState5 U, double* partials)
{
    double acc[5] = { 0, 0, 0, 0, 0 };
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < g.ncell; o += stride)
#pragma unroll
        for (int v = 0; v < 5; ++v) acc[v] += (double)reinterpret_cast<const ST*>(U.q[v])[o];
    __shared__ double s[5][TPB / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int v = 0; v < 5; ++v) {
#pragma unroll
        for (int off = 16; off > 0; off >>= 1) acc[v] += __shfl_xor_sync(0xffffffffu, acc[v], off);
        if (lane == 0) s[v][warp] = acc[v];
    }
    __syncthreads();
    if (threadIdx.x < 5) {
        double t = 0.0;
        for (int w = 0; w < TPB / 32; ++w) t += s[threadIdx.x][w];
        partials[(long long)threadIdx.x * gridDim.x + blockIdx.x] = t;
    }
}

int launch_totals(const Grid& g, CState5 U, double* partials, int nblocks, cudaStream_t st)
{
    if (g.state32) k_totals<float><<<nblocks, TPB, 0, st>>>(g, U, partials); else k_totals<double><<<nblocks, TPB, 0, st>>>(g, U, partials);
    return 1;
}

// =========================================================================== state precision (reading A19): double <-> float copies of a state
// n elements per component; `src`/`dst` component pointers are already spaced for their own element type
__global__ void __launch_bounds__(TPB) k_state_to_f32(long long n, CState5 src, State5 dst)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += stride)
#pragma unroll
        for (int v = 0; v < 5; ++v) reinterpret_cast<float*>(dst.q[v])[o] = (float)src.q[v][o];       // round to nearest even
}
__global__ void __launch_bounds__(TPB) k_state_to_f64(long long n, CState5 src, State5 dst)
{
    const long long stride = (long long)gridDim.x * blockDim.x;
    for (long long o = (long long)blockIdx.x * blockDim.x + threadIdx.x; o < n; o += stride)
#pragma unroll
        for (int v = 0; v < 5; ++v) dst.q[v][o] = (double)reinterpret_cast<const float*>(src.q[v])[o];
}
int launch_state_convert(long long n, int to_f32, CState5 src, State5 dst, int num_sms, cudaStream_t st)
{
    long long nb = (n + TPB - 1) / TPB;
    if (nb > 32LL * num_sms) nb = 32LL * num_sms;
    if (to_f32) k_state_to_f32<<<(unsigned int)nb, TPB, 0, st>>>(n, src, dst); else k_state_to_f64<<<(unsigned int)nb, TPB, 0, st>>>(n, src, dst);
    return 1;
}

} // namespace mf
