// mf_fused.cu — fused path (MF_PATH_FUSED) for fully 3D grids: per RK stage one small predictor kernel and ONE sweep kernel.
//
// k_delta_stage (a3+a4): one thread per cell of the grid plus a one-cell ghost ring; limited slopes in x, y, z, the six
//   face fluxes of Eq.13 and the Hancock increment delta (5 doubles per cell) — the only intermediate that goes to HBM.
// k_sweep_stage (a1, a3, a5, a6, a7, a8): a CTA of 32 x TYB threads owns (32-2) x (TYB-2) cells in (x, y) plus a one-cell
//   ring and marches through a chunk of z planes (2.5D streaming).  Per plane kk every thread rebuilds the six evolved face
//   states of its cell, U -/+ slope/2 + delta, in registers (ring cells too: this costs a handful of instructions, which
//   is why delta is computed once per cell by the kernel above instead of once per tile), then
//     z: MUSTA flux at kk-1/2 from the thread's own saved U~zR(kk-1) and fresh U~zL(kk); plane kk-1 is finalised:
//        L = -((Fx+ - Fx-) + (Fy+ - Fy-) + (Fz+ - Fz-))/dx, source, RK combine, ONE store of the new stage state;
//     x: MUSTA flux at i+1/2, right state from lane+1 by warp shuffle, F(i-1/2) from lane-1 by shuffle;
//     y: MUSTA flux at j+1/2, right state and F(j-1/2) from the neighbouring warp through shared memory.
//   Face states, fluxes and flux differences never touch HBM.
// The arithmetic per cell and per interface is the same sequence as in the staged path, so the strict build stays
// bit-identical to the oracle.
#include "mf_kernels.h"

namespace mf {

namespace {

constexpr int TXB = 32;          // threads along x = one warp
constexpr int IX = TXB - 2;      // interior cells per tile row
constexpr int TPB_D = 256;

__device__ __forceinline__ double shfl_down1(double v) { return __shfl_down_sync(0xffffffffu, v, 1); }
__device__ __forceinline__ double shfl_up1(double v) { return __shfl_up_sync(0xffffffffu, v, 1); }

__device__ __forceinline__ double jet_source_f(const Grid& g, const Source& s, int i, int j, int k, double t)
{
    double x = (i + 0.5 - g.n[0] / 2.0) * g.dx - (s.x0 + t);
    double y = (j + 0.5 - g.n[1] / 2.0) * g.dx - s.y0;
    double z = (k + 0.5 - g.n[2] / 2.0) * g.dx - s.z0;
    double r2 = x * x + y * y + z * z;
    double arg = -r2 * s.inv_two_s2;
#ifndef MF_STRICT
    if (arg < -745.0) return 0.0;
#endif
    return s.dEdx * s.norm * exp(arg);
}

__device__ __forceinline__ double rk_form_f(const Stage& sg, double ua, double ub, double dt, double L)
{
    if (sg.form == 0) return ua + dt * L;
    if (sg.form == 1) return 0.5 * (ua + ub + dt * L);
    if (sg.form == 2) return sg.ca * ua + sg.cb * ub + (sg.cdt * dt) * L;
    return L;
}

// ------------------------------------------------------------------------------------------------ a3 + a4 -> delta
template <int LIM>
__global__ void __launch_bounds__(TPB_D) k_delta_stage(Grid g, Eos q, CState5 V, State5 D, const StepState* __restrict__ ds)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.next) return;
    const int ie = (int)(p % g.e[0]);
    const long long r = p / g.e[0];
    const int je = (int)(r % g.e[1]), ke = (int)(r / g.e[1]);
    const int cx = ie - 1, cy = je - 1, cz = ke - 1;
    const int per = g.periodic;
    const long long ox0 = bc_index(cx, g.n[0], per), oxm = bc_index(cx - 1, g.n[0], per), oxp = bc_index(cx + 1, g.n[0], per);
    const long long oy0 = bc_index(cy, g.n[1], per) * g.ns[1], oym = bc_index(cy - 1, g.n[1], per) * g.ns[1], oyp = bc_index(cy + 1, g.n[1], per) * g.ns[1];
    const long long oz0 = bc_index(cz, g.n[2], per) * g.ns[2], ozm = bc_index(cz - 1, g.n[2], per) * g.ns[2], ozp = bc_index(cz + 1, g.n[2], per) * g.ns[2];
    const long long o0 = ox0 + oy0 + oz0;
    double xL[5], xR[5], yL[5], yR[5], zL[5], zR[5];
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double* Vv = V.q[v];
        double u0 = Vv[o0];
        double a = u0 - Vv[oxm + oy0 + oz0], b = Vv[oxp + oy0 + oz0] - u0;
        double s = slope2<LIM>(a, b);
        xL[v] = u0 - 0.5 * s; xR[v] = u0 + 0.5 * s;
        a = u0 - Vv[ox0 + oym + oz0]; b = Vv[ox0 + oyp + oz0] - u0;
        s = slope2<LIM>(a, b);
        yL[v] = u0 - 0.5 * s; yR[v] = u0 + 0.5 * s;
        a = u0 - Vv[ox0 + oy0 + ozm]; b = Vv[ox0 + oy0 + ozp] - u0;
        s = slope2<LIM>(a, b);
        zL[v] = u0 - 0.5 * s; zR[v] = u0 + 0.5 * s;
    }
    const double hl = ds->hl;
    double Fl[5], Fr[5], delta[5];
    flux_eval<0>(q, xL, Fl); flux_eval<0>(q, xR, Fr);
#pragma unroll
    for (int v = 0; v < 5; ++v) delta[v] = hl * (Fl[v] - Fr[v]);
    flux_eval<1>(q, yL, Fl); flux_eval<1>(q, yR, Fr);
#pragma unroll
    for (int v = 0; v < 5; ++v) delta[v] = delta[v] + hl * (Fl[v] - Fr[v]);
    flux_eval<2>(q, zL, Fl); flux_eval<2>(q, zR, Fr);
#pragma unroll
    for (int v = 0; v < 5; ++v) D.q[v][p] = delta[v] + hl * (Fl[v] - Fr[v]);
}

// ------------------------------------------------------------------------------------------------ sweep
template <int LIM, int TYB, int MINB>
__global__ void __launch_bounds__(TXB * TYB, MINB)
k_sweep_stage(Grid g, Eos q, int predictor, int k, int TZ, int ntx, int nty, CState5 V, CState5 D, Stage sg, CState5 Ua, State5 out,
              Source src, const StepState* __restrict__ ds)
{
    constexpr int NT = TXB * TYB;
    extern __shared__ double sm[];
    double* s_zR = sm;                 // U~zR of the previous plane            [5][NT]
    double* s_Fz = sm + 5 * NT;        // F_z at the lower face of plane kk-1   [5][NT]
    double* s_xy = sm + 10 * NT;       // (Fx+ - Fx-) + (Fy+ - Fy-) of plane kk-1
    double* s_yL = sm + 15 * NT;       // U~yL of this plane, read by the warp below
    double* s_Fy = sm + 20 * NT;       // F_y(j+1/2) of this plane, read by the warp above

    const int lx = threadIdx.x, ly = threadIdx.y, tid = ly * TXB + lx;
    const int item = blockIdx.x;
    const int tx = item % ntx, ty = (item / ntx) % nty, tz = item / (ntx * nty);
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int z0 = tz * TZ, z1 = min(z0 + TZ, nz);
    const int cx = tx * IX - 1 + lx, cy = ty * (TYB - 2) - 1 + ly;          // this thread's cell; -1 and n are ghosts

    const bool xin = lx >= 1 && lx <= TXB - 2, yin = ly >= 1 && ly <= TYB - 2;
    const bool cell_ok = cx <= nx && cy <= ny && (xin || yin);              // corners of the ring are never needed
    const bool interior = xin && yin && cx < nx && cy < ny;
    const bool xint_ok = yin && lx <= TXB - 2 && cx <= nx - 1 && cy <= ny - 1;   // interface (cx+1/2, cy)
    const bool yint_ok = xin && ly <= TYB - 2 && cy <= ny - 1 && cx <= nx - 1;   // interface (cx, cy+1/2)

    // a1: boundary handling as index mapping (outflow = clamp, periodic = wrap), per axis
    long long ox0 = 0, oxm = 0, oxp = 0, oy0 = 0, oym = 0, oyp = 0, pe = 0;
    if (cell_ok) {
        ox0 = bc_index(cx, nx, g.periodic); oxm = bc_index(cx - 1, nx, g.periodic); oxp = bc_index(cx + 1, nx, g.periodic);
        oy0 = (long long)bc_index(cy, ny, g.periodic) * g.ns[1];
        oym = (long long)bc_index(cy - 1, ny, g.periodic) * g.ns[1];
        oyp = (long long)bc_index(cy + 1, ny, g.periodic) * g.ns[1];
        pe = (cx + 1) + (long long)(cy + 1) * g.es[1];                       // position in the extended layout (delta)
    }
    const double dt = ds->dt, lam = ds->lam, c_lw = ds->c_lw, c_lf = ds->c_lf;

    for (int kk = z0 - 1; kk <= z1; ++kk) {
        // ------------------------------------------------------------------ evolved face states of (cx, cy, kk)
        double xL[5], xR[5], yL[5], yR[5], zL[5], zR[5];
        if (cell_ok) {
            const long long oz0 = (long long)bc_index(kk, nz, g.periodic) * g.ns[2];
            const long long ozm = (long long)bc_index(kk - 1, nz, g.periodic) * g.ns[2];
            const long long ozp = (long long)bc_index(kk + 1, nz, g.periodic) * g.ns[2];
            const long long o0 = ox0 + oy0 + oz0;
            const long long pd = pe + (long long)(kk + 1) * g.es[2];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
                const double* Vv = V.q[v];
                const double u0 = Vv[o0];
                const double dl = predictor ? D.q[v][pd] : 0.0;
                double a = u0 - Vv[oxm + oy0 + oz0], b = Vv[oxp + oy0 + oz0] - u0;
                double s = slope2<LIM>(a, b);                                  // Eq.15-17
                xL[v] = u0 - 0.5 * s; xR[v] = u0 + 0.5 * s;                    // Eq.12
                a = u0 - Vv[ox0 + oym + oz0]; b = Vv[ox0 + oyp + oz0] - u0;
                s = slope2<LIM>(a, b);
                yL[v] = u0 - 0.5 * s; yR[v] = u0 + 0.5 * s;
                a = u0 - Vv[ox0 + oy0 + ozm]; b = Vv[ox0 + oy0 + ozp] - u0;
                s = slope2<LIM>(a, b);
                zL[v] = u0 - 0.5 * s; zR[v] = u0 + 0.5 * s;
                if (predictor) { xL[v] += dl; xR[v] += dl; yL[v] += dl; yR[v] += dl; zL[v] += dl; zR[v] += dl; }   // Eq.13
            }
        } else {
#pragma unroll
            for (int v = 0; v < 5; ++v) { double u = (v == 0 || v == 4) ? 1.0 : 0.0; xL[v] = xR[v] = yL[v] = yR[v] = zL[v] = zR[v] = u; }
        }
        // the warp below needs this plane's U~yL
#pragma unroll
        for (int v = 0; v < 5; ++v) s_yL[v * NT + tid] = yL[v];

        // ------------------------------------------------------------------ z interface kk-1/2 and finalisation of plane kk-1
        if (interior && kk >= z0) {
            double A[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) A[v] = s_zR[v * NT + tid];
            musta_flux<2>(q, k, lam, c_lw, c_lf, A, zL, F);
            if (kk > z0) {
                const int kc = kk - 1;
                const long long o = (long long)cx + (long long)cy * g.ns[1] + (long long)kc * g.ns[2];
                double S = 0.0;
                if (src.on) S = jet_source_f(g, src, cx, cy, kc, ds->t + sg.ts * dt);
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    double acc = s_xy[v * NT + tid] + (F[v] - s_Fz[v * NT + tid]);
                    double L = -acc / g.dx;
                    if (src.on && v < 2) L = L + S;
                    double ua = sg.form == 3 ? 0.0 : Ua.q[v][o];
                    double ub = (sg.form == 1 || sg.form == 2) ? V.q[v][o] : 0.0;
                    out.q[v][o] = rk_form_f(sg, ua, ub, dt, L);
                }
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) s_Fz[v * NT + tid] = F[v];
        }
#pragma unroll
        for (int v = 0; v < 5; ++v) s_zR[v * NT + tid] = zR[v];

        const bool plane_ok = kk >= z0 && kk < z1;               // x and y interfaces are needed on planes of the chunk only
        // ------------------------------------------------------------------ x interface (cx+1/2): neighbours by warp shuffle
        double xd[5];
        {
            double B[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { B[v] = shfl_down1(xL[v]); F[v] = 0.0; }
            if (plane_ok && xint_ok) musta_flux<0>(q, k, lam, c_lw, c_lf, xR, B, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) xd[v] = F[v] - shfl_up1(F[v]);
        }
        // ------------------------------------------------------------------ y interface (cy+1/2): neighbours through shared memory
        __syncthreads();                                          // s_yL of this plane is complete; s_Fy of the previous plane is consumed
        {
            double B[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) F[v] = 0.0;
            if (plane_ok && yint_ok) {
#pragma unroll
                for (int v = 0; v < 5; ++v) B[v] = s_yL[v * NT + tid + TXB];
                musta_flux<1>(q, k, lam, c_lw, c_lf, yR, B, F);
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) s_Fy[v * NT + tid] = F[v];
            __syncthreads();                                      // s_Fy complete; everybody is done reading s_yL
            if (plane_ok && interior) {
#pragma unroll
                for (int v = 0; v < 5; ++v) s_xy[v * NT + tid] = xd[v] + (F[v] - s_Fy[v * NT + tid - TXB]);
            }
        }
    }
}

template <int TYB, int MINB>
int launch_sweep(const Grid& g, const Eos& q, int limiter, int predictor, int k, CState5 V, CState5 D, Stage sg, CState5 Ua, State5 out,
                 Source src, const StepState* ds, int num_sms, cudaStream_t st)
{
    const int ntx = (g.n[0] + IX - 1) / IX, nty = (g.n[1] + (TYB - 2) - 1) / (TYB - 2);
    // z chunk: all of z, or the largest of {64, 32, 16, 8} planes for which the items fill the resident CTA slots ~8 times over
    int TZ = g.n[2];
    const int cands[4] = { 64, 32, 16, 8 };
    for (int c = 0; c < 4; ++c) {
        long long items = (long long)ntx * nty * ((g.n[2] + TZ - 1) / TZ);
        if (items >= 8LL * num_sms * MINB) break;
        if (cands[c] < TZ) TZ = cands[c];
    }
    const int ntz = (g.n[2] + TZ - 1) / TZ;
    const unsigned int grid = (unsigned int)(ntx * nty * ntz);
    const size_t smem = sizeof(double) * 25 * TXB * TYB;
    dim3 block(TXB, TYB);
#define MF_CASE(L) case L: { \
        static bool attr_set = false; \
        if (!attr_set) { cudaFuncSetAttribute(k_sweep_stage<L, TYB, MINB>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); attr_set = true; } \
        k_sweep_stage<L, TYB, MINB><<<grid, block, smem, st>>>(g, q, predictor, k, TZ, ntx, nty, V, D, sg, Ua, out, src, ds); } break;
    switch (limiter) {
        MF_CASE(LIM_NONE) MF_CASE(LIM_MINMOD) MF_CASE(LIM_SUPERBEE) MF_CASE(LIM_VANALBADA) MF_CASE(LIM_VANLEER) MF_CASE(LIM_MC) MF_CASE(LIM_FIRST)
    default: return 0;
    }
#undef MF_CASE
    return 1;
}

} // namespace

bool fused_supported(const Grid& g) { return g.act[0] && g.act[1] && g.act[2]; }

int launch_delta_stage(const Grid& g, const Eos& q, int limiter, CState5 V, State5 D, const StepState* ds, cudaStream_t st)
{
    const unsigned int nb = (unsigned int)((g.next + TPB_D - 1) / TPB_D);
    switch (limiter) {
#define MF_CASE(L) case L: k_delta_stage<L><<<nb, TPB_D, 0, st>>>(g, q, V, D, ds); break;
        MF_CASE(LIM_NONE) MF_CASE(LIM_MINMOD) MF_CASE(LIM_SUPERBEE) MF_CASE(LIM_VANALBADA) MF_CASE(LIM_VANLEER) MF_CASE(LIM_MC) MF_CASE(LIM_FIRST)
#undef MF_CASE
    default: return 0;
    }
    return 1;
}

int launch_fused_stage(const Grid& g, const Eos& q, int limiter, int predictor, int k, CState5 V, CState5 D, Stage sg, CState5 Ua,
                       State5 out, Source src, const StepState* ds, int num_sms, int variant, cudaStream_t st)
{
    if (variant == 1) return launch_sweep<8, 3>(g, q, limiter, predictor, k, V, D, sg, Ua, out, src, ds, num_sms, st);
    if (variant == 2) return launch_sweep<16, 1>(g, q, limiter, predictor, k, V, D, sg, Ua, out, src, ds, num_sms, st);
    return launch_sweep<24, 1>(g, q, limiter, predictor, k, V, D, sg, Ua, out, src, ds, num_sms, st);
}

} // namespace mf
