// mf_fused.cu — fused path (MF_PATH_FUSED) for fully 3D grids: per RK stage one small predictor kernel and ONE tile kernel.
//
// k_delta_stage (a3+a4): one thread per cell of the grid plus a one-cell ghost ring; limited slopes in x, y, z, the six
//   face fluxes of Eq.13 and the Hancock increment delta (5 doubles per cell) — the only intermediate that goes to HBM.
// k_tile_stage (mf_tile.cu): a1, a3, a5, a6, a7, a8 with face states, fluxes and flux differences on chip.
// The arithmetic per cell and per interface is the same sequence as in the staged path, so the strict build stays
// bit-identical to the oracle.
#include "mf_kernels.h"

namespace mf {

namespace {

constexpr int TPB_D = 256;

// ------------------------------------------------------------------------------------------------ a3 + a4 -> delta
template <int LIM>
__global__ void __launch_bounds__(TPB_D) k_delta_stage(Grid g, Eos q, CState5 V, State5 D, const StepState* __restrict__ ds)
{
    const long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= g.next) return;
    int ie, je, ke;
    unflatten3((unsigned int)p, g.dv[0][2 * g.h[0]], g.dv[1][2 * g.h[1]], ie, je, ke);
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
                       State5 out, Source src, const StepState* ds, int num_sms, int, cudaStream_t st)
{
    return launch_tile_stage(g, q, limiter, predictor, k, V, D, sg, Ua, out, src, ds, num_sms, st);
}

} // namespace mf
