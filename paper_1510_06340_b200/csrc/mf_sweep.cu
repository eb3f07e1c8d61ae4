// mf_sweep.cu — sweep path (MF_PATH_SWEEP): per-direction sweep kernels that read the cell averages themselves.
//
// Each interface thread loads the four cell averages around its interface along the sweep axis (a +-2-cell halo, boundary
// handling a1 as index mapping), limits the two slopes it needs in registers (a3, Eq.12, 15-22 :155-211), runs MUSTA_k with
// FORCE-alpha and the closed-form con2prim (a5, a6) and writes the interface flux once.  No face states, half slopes or
// W = U + delta ever go to HBM: with the Hancock half step off (reading A4: MUSCL + RK, what BASELINE.json's north_star
// pictures as "a fused per-direction sweep kernel with a +-2-cell halo along the sweep axis") an RK stage is three launches
// and touches 40 (y) + 40 (z) + 40 (x) bytes of U per cell instead of a 200 B/cell cell stage plus 80 B/cell per direction.
// With the half step on (3D grids), k_delta_stage (mf_fused.cu) writes the increment delta of Eq.13 once per cell (40 B) and
// the sweeps add it to both face states (A3).
//
//   k_sweep_flux<D, PRED>            y and z interfaces: F_y, F_z to HBM (extended layout, like the staged path)
//   k_sweep_xcombine<PRED,FORM,CFL>  x interfaces + divergence + source + RK combine (+ CFL reduction): F_x stays on chip
//
// The arithmetic per interface is the staged path's, so the strict build stays bit-identical to the oracle.
// p = cs2*e only; the tabulated EOS runs on the staged path.
#include "mf_kernels.h"
#include "mf_blocks.cuh"

namespace mf {

namespace {

// Face states at the interface between cells c and c+1 along one axis from the averages of cells c-1, c, c+1, c+2:
// A = U~_c^R = U_c + slope_c/2, B = U~_{c+1}^L = U_{c+1} - slope_{c+1}/2 (Eq.12 :157-161, reading A2).
template <int LIM>
__device__ __forceinline__ void face_pair(const double (&um)[5], const double (&u0)[5], const double (&u1)[5], const double (&u2)[5],
                                          double (&A)[5], double (&B)[5])
{
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double d0 = u0[v] - um[v], d1 = u1[v] - u0[v], d2 = u2[v] - u1[v];
#ifdef MF_STRICT
        A[v] = u0[v] + 0.5 * slope2<LIM>(d0, d1);                            // the oracle's order: U + 0.5*s, U - 0.5*s
        B[v] = u1[v] - 0.5 * slope2<LIM>(d1, d2);
#else
        A[v] = u0[v] + half_slope2<LIM>(d0, d1);
        B[v] = u1[v] - half_slope2<LIM>(d1, d2);
#endif
    }
}

// the limiter is uniform over the launch: one switch per thread, outside the component loop
__device__ __forceinline__ void face_pair_rt(int lim, const double (&um)[5], const double (&u0)[5], const double (&u1)[5], const double (&u2)[5],
                                             double (&A)[5], double (&B)[5])
{
    switch (lim) {
    case LIM_MINMOD:    face_pair<LIM_MINMOD>(um, u0, u1, u2, A, B); break;
    case LIM_SUPERBEE:  face_pair<LIM_SUPERBEE>(um, u0, u1, u2, A, B); break;
    case LIM_MC:        face_pair<LIM_MC>(um, u0, u1, u2, A, B); break;
    case LIM_VANLEER:   face_pair<LIM_VANLEER>(um, u0, u1, u2, A, B); break;
    case LIM_VANALBADA: face_pair<LIM_VANALBADA>(um, u0, u1, u2, A, B); break;
    case LIM_NONE:      face_pair<LIM_NONE>(um, u0, u1, u2, A, B); break;
    default:            face_pair<LIM_FIRST>(um, u0, u1, u2, A, B); break;
    }
}

// offsets (interior layout, in units of the axis stride) of cells c-1 .. c+2 along an axis of extent n
__device__ __forceinline__ void halo4(int c, int n, int periodic, unsigned int stride, unsigned int base, unsigned int (&o)[4])
{
#pragma unroll
    for (int s = 0; s < 4; ++s) o[s] = base + (unsigned int)bc_index(c - 1 + s, n, periodic) * stride;
}

// =========================================================================== a1 + a3 + a5 + a6 along y or z
// One thread per interface between cells c and c+e_D; c runs over -1..n_D-1 along D and the interior on the other axes.
template <int D, bool PRED, class ST>
__device__ __forceinline__ void sweep_flux_body(const Grid& g, const Eos& q, int lim, int k, const CState5& V, const CState5& Dl, const Fluxes& fx,
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
    const unsigned int ns[3] = { (unsigned int)g.ns[0], (unsigned int)g.ns[1], (unsigned int)g.ns[2] };
    const unsigned int es[3] = { (unsigned int)g.es[0], (unsigned int)g.es[1], (unsigned int)g.es[2] };
    unsigned int base = blockIdx.y * (unsigned int)g.ncell;
#pragma unroll
    for (int a = 0; a < 3; ++a) if (a != D) base += (unsigned int)c[a] * ns[a];
    unsigned int o[4];
    halo4(c[D], g.n[D], g.periodic, ns[D], base, o);
    const unsigned int p = blockIdx.y * (unsigned int)g.next + (c[0] + g.h[0]) * es[0] + (c[1] + g.h[1]) * es[1] + (c[2] + g.h[2]) * es[2];
    ds += blockIdx.y;
    double A[5], B[5], F[5];
    {
        double um[5], u0[5], u1[5], u2[5];
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            const ST* Vv = reinterpret_cast<const ST*>(V.q[v]);                  // state element type (reading A19): widened on the load
            um[v] = (double)__ldg(Vv + o[0]); u0[v] = (double)__ldg(Vv + o[1]); u1[v] = (double)__ldg(Vv + o[2]); u2[v] = (double)__ldg(Vv + o[3]);
        }
        face_pair_rt(lim, um, u0, u1, u2, A, B);
    }
    if (PRED) {                                                              // Eq.13: the same increment on every face of a cell (A3)
#pragma unroll
        for (int v = 0; v < 5; ++v) { A[v] = A[v] + __ldg(&Dl.q[v][p]); B[v] = B[v] + __ldg(&Dl.q[v][p + es[D]]); }
    }
    musta_flux<D, 0>(q, k, musta_coef_of(ds), A, B, F);
#pragma unroll
    for (int v = 0; v < 5; ++v) fx.f[D][v][p] = F[v];
}

template <int D, bool PRED, class ST>
__global__ void __launch_bounds__(TPB, 3) k_sweep_flux(Grid g, Eos q, int lim, int k, CState5 V, CState5 Dl, Fluxes fx, const StepState* ds)
{
    sweep_flux_body<D, PRED, ST>(g, q, lim, k, V, Dl, fx, ds, blockIdx.x);
}

// the y and the z sweep of a stage are independent: one launch for both, one kernel boundary less
template <bool PRED, class ST>
__global__ void __launch_bounds__(TPB, 3) k_sweep_flux_yz(Grid g, Eos q, int lim, int k, CState5 V, CState5 Dl, Fluxes fx, const StepState* ds, unsigned int nby)
{
    // even blocks take y, odd blocks z of the same stretch of cells (the lines one reads are still in L2 when the other reads them)
    const unsigned int b = blockIdx.x >> 1;
    if ((blockIdx.x & 1u) == 0) { if (b < nby) sweep_flux_body<1, PRED, ST>(g, q, lim, k, V, Dl, fx, ds, b); }
    else sweep_flux_body<2, PRED, ST>(g, q, lim, k, V, Dl, fx, ds, b);
}

// =========================================================================== a1 + a3 + a5 (x) + a6 + a7 + a8 (+ a2)
// The x sweep is the last one of a stage and finishes the cells, like k_xflux_combine of the staged path: thread t of a block owns
// x interface I = (XT-1)*block + t (linear over all rows, nx+1 per row), leaves its MUSTA flux in shared memory, and the cell to the right
// of the interface then has both of its x fluxes on chip, reads F_y, F_z of its four other faces, and is done: one store per cell.
#ifndef MF_XT
#define MF_XT 128
#endif
#ifndef MF_XB
#define MF_XB 5
#endif
constexpr int XT = MF_XT, XB = MF_XB;                // threads per block of the x sweep, blocks per SM (96 registers: the combine holds its operands across the barrier)
template <bool PRED, int FORM, bool CFL, class ST>
__global__ void __launch_bounds__(XT, XB) k_sweep_xcombine(Grid g, Eos q, int lim, int k, CState5 V, CState5 Dl, Fluxes fx, Stage sg, CState5 Ua,
                                                           State5 out, Source src, StepState* ds)
{
    __shared__ double sF[5][XT];
    const int t = threadIdx.x;
    const int nf = g.n[0] + 1;                                              // x interfaces per row
    const long long nrows = (long long)g.n[1] * g.n[2];
    const long long I = (long long)blockIdx.x * (XT - 1) + t;
    const bool live = I < nrows * nf;
    int f = 0, j = 0, kz = 0;
    unsigned int p = 0, row = 0;
    double F[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
    const unsigned int eo = blockIdx.y * (unsigned int)g.ncell, ep = blockIdx.y * (unsigned int)g.next;   // this block's event
    ds += blockIdx.y;
    if (live) {
        unflatten3((unsigned int)I, g.dv[0][1], g.dv[1][0], f, j, kz);                       // f: interface between cells f-1 and f of row (j, kz)
        row = eo + (unsigned int)j * (unsigned int)g.ns[1] + (unsigned int)kz * (unsigned int)g.ns[2];
        p = ep + f + (unsigned int)(j + g.h[1]) * (unsigned int)g.es[1] + (unsigned int)(kz + g.h[2]) * (unsigned int)g.es[2];   // extended index of cell f-1
        unsigned int o[4];
        halo4(f - 1, g.n[0], g.periodic, 1u, row, o);
        double A[5], B[5];
        {
            double um[5], u0[5], u1[5], u2[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) {
            const ST* Vv = reinterpret_cast<const ST*>(V.q[v]);                  // state element type (reading A19): widened on the load
            um[v] = (double)__ldg(Vv + o[0]); u0[v] = (double)__ldg(Vv + o[1]); u1[v] = (double)__ldg(Vv + o[2]); u2[v] = (double)__ldg(Vv + o[3]);
        }
            face_pair_rt(lim, um, u0, u1, u2, A, B);
        }
        if (PRED) {
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = A[v] + __ldg(&Dl.q[v][p]); B[v] = B[v] + __ldg(&Dl.q[v][p + 1]); }
        }
        musta_flux<0, 0>(q, k, musta_coef_of(ds), A, B, F);
    }
    // The combine's operands: all loaded before the first store (`out` may alias the inputs as far as the compiler knows: loads written after
    // a store would wait for it - five dependent round trips to memory instead of one), and issued before the barrier, so that their
    // latency runs while the block's other warps finish MUSTA.
    const bool owns_cell = live && t < XT - 1 && f < g.n[0];                // cell (f, j, kz): lower x face = this interface, upper = thread t+1's
    const unsigned int pc = p + 1;
    const unsigned int oc = row + f;
    double fy1[5], fy0[5], fz1[5], fz0[5], ua5[5], ub5[5];
    if (owns_cell) {
#pragma unroll
        for (int v = 0; v < 5; ++v) {
            if (g.act[1]) { fy1[v] = fx.f[1][v][pc]; fy0[v] = fx.f[1][v][pc - (unsigned int)g.es[1]]; }
            if (g.act[2]) { fz1[v] = fx.f[2][v][pc]; fz0[v] = fx.f[2][v][pc - (unsigned int)g.es[2]]; }
            ua5[v] = FORM == 3 ? 0.0 : ld_state<ST>(Ua.q[v], oc);
            ub5[v] = (FORM == 1 || FORM == 2) ? ld_state<ST>(V.q[v], oc) : 0.0;           // U_(s) is the state the sweep ran on
        }
    }
#pragma unroll
    for (int v = 0; v < 5; ++v) sF[v][t] = F[v];
    __syncthreads();
    double smax = 0.0;
    int bad = 0;
    if (owns_cell) {
        const double dt = ds->dt;
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
            if (FORM == 3) out.q[v][oc] = W[v];                            // L itself (mf_eval_L): double whatever the state precision
            else st_state<ST>(out.q[v], oc, W[v]);
        }
        if (CFL) {                                                         // S_max of the STORED (rounded) new state
#pragma unroll
            for (int v = 0; v < 5; ++v) W[v] = as_stored<ST>(W[v]);
            smax = signal_speed<0>(q, W[0], W[1], W[2], W[3], W[4], bad);
        }
    }
    if (CFL) block_reduce_smax<XT>(smax, bad, ds);
}

} // namespace

bool sweep_supported(const Grid& g, int eos_kind, int predictor)
{
    if (!g.act[0] || eos_kind != 0) return false;                             // the x sweep finishes the cells; closed-form EOS only
    if (g.state32 && predictor) return false;                                 // k_delta_stage reads an fp64 state
    if (predictor && !(g.act[1] && g.act[2] && g.nev == 1)) return false;     // delta comes from k_delta_stage (3D, one event)
    return true;
}

int launch_sweep_flux(const Grid& g, const Eos& q, int limiter, int k, bool pred, CState5 V, CState5 Dl, Fluxes fx, const StepState* ds, cudaStream_t st)
{
    int launches = 0;
    if (g.act[1] && g.act[2]) {
        const unsigned int nby = (unsigned int)(((long long)g.n[0] * (g.n[1] + 1) * g.n[2] + TPB - 1) / TPB);
        const unsigned int nbz = (unsigned int)(((long long)g.n[0] * g.n[1] * (g.n[2] + 1) + TPB - 1) / TPB);
        const dim3 nb(2 * (nby > nbz ? nby : nbz), g.nev);
#define MF_SFYZ(ST_) do { if (pred) k_sweep_flux_yz<true, ST_><<<nb, TPB, 0, st>>>(g, q, limiter, k, V, Dl, fx, ds, nby); \
                          else k_sweep_flux_yz<false, ST_><<<nb, TPB, 0, st>>>(g, q, limiter, k, V, Dl, fx, ds, nby); } while (0)
        if (g.state32) MF_SFYZ(float); else MF_SFYZ(double);
#undef MF_SFYZ
        return 1;
    }
    for (int d = 1; d < 3; ++d) {
        if (!g.act[d]) continue;
        long long total = 1;
        for (int a = 0; a < 3; ++a) total *= (a == d) ? g.n[a] + 1 : g.n[a];
        const dim3 nb((unsigned int)((total + TPB - 1) / TPB), g.nev);
#define MF_SF(D_, ST_) do { if (pred) k_sweep_flux<D_, true, ST_><<<nb, TPB, 0, st>>>(g, q, limiter, k, V, Dl, fx, ds); \
                            else k_sweep_flux<D_, false, ST_><<<nb, TPB, 0, st>>>(g, q, limiter, k, V, Dl, fx, ds); } while (0)
        if (d == 1) { if (g.state32) MF_SF(1, float); else MF_SF(1, double); }
        else        { if (g.state32) MF_SF(2, float); else MF_SF(2, double); }
#undef MF_SF
        ++launches;
    }
    return launches;
}

int launch_sweep_xcombine(const Grid& g, const Eos& q, int limiter, int k, bool pred, CState5 V, CState5 Dl, Fluxes fx, Stage sg, CState5 Ua, State5 out,
                          Source src, StepState* ds, cudaStream_t st)
{
    const long long total = (long long)(g.n[0] + 1) * g.n[1] * g.n[2];
    const dim3 nb((unsigned int)((total + XT - 2) / (XT - 1)), g.nev);
#define MF_SXC(P_, FORM_, CFL_) do { if (g.state32) k_sweep_xcombine<P_, FORM_, CFL_, float><<<nb, XT, 0, st>>>(g, q, limiter, k, V, Dl, fx, sg, Ua, out, src, ds); \
                                     else k_sweep_xcombine<P_, FORM_, CFL_, double><<<nb, XT, 0, st>>>(g, q, limiter, k, V, Dl, fx, sg, Ua, out, src, ds); } while (0)
#define MF_SXC_FORMS(P_) \
    if (sg.form == 0) { if (sg.cfl) MF_SXC(P_, 0, true); else MF_SXC(P_, 0, false); } \
    else if (sg.form == 1) { if (sg.cfl) MF_SXC(P_, 1, true); else MF_SXC(P_, 1, false); } \
    else if (sg.form == 2) { if (sg.cfl) MF_SXC(P_, 2, true); else MF_SXC(P_, 2, false); } \
    else MF_SXC(P_, 3, false);
    if (pred) { MF_SXC_FORMS(true) } else { MF_SXC_FORMS(false) }
#undef MF_SXC_FORMS
#undef MF_SXC
    return 1;
}

} // namespace mf
