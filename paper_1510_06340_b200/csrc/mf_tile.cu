// mf_tile.cu — fused path, tile kernel (one launch per RK stage after k_delta_stage): a1, a3, a5, a6, a7, a8 on chip.
//
// A CTA of 256 threads owns a tile of 32 x 7 cells in (x, y) and marches through a chunk of z planes.  Work inside the CTA is a
// pool of INTERFACE TASKS, not a thread-per-cell map, so that no thread idles on a ring cell.  Per plane kk:
//   cell parts : 34 x 7 threads rebuild the x face states U~xL, U~xR of the tile's cells and of the two ring cells of each row,
//                32 x 9 threads the y face states (U -/+ slope/2 + delta: a dozen FP64 instructions per component), and drop them
//                into the task arrays in shared memory;                                                              barrier 1
//   tasks      : thread t runs MUSTA on x interface t (33 x 7 = 231 of them), on y interface t (32 x 8 = 256) and, thread-private,
//                on the z interface kk-1/2 of its own column (U~zR(kk-1), U~zL(kk) rebuilt from global memory), after which cell
//                (i, j, kk-1) is complete: L = -((Fx+ - Fx-) + (Fy+ - Fy-) + (Fz+ - Fz-))/dx, source, RK combine, ONE store;   barrier 2
//   differences: (Fx+ - Fx-) + (Fy+ - Fy-) of plane kk per cell, kept in shared memory for the next pass;               barrier 3
// Face states, fluxes and flux differences never touch HBM.  Three CTAs per SM (24 warps) run out of phase with one another.
// Arithmetic per cell and per interface is the staged path's, in the same order: the strict build stays bit-identical to the oracle.
#include "mf_kernels.h"
#include "mf_blocks.cuh"
#include <cuda/barrier>
#include <cstring>

namespace mf {

namespace {

constexpr int NT = 256;
constexpr int TX = 32;               // tile cells along x
constexpr int TY = 7;                // tile cells along y
constexpr int NFX = (TX + 1) * TY;   // x interface tasks = 231
constexpr int NCX = (TX + 2) * TY;   // x cell parts      = 238

// Evolved face states along one axis of the cell at offset o0 (neighbours at om, op; delta at pe in the extended layout):
// lo = U - s/2 + delta, hi = U + s/2 + delta  (Eq.12, Eq.15-17, Eq.13).  Offsets already carry the boundary mapping (a1).
template <int LIM>
__device__ __forceinline__ void faces_at(int predictor, const CState5& V, const CState5& Dl, long long o0, long long om, long long op,
                                         long long pe, double (&lo)[5], double (&hi)[5])
{
#pragma unroll
    for (int v = 0; v < 5; ++v) {
        const double u0 = __ldg(&V.q[v][o0]);
        const double a = u0 - __ldg(&V.q[v][om]), b = __ldg(&V.q[v][op]) - u0;
        const double s = slope2<LIM>(a, b);
        lo[v] = u0 - 0.5 * s;
        hi[v] = u0 + 0.5 * s;
        if (predictor) { const double dl = __ldg(&Dl.q[v][pe]); lo[v] += dl; hi[v] += dl; }
    }
}

// Same face states taken from the scratch arrays that k_cell_stage wrote (hybrid variant): pe indexes the extended layout.
// Strict build: U~dL, U~dR are stored as such; product build: W = U + delta and the half slope H_d (see mf_kernels.cu).
template <int LIM, bool PRE, int D>
__device__ __forceinline__ void faces_any(int predictor, const CState5& V, const CState5& Dl, const Faces& fc, long long o0, long long om,
                                          long long op, long long pe, double (&lo)[5], double (&hi)[5])
{
    if (PRE) {
#pragma unroll
        for (int v = 0; v < 5; ++v) {
#ifdef MF_STRICT
            lo[v] = __ldg(&fc.f[D][0][v][pe]); hi[v] = __ldg(&fc.f[D][1][v][pe]);
#else
            const double w = __ldg(&fc.f[0][1][v][pe]), h = __ldg(&fc.f[D][0][v][pe]);
            lo[v] = w - h; hi[v] = w + h;
#endif
        }
    } else {
        faces_at<LIM>(predictor, V, Dl, o0, om, op, pe, lo, hi);
    }
}

// offsets in the (x, y) plane of a cell that may be a ghost: interior-layout offset with the boundary mapping, extended-layout offset
struct PlaneCell {
    long long o;     // bc(x) + bc(y)*ns1
    long long pe;    // (x+1) + (y+1)*es1
};
__device__ __forceinline__ PlaneCell plane_cell(const Grid& g, int x, int y)
{
    PlaneCell c;
    c.o = (long long)bc_index(x, g.n[0], g.periodic) + (long long)bc_index(y, g.n[1], g.periodic) * g.ns[1];
    c.pe = (x + 1) + (long long)(y + 1) * g.es[1];
    return c;
}

template <int LIM, bool PRE>
__global__ void __launch_bounds__(NT, 3)
k_tile_stage(Grid g, Eos q, int predictor, int k, int TZ, int ntx, int nty, CState5 V, CState5 Dl, Faces fc, Stage sg, CState5 Ua, State5 out,
             Source src, const StepState* __restrict__ ds)
{
    extern __shared__ double sm[];     // 7 arrays of [5][NT] doubles = 70 KB (dynamic: above the 48 KB static limit)
    typedef double (*arr5)[NT];
    arr5 s_Ax = reinterpret_cast<arr5>(sm);                // x tasks: U_L^(0) in, F_x out (task (f, j) = interface between cells f-1, f of row j)
    arr5 s_Bx = reinterpret_cast<arr5>(sm + 5 * NT);       // x tasks: U_R^(0)
    arr5 s_Ay = reinterpret_cast<arr5>(sm + 10 * NT);      // y tasks: U_L^(0) in, F_y out (task (i, f) = interface between rows f-1, f of column i)
    arr5 s_By = reinterpret_cast<arr5>(sm + 15 * NT);      // y tasks: U_R^(0)
    arr5 s_xy = reinterpret_cast<arr5>(sm + 20 * NT);      // per cell: (Fx+ - Fx-) + (Fy+ - Fy-) of the previous plane
    arr5 s_Fz = reinterpret_cast<arr5>(sm + 25 * NT);      // per cell: F_z at the lower face of the previous plane
    arr5 s_zR = reinterpret_cast<arr5>(sm + 30 * NT);      // per cell: U~zR of the previous plane
    // split barrier (arrive ... wait) for "fluxes complete": the thread-private z part runs between arrive and wait and absorbs the skew
#pragma nv_diag_suppress static_var_with_dynamic_init
    __shared__ cuda::barrier<cuda::thread_scope_block> bar_flux;
#pragma nv_diag_default static_var_with_dynamic_init
    if (threadIdx.x == 0) init(&bar_flux, NT);
    __syncthreads();

    const int t = threadIdx.x;
    const int item = blockIdx.x;
    const int tx = item % ntx, ty = (item / ntx) % nty, tz = item / (ntx * nty);
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int x0 = tx * TX, y0 = ty * TY;
    const int z0 = tz * TZ, z1 = min(z0 + TZ, nz);
    const double dt = ds->dt;
    const MustaCoef mcf = musta_coef_of(ds);
    const long long ns2 = g.ns[2], es2 = g.es[2];

    // ---- roles of this thread, fixed for the whole march (plane offsets fit in 32 bits)
    // x cell part: cell (x0 + xc, y0 + xj), xc = -1 .. 32
    const int xj = t / (TX + 2), xc = t % (TX + 2) - 1;
    const bool xpart = t < NCX && x0 + xc <= nx && y0 + xj < ny;
    int xo0 = 0, xom = 0, xop = 0, xpe = 0;
    if (xpart) {
        PlaneCell c = plane_cell(g, x0 + xc, y0 + xj);
        xo0 = (int)c.o; xpe = (int)c.pe;
        xom = (int)plane_cell(g, x0 + xc - 1, y0 + xj).o; xop = (int)plane_cell(g, x0 + xc + 1, y0 + xj).o;
    }
    // y cell part: cell (x0 + yi, y0 + yc), yc = -1 .. 6 (the top ring row yc = 7 is a second part of warp 0)
    const int yi = t % TX, yc = t / TX - 1;
    const bool ypart = x0 + yi < nx && y0 + yc <= ny;
    int yo0 = 0, yom = 0, yop = 0, ype = 0;
    if (ypart) {
        PlaneCell c = plane_cell(g, x0 + yi, y0 + yc);
        yo0 = (int)c.o; ype = (int)c.pe;
        yom = (int)plane_cell(g, x0 + yi, y0 + yc - 1).o; yop = (int)plane_cell(g, x0 + yi, y0 + yc + 1).o;
    }
    const bool ypart2 = t < TX && x0 + t < nx && y0 + TY <= ny;
    // tasks
    const bool xtask = t < NFX && x0 + t % (TX + 1) <= nx && y0 + t / (TX + 1) < ny;
    const bool ytask = y0 + t / TX <= ny && x0 + yi < nx;
    // own cell (z part, differences): t = cj*32 + ci
    const int ci = t % TX, cj = t / TX;
    const int gx = x0 + ci, gy = y0 + cj;
    const bool cell_ok = cj < TY && gx < nx && gy < ny;
    const int co = gx + gy * (int)g.ns[1], cpe = (gx + 1) + (gy + 1) * (int)g.es[1];

    for (int kk = z0; kk <= z1; ++kk) {
        const bool plane = kk < z1;                                  // the last pass only closes plane z1-1
        // ---------------------------------------------------------------- cell parts of plane kk -> task arrays
        if (plane) {
            const long long oz = (long long)kk * ns2, pz = (long long)(kk + 1) * es2;
            if (xpart) {
                double lo[5], hi[5];
                faces_any<LIM, PRE, 0>(predictor, V, Dl, fc,xo0 + oz, xom + oz, xop + oz, xpe + pz, lo, hi);
                if (xc <= TX - 1) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) s_Ax[v][xj * (TX + 1) + xc + 1] = hi[v];   // U~xR of cell c is U_L^(0) of interface c+1/2
                }
                if (xc >= 0) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) s_Bx[v][xj * (TX + 1) + xc] = lo[v];       // U~xL of cell c is U_R^(0) of interface c-1/2
                }
            }
            if (ypart) {
                double lo[5], hi[5];
                faces_any<LIM, PRE, 1>(predictor, V, Dl, fc,yo0 + oz, yom + oz, yop + oz, ype + pz, lo, hi);
#pragma unroll
                for (int v = 0; v < 5; ++v) s_Ay[v][(yc + 1) * TX + yi] = hi[v];
                if (yc >= 0) {
#pragma unroll
                    for (int v = 0; v < 5; ++v) s_By[v][yc * TX + yi] = lo[v];
                }
            }
            if (ypart2) {                                            // top ring row: only its lower face is needed
                double lo[5], hi[5];
                PlaneCell c = plane_cell(g, x0 + t, y0 + TY);
                faces_any<LIM, PRE, 1>(predictor, V, Dl, fc,c.o + oz, plane_cell(g, x0 + t, y0 + TY - 1).o + oz, plane_cell(g, x0 + t, y0 + TY + 1).o + oz,
                              c.pe + pz, lo, hi);
#pragma unroll
                for (int v = 0; v < 5; ++v) s_By[v][TY * TX + t] = lo[v];
            }
        }
        __syncthreads();                                             // 1: task inputs complete
        // ---------------------------------------------------------------- tasks
        if (plane && xtask) {
            double A[5], B[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = s_Ax[v][t]; B[v] = s_Bx[v][t]; }
            musta_flux<0>(q, k, mcf, A, B, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) s_Ax[v][t] = F[v];           // only this task reads slot t
        }
        if (plane && ytask) {
            double A[5], B[5], F[5];
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = s_Ay[v][t]; B[v] = s_By[v][t]; }
            musta_flux<1>(q, k, mcf, A, B, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) s_Ay[v][t] = F[v];
        }
        auto token = bar_flux.arrive();                              // 2a: this thread's x and y fluxes of plane kk are in shared memory
        if (cell_ok) {                                               // z interface kk-1/2: thread-private, overlaps the other warps' tasks
            const long long zm1 = (long long)bc_index(kk - 1, nz, g.periodic) * ns2;
            const long long zc = (long long)bc_index(kk, nz, g.periodic) * ns2, zp1 = (long long)bc_index(kk + 1, nz, g.periodic) * ns2;
            double A[5], B[5], F[5], hi[5];
            if (kk == z0) {                                          // first pass of the chunk: U~zR of plane kk-1 is not carried yet
                const long long zm2 = (long long)bc_index(kk - 2, nz, g.periodic) * ns2;
                faces_any<LIM, PRE, 2>(predictor, V, Dl, fc,co + zm1, co + zm2, co + zc, cpe + (long long)kk * es2, B, A);
            } else {
#pragma unroll
                for (int v = 0; v < 5; ++v) A[v] = s_zR[v][t];
            }
            faces_any<LIM, PRE, 2>(predictor, V, Dl, fc,co + zc, co + zm1, co + zp1, cpe + (long long)(kk + 1) * es2, B, hi);    // U~zL, U~zR of plane kk
#pragma unroll
            for (int v = 0; v < 5; ++v) s_zR[v][t] = hi[v];
            if (kk + 1 < z1) {                                       // pull the next new plane towards L2 while MUSTA runs
                const long long zp2 = (long long)bc_index(kk + 2, nz, g.periodic) * ns2;
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    if (PRE) { prefetch_l2(&fc.f[0][1][v][cpe + (long long)(kk + 2) * es2]); prefetch_l2(&fc.f[2][0][v][cpe + (long long)(kk + 2) * es2]); }
                    else { prefetch_l2(&V.q[v][co + zp2]); prefetch_l2(&Dl.q[v][cpe + (long long)(kk + 2) * es2]); }
                }
            }
            musta_flux<2>(q, k, mcf, A, B, F);
            if (kk > z0) {                                           // cell (gx, gy, kk-1) is complete
                const int kc = kk - 1;
                const long long o = co + (long long)kc * ns2;
                double S = 0.0;
                if (src.on) S = jet_source(g, src, gx, gy, kc, ds->t + sg.ts * dt);
                double ua5[5], ub5[5];                                   // loaded before the first store (`out` may alias them for all the compiler knows)
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    ua5[v] = sg.form == 3 ? 0.0 : Ua.q[v][o];
                    ub5[v] = (sg.form == 1 || sg.form == 2) ? V.q[v][o] : 0.0;
                }
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    double acc = s_xy[v][t] + (F[v] - s_Fz[v][t]);
#ifdef MF_STRICT
                    double L = -acc / g.dx;
#else
                    double L = -acc * g.inv_dx;
#endif
                    if (src.on && v < 2) L = L + S;
                    out.q[v][o] = rk_form(sg, ua5[v], ub5[v], dt, L);
                }
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) s_Fz[v][t] = F[v];
        }
        bar_flux.wait(std::move(token));                             // 2b: fluxes of plane kk complete
        if (!plane) break;
        if (cell_ok) {
#pragma unroll
            for (int v = 0; v < 5; ++v)
                s_xy[v][t] = (s_Ax[v][cj * (TX + 1) + ci + 1] - s_Ax[v][cj * (TX + 1) + ci]) + (s_Ay[v][(cj + 1) * TX + ci] - s_Ay[v][cj * TX + ci]);
        }
        __syncthreads();                                             // 3: the task arrays may be overwritten
    }
}

} // namespace

static int tile_chunk(const Grid& g, int ntx, int nty, int num_sms)
{
    // z chunk: all of z, or the largest of {64, 32, 16, 8} planes for which the items fill the 3 resident CTA slots per SM ~6 times over
    int TZ = g.n[2];
    const int cands[4] = { 64, 32, 16, 8 };
    for (int c = 0; c < 4; ++c) {
        long long items = (long long)ntx * nty * ((g.n[2] + TZ - 1) / TZ);
        if (items >= 18LL * num_sms) break;
        if (cands[c] < TZ) TZ = cands[c];
    }
    return TZ;
}

int launch_tile_stage(const Grid& g, const Eos& q, int limiter, int predictor, int k, CState5 V, CState5 D, Stage sg, CState5 Ua, State5 out,
                      Source src, const StepState* ds, int num_sms, cudaStream_t st)
{
    const int ntx = (g.n[0] + TX - 1) / TX, nty = (g.n[1] + TY - 1) / TY;
    const int TZ = tile_chunk(g, ntx, nty, num_sms);
    const unsigned int grid = (unsigned int)(ntx * nty * ((g.n[2] + TZ - 1) / TZ));
    const size_t smem = sizeof(double) * 35 * NT;
    Faces none; memset(&none, 0, sizeof(none));
#define MF_CASE(L) case L: { \
        static DeviceOnce once; \
        if (once.first()) cudaFuncSetAttribute(k_tile_stage<L, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem); \
        k_tile_stage<L, false><<<grid, NT, smem, st>>>(g, q, predictor, k, TZ, ntx, nty, V, D, none, sg, Ua, out, src, ds); } break;
    switch (limiter) {
        MF_CASE(LIM_NONE) MF_CASE(LIM_MINMOD) MF_CASE(LIM_SUPERBEE) MF_CASE(LIM_VANALBADA) MF_CASE(LIM_VANLEER) MF_CASE(LIM_MC) MF_CASE(LIM_FIRST)
    default: return 0;
    }
#undef MF_CASE
    return 1;
}

// hybrid: face states come from k_cell_stage's scratch (fc); the tile kernel does the three flux directions and the combine
int launch_tile_stage_pre(const Grid& g, const Eos& q, int k, Faces fc, CState5 V, Stage sg, CState5 Ua, State5 out, Source src,
                          const StepState* ds, int num_sms, cudaStream_t st)
{
    const int ntx = (g.n[0] + TX - 1) / TX, nty = (g.n[1] + TY - 1) / TY;
    const int TZ = tile_chunk(g, ntx, nty, num_sms);
    const unsigned int grid = (unsigned int)(ntx * nty * ((g.n[2] + TZ - 1) / TZ));
    const size_t smem = sizeof(double) * 35 * NT;
    static DeviceOnce once;
    if (once.first()) cudaFuncSetAttribute(k_tile_stage<LIM_NONE, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    k_tile_stage<LIM_NONE, true><<<grid, NT, smem, st>>>(g, q, 0, k, TZ, ntx, nty, V, V, fc, sg, Ua, out, src, ds);
    return 1;
}

} // namespace mf
