// mf_tile.cu — the two tile kernels (3D grids, p = cs2*e, one event):
//
//   k_tile3      (MF_PATH_HYBRID, round 2): fed by the staged cell stage's scratch (W = U + delta, half slopes); a CTA of 256 threads owns
//                32 x 7 cells and marches in z; every x, y and z interface is a TASK of one thread, which loads its own operands from
//                global memory (L1/L2, the next plane prefetched line by line) and runs MUSTA; only the finished fluxes go through shared
//                memory; divergence, source, RK combine and the CFL reduction of plane k-1 follow the z interface that completes it; ONE
//                split barrier per plane.  See the comment above the kernel.
//   k_tile_stage (MF_PATH_FUSED, round 1): one launch per RK stage after k_delta_stage: a1, a3, a5, a6, a7, a8 on chip.
//
// k_tile_stage: a CTA of 256 threads owns a tile of 32 x 7 cells in (x, y) and marches through a chunk of z planes.  Work inside the CTA is a
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
#include "mf_stepconst.cuh"
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

// ================================================================================================ hybrid path, second form
// k_tile3: the three flux directions + divergence + source + RK combine (+ CFL reduction) of one RK stage, fed by the cell stage's scratch
// (W = U + delta and the half slopes H_d in the extended layout, so no boundary mapping here).  Same tile and z march as k_tile_stage, but
//   * every interface task loads its own operands from global memory (L1/L2), exactly like the staged flux kernels do - there is no
//     "cell part" phase, no face-state staging in shared memory and no barrier in front of the tasks;
//   * only the finished fluxes go through shared memory (F_x, F_y double-buffered by plane parity, F_z in a thread-private slot), and the
//     divergence of plane kk-1 is formed one iteration later, right after the z interface kk-1/2 that completes it;
//   * ONE split barrier per plane: arrive after the x and y fluxes of plane kk are stored, wait after the next iteration's z MUSTA - a
//     third of an iteration's work lies between the two, so the wait rarely blocks;
//   * the lines of the next plane (W, H_x, H_y, H_z, U^n, U_(s)) are pulled towards L2 by one prefetch per 128 B line, not per thread;
//   * the signal speed of the new state goes into the block reduction on the last stage (a2), so the hybrid path needs no separate CFL pass.
// Iteration kk:  z task (kk-1/2) | wait(kk-1) | combine plane kk-1 | x tasks, y tasks of plane kk -> sF[kk&1] | arrive(kk)
template <bool CFL, bool UC>
__global__ void __launch_bounds__(NT, 3)
k_tile3(Grid g, Eos q, int k, int TZ, int ntx, int nty, Faces fc, CState5 Wc, CState5 V, Stage sg, CState5 Ua, State5 out, Source src, StepState* ds)
{
    __shared__ double sFx[2][5][NFX];
    __shared__ double sFy[2][5][NT];
    __shared__ double sFz[5][TX * TY];
#pragma nv_diag_suppress static_var_with_dynamic_init
    __shared__ cuda::barrier<cuda::thread_scope_block> bar;
#pragma nv_diag_default static_var_with_dynamic_init
    if (threadIdx.x == 0) init(&bar, NT);
    __syncthreads();

    const int t = threadIdx.x;
    const int item = blockIdx.x;
    const int tx = item % ntx, ty = (item / ntx) % nty, tz = item / (ntx * nty);
    const int nx = g.n[0], ny = g.n[1], nz = g.n[2];
    const int x0 = tx * TX, y0 = ty * TY;
    const int z0 = tz * TZ, z1 = min(z0 + TZ, nz);
    const StepConst sc = step_scalars<UC>(g, ds);
    const MustaCoef mcf = musta_coef(sc);
    const unsigned int es1 = (unsigned int)g.es[1], es2 = (unsigned int)g.es[2], ns1 = (unsigned int)g.ns[1], ns2 = (unsigned int)g.ns[2];

    // ---- roles of this thread, fixed for the whole march.  Offsets are in-plane; the plane is added per iteration.
    // x task: interface f = t % 33 of row j = t / 33, between cells (x0+f-1, y0+j) and (x0+f, y0+j); xp = extended offset of the left cell
    const int xf = t % (TX + 1), xj = t / (TX + 1);
    const bool xtask = t < NFX && x0 + xf <= nx && y0 + xj < ny;
    const unsigned int xp = (unsigned int)(x0 + xf) + (unsigned int)(y0 + xj + 1) * es1;
    // y task: interface f = t / 32 of column i = t % 32, between cells (x0+i, y0+f-1) and (x0+i, y0+f); yp = extended offset of the lower cell
    const int yi = t % TX, yf = t / TX;
    const bool ytask = x0 + yi < nx && y0 + yf <= ny;
    const unsigned int yp = (unsigned int)(x0 + yi + 1) + (unsigned int)(y0 + yf) * es1;
    // own cell (z task, combine): t = cj*32 + ci
    const int ci = yi, cj = yf;
    const int gx = x0 + ci, gy = y0 + cj;
    const bool cell_ok = cj < TY && gx < nx && gy < ny;
    const unsigned int co = (unsigned int)gx + (unsigned int)gy * ns1, cpe = (unsigned int)(gx + 1) + (unsigned int)(gy + 1) * es1;

    double smax = 0.0;
    int bad = 0;
    cuda::barrier<cuda::thread_scope_block>::arrival_token token;
    for (int kk = z0; kk <= z1; ++kk) {
        const int buf = kk & 1;
        // ---------------------------------------------------------------- lines of the next plane towards L2: one prefetch per line
        if (kk + 1 < z1) {
            if (t < 20 * (TY + 2)) {                                 // W, H_x, H_y, H_z (5 components each), rows y0-1 .. y0+TY of the tile
                const int a = t / (TY + 2), r = t - a * (TY + 2);
                if (y0 + r <= ny + 1) {
                    // (no run-time index into the kernel parameters: the scratch arrays are consecutive slots of one allocation - H_x 0..4, W 5..9,
                    //  H_y 10..14, H_z 20..24 in units of g.next, see faces_of in mf_api.cu)
                    const double* base = fc.f[0][0][0] + (unsigned long long)(a < 15 ? a : a + 5) * (unsigned long long)g.next;
                    const char* p0 = reinterpret_cast<const char*>(base + (unsigned int)x0 + (unsigned int)(y0 + r) * es1 + (unsigned int)(kk + 2) * es2);
                    const int len = 8 * min(TX + 2, nx + 2 - x0);
                    for (int off = 0; off < len; off += 128) prefetch_l2(p0 + off);
                    prefetch_l2(p0 + len - 8);
                }
            } else if (t < 20 * (TY + 2) + 10 * TY) {                // U^n and U_(s) of the cells that the next iteration finishes ... of plane kk
                const int u = t - 20 * (TY + 2);
                const int a = u / TY, r = u - a * TY;
                if (y0 + r < ny) {
                    const double* base = (a < 5 ? Ua.q[0] : V.q[0]) + (unsigned long long)(a < 5 ? a : a - 5) * (unsigned long long)g.ncell;
                    const char* p0 = reinterpret_cast<const char*>(base + (unsigned int)x0 + (unsigned int)(y0 + r) * ns1 + (unsigned int)kk * ns2);
                    const int len = 8 * min(TX, nx - x0);
                    for (int off = 0; off < len; off += 128) prefetch_l2(p0 + off);
                    prefetch_l2(p0 + len - 8);
                }
            }
        }
        // ---------------------------------------------------------------- z interface kk-1/2 of the own column
        double Fz[5] = { 0.0, 0.0, 0.0, 0.0, 0.0 };
        if (cell_ok) {
            const unsigned int p = cpe + (unsigned int)kk * es2, pn = p + es2;      // extended plane kk holds interior plane kk-1
            double A[5], B[5];
#ifdef MF_STRICT
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = fc.f[2][1][v][p]; B[v] = fc.f[2][0][v][pn]; }
#else
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = Wc.q[v][p] + fc.f[2][0][v][p]; B[v] = Wc.q[v][pn] - fc.f[2][0][v][pn]; }
#endif
            musta_flux<2>(q, k, mcf, A, B, Fz);
        }
        if (kk > z0) bar.wait(std::move(token));                     // F_x, F_y of plane kk-1 are complete; buffer `buf` is free again
        if (cell_ok) {
            if (kk > z0) {                                           // cell (gx, gy, kk-1) is complete
                const int kc = kk - 1, pb = buf ^ 1;
                const unsigned int o = co + (unsigned int)kc * ns2;
                const double dt = sc.dt;
                double S = 0.0;
                if (src.on) S = jet_source(g, src, gx, gy, kc, ds->t + sg.ts * dt);
                double ua5[5], ub5[5];                               // loaded before the first store (`out` may alias them for all the compiler knows)
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    ua5[v] = sg.form == 3 ? 0.0 : Ua.q[v][o];
                    ub5[v] = (sg.form == 1 || sg.form == 2) ? V.q[v][o] : 0.0;
                }
                double W[5];
#pragma unroll
                for (int v = 0; v < 5; ++v) {
                    double acc = sFx[pb][v][cj * (TX + 1) + ci + 1] - sFx[pb][v][cj * (TX + 1) + ci];
                    acc = acc + (sFy[pb][v][(cj + 1) * TX + ci] - sFy[pb][v][cj * TX + ci]);
                    acc = acc + (Fz[v] - sFz[v][t]);
#ifdef MF_STRICT
                    double L = -acc / g.dx;                          // Eq.1 :43
#else
                    double L = -acc * g.inv_dx;
#endif
                    if (src.on && v < 2) L = L + S;
                    W[v] = rk_form(sg, ua5[v], ub5[v], dt, L);
                    out.q[v][o] = W[v];
                }
                if (CFL) smax = fmax(smax, signal_speed<0>(q, W[0], W[1], W[2], W[3], W[4], bad));
            }
#pragma unroll
            for (int v = 0; v < 5; ++v) sFz[v][t] = Fz[v];
        }
        if (kk == z1) break;                                         // the last pass only closes plane z1-1
        // ---------------------------------------------------------------- x and y interfaces of plane kk
        const unsigned int pz = (unsigned int)(kk + 1) * es2;
        if (xtask) {
            const unsigned int p = xp + pz;
            double A[5], B[5], F[5];
#ifdef MF_STRICT
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = fc.f[0][1][v][p]; B[v] = fc.f[0][0][v][p + 1]; }
#else
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = Wc.q[v][p] + fc.f[0][0][v][p]; B[v] = Wc.q[v][p + 1] - fc.f[0][0][v][p + 1]; }
#endif
            musta_flux<0>(q, k, mcf, A, B, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) sFx[buf][v][t] = F[v];
        }
        if (ytask) {
            const unsigned int p = yp + pz, pn = p + es1;
            double A[5], B[5], F[5];
#ifdef MF_STRICT
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = fc.f[1][1][v][p]; B[v] = fc.f[1][0][v][pn]; }
#else
#pragma unroll
            for (int v = 0; v < 5; ++v) { A[v] = Wc.q[v][p] + fc.f[1][0][v][p]; B[v] = Wc.q[v][pn] - fc.f[1][0][v][pn]; }
#endif
            musta_flux<1>(q, k, mcf, A, B, F);
#pragma unroll
            for (int v = 0; v < 5; ++v) sFy[buf][v][t] = F[v];
        }
        token = bar.arrive();
    }
    if (CFL) block_reduce_smax<NT>(smax, bad, ds);
}

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
                          StepState* ds, int num_sms, cudaStream_t st)
{
    const int ntx = (g.n[0] + TX - 1) / TX, nty = (g.n[1] + TY - 1) / TY;
    const int TZ = tile_chunk(g, ntx, nty, num_sms);
    const unsigned int grid = (unsigned int)(ntx * nty * ((g.n[2] + TZ - 1) / TZ));
    CState5 Wc;
    for (int v = 0; v < 5; ++v) Wc.q[v] = fc.f[0][1][v];
    if (g.cslot >= 0) {
        if (sg.cfl) k_tile3<true, true><<<grid, NT, 0, st>>>(g, q, k, TZ, ntx, nty, fc, Wc, V, sg, Ua, out, src, ds);
        else k_tile3<false, true><<<grid, NT, 0, st>>>(g, q, k, TZ, ntx, nty, fc, Wc, V, sg, Ua, out, src, ds);
    } else {
        if (sg.cfl) k_tile3<true, false><<<grid, NT, 0, st>>>(g, q, k, TZ, ntx, nty, fc, Wc, V, sg, Ua, out, src, ds);
        else k_tile3<false, false><<<grid, NT, 0, st>>>(g, q, k, TZ, ntx, nty, fc, Wc, V, sg, Ua, out, src, ds);
    }
    return 1;
}

int upload_step_const_tile(const StepConst* dsc, int slot, int nev, cudaStream_t st) { return upload_step_const(dsc, slot, nev, st); }
bool tile_reduces_cfl() { return true; }

} // namespace mf
