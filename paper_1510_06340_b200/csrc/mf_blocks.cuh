// mf_blocks.cuh — block-level device helpers shared by the staged (mf_kernels.cu) and sweep (mf_sweep.cu) kernels.
#pragma once
#include "mf_types.h"

namespace mf {

constexpr int TPB = 256;                  // threads per block of every staged / sweep kernel

// a2 (reading A10), block part of the CFL reduction:
// warp shuffle max, then one value per warp through shared memory, then ONE atomic per block; every thread of the block must call it
template <int NT = TPB>                   // NT: threads per block
__device__ __forceinline__ void block_reduce_smax(double smax, int bad, StepState* ds)
{
#pragma unroll
    for (int off = 16; off > 0; off >>= 1) {
        smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, off));
        bad |= __shfl_xor_sync(0xffffffffu, bad, off);
    }
    __shared__ double s_max[NT / 32];
    __shared__ int s_bad[NT / 32];
    const int tid = threadIdx.y * blockDim.x + threadIdx.x;          // NT threads per block, whatever its shape
    const int lane = tid & 31, warp = tid >> 5;
    if (lane == 0) { s_max[warp] = smax; s_bad[warp] = bad; }
    __syncthreads();
    if (warp == 0) {
        smax = lane < NT / 32 ? s_max[lane] : 0.0;
        bad = lane < NT / 32 ? s_bad[lane] : 0;
#pragma unroll
        for (int off = 4; off > 0; off >>= 1) {
            smax = fmax(smax, __shfl_xor_sync(0xffffffffu, smax, off));
            bad |= __shfl_xor_sync(0xffffffffu, bad, off);
        }
        if (lane == 0) {
            atomicMax(&ds->smax_bits, (unsigned long long)__double_as_longlong(smax));   // smax >= 0: bit order == value order
            if (bad) atomicOr(&ds->status, 1);
        }
    }
}

// a8 (reading A14): the moving Gaussian source at cell (i, j, k) and time t
__device__ __forceinline__ double jet_source(const Grid& g, const Source& s, int i, int j, int k, double t)
{
    double x = (i + 0.5 - g.n[0] / 2.0) * g.dx - (s.x0 + t);
    double y = (j + 0.5 - g.n[1] / 2.0) * g.dx - s.y0;
    double z = (k + 0.5 - g.n[2] / 2.0) * g.dx - s.z0;
    double r2 = x * x + y * y + z * z;
    double arg = -r2 * s.inv_two_s2;
#ifndef MF_STRICT
    // Product build: beyond 14 sigma the source is below e^-100 = 4e-44 of its peak - 30 orders of magnitude under the parity bar relative to any
    // state it could be added to - and exp() costs ~40 FP64 instructions per cell and stage, so it is taken as zero there.  (The strict build
    // evaluates it everywhere, like the oracle.)
    if (arg < -100.0) return 0.0;
#endif
    return s.dEdx * s.norm * exp(arg);
}

__device__ __forceinline__ double rk_form(const Stage& sg, double ua, double ub, double dt, double L)
{
    if (sg.form == 0) return ua + dt * L;                          // U + dt L            (Eq.6/7 first line)
    if (sg.form == 1) return 0.5 * (ua + ub + dt * L);             // Eq.6 second line :105
    if (sg.form == 2) return sg.ca * ua + sg.cb * ub + (sg.cdt * dt) * L;   // Eq.7 lines 2, 3 :112-114
    return L;                                                      // form 3: L itself (mf_eval_L)
}

} // namespace mf
