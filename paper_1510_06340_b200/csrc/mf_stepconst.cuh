// mf_stepconst.cuh — the per-step scalars in CONSTANT memory, one copy per translation unit that includes this header (a __constant__
// object cannot be shared between separately compiled units without relocatable device code).  k_begin_step writes the scalars of every
// event to a device array; `upload_step_const` copies that array into this unit's c_step (a stream-ordered device-to-device copy, also
// valid inside a graph capture) before the unit's kernels of that step run.  A context owns the slots [g.cslot, g.cslot + g.nev).
#pragma once
#include "mf_types.h"

namespace mf {

static __constant__ StepConst c_step[MF_CSLOTS];

static inline int upload_step_const(const StepConst* dsc, int slot, int nev, cudaStream_t st)
{
    return cudaMemcpyToSymbolAsync(c_step, dsc, sizeof(StepConst) * (size_t)nev, sizeof(StepConst) * (size_t)slot, cudaMemcpyDeviceToDevice, st)
               == cudaSuccess ? 0 : -1;
}

// The step scalars of this block's event (blockIdx.y).  UC: from constant memory (uniform registers / constant-bank operands);
// otherwise from the StepState in global memory (contexts that found no free constant slots, e.g. batches of more than MF_CSLOTS events).
template <bool UC>
__device__ __forceinline__ StepConst step_scalars(const Grid& g, const StepState* ds)
{
    StepConst k;
    if (UC) {
        const StepConst& c = c_step[g.cslot + blockIdx.y];
        k.dt = c.dt; k.lam = c.lam; k.hl = c.hl; k.c_lw = c.c_lw; k.c_lf = c.c_lf; k.nc_lw = c.nc_lw; k.nc2_lf = c.nc2_lf; k.nhlam = c.nhlam;
    } else {
        ds += blockIdx.y;
        k.dt = ds->dt; k.lam = ds->lam; k.hl = ds->hl; k.c_lw = ds->c_lw; k.c_lf = ds->c_lf;
        k.nc_lw = -k.c_lw; k.nc2_lf = -2.0 * k.c_lf; k.nhlam = -0.5 * k.lam;
    }
    return k;
}

__device__ __forceinline__ MustaCoef musta_coef(const StepConst& k)
{
    MustaCoef m;
    m.lam = k.lam; m.c_lw = k.c_lw; m.c_lf = k.c_lf; m.nc_lw = k.nc_lw; m.nc2_lf = k.nc2_lf; m.nhlam = k.nhlam;
    return m;
}

} // namespace mf
