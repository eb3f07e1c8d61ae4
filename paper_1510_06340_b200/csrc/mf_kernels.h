// mf_kernels.h — launch wrappers of the CUDA kernels (defined in mf_kernels.cu, mf_fused.cu, mf_probe.cu).
// Each wrapper enqueues on `st` and returns the number of kernel launches it issued.
#pragma once
#include "mf_types.h"

#include <atomic>

namespace mf {

// "once per DEVICE" for function attributes (cudaFuncSetAttribute applies to the current device only): first() is true the first time it is
// called with a given device current, in any thread.
struct DeviceOnce {
    std::atomic<unsigned long long> done[4];      // one bit per device ordinal, 256 devices
    DeviceOnce() { for (auto& d : done) d.store(0ull); }
    bool first()
    {
        int dev = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 256) return true;
        const unsigned long long bit = 1ull << (dev & 63);
        return (done[dev >> 6].fetch_or(bit) & bit) == 0;
    }
};

// a2: CFL reduction of `U` into ds->smax_bits / ds->status (accumulator must have been reset by begin_step of the previous step or by reset_smax)
int launch_cfl(const Grid& g, const Eos& q, CState5 U, StepState* ds, int num_sms, cudaStream_t st);
// per-step scalars on the device: mode 0: dt = value*dx/smax (cfl), mode 1: dt = value (fixed); resets the smax accumulator
int launch_begin_step(StepState* ds, StepConst* dsc, int nev, int mode, double value, double dx, double alpha, cudaStream_t st);   // ds, dsc: one per event
// copy dsc[0..nev) into the constant-memory step scalars of the translation unit that holds the staged kernels (mf_stepconst.cuh); 0 = ok
int upload_step_const_staged(const StepConst* dsc, int slot, int nev, cudaStream_t st);
int launch_end_step(StepState* ds, int nev, cudaStream_t st);
int launch_reset(StepState* ds, int nev, cudaStream_t st);

// ---- staged path (MF_PATH_STAGED): a3+a4, a5, a7(+a8) as three kernels, face states and fluxes through HBM
int launch_cell_stage(const Grid& g, const Eos& q, int limiter, int predictor, CState5 V, Faces fc, const StepState* ds, cudaStream_t st);
int launch_flux_stage(const Grid& g, const Eos& q, int k, int dmask /* bit d: compute direction d */, Faces fc, Fluxes fx, const StepState* ds, cudaStream_t st);
int launch_combine(const Grid& g, const Eos& q, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out, Source src, StepState* ds, cudaStream_t st);   // sg.cfl: + a2

// x fluxes fused with divergence + source + RK combine (+ a2 when sg.cfl); F_y, F_z must already be in fx (needs an active x axis)
int launch_xflux_combine(const Grid& g, const Eos& q, int k, Faces fc, Fluxes fx, Stage sg, CState5 Ua, CState5 Ub, State5 out, Source src,
                         StepState* ds, cudaStream_t st);

// ---- fused path (MF_PATH_FUSED): one kernel per RK stage
bool fused_supported(const Grid& g);
int launch_delta_stage(const Grid& g, const Eos& q, int limiter, CState5 V, State5 D, const StepState* ds, cudaStream_t st);
int launch_fused_stage(const Grid& g, const Eos& q, int limiter, int predictor, int k, CState5 V, CState5 D, Stage sg, CState5 Ua,
                       State5 out, Source src, const StepState* ds, int num_sms, int variant, cudaStream_t st);

int launch_tile_stage(const Grid& g, const Eos& q, int limiter, int predictor, int k, CState5 V, CState5 D, Stage sg, CState5 Ua, State5 out,
                      Source src, const StepState* ds, int num_sms, cudaStream_t st);

// hybrid path: W and the half slopes from launch_cell_stage's scratch; all three flux directions, divergence, source, RK combine and (sg.cfl)
// the CFL reduction of the new state in one kernel
int launch_tile_stage_pre(const Grid& g, const Eos& q, int k, Faces fc, CState5 V, Stage sg, CState5 Ua, State5 out, Source src,
                          StepState* ds, int num_sms, cudaStream_t st);
int upload_step_const_tile(const StepConst* dsc, int slot, int nev, cudaStream_t st);   // the tile unit's constant-memory step scalars; 0 = ok
bool tile_reduces_cfl();

// ---- small 1D grids (MF_PATH_SMALL, mf_small.cu): all n steps of a call in ONE launch of ONE block (S_max, dt, RK stages, clock on the device)
bool small_supported(const Grid& g, int eos_kind);
int launch_small_steps(const Grid& g, const Eos& q, int limiter, int predictor, int k, int rk, double alpha, int mode, double value, int nsteps,
                       int cur, double* const U[3], Source src, StepState* ds, cudaStream_t st);

// ---- sweep path (MF_PATH_SWEEP, mf_sweep.cu): per-direction sweeps that limit the slopes themselves from a +-2-cell halo of V; with pred the
// Hancock increment Dl (extended layout, from launch_delta_stage) is added to both face states.  F_y, F_z go to fx, the x sweep finishes the cells.
bool sweep_supported(const Grid& g, int eos_kind, int predictor);
int launch_sweep_flux(const Grid& g, const Eos& q, int limiter, int k, bool pred, CState5 V, CState5 Dl, Fluxes fx, const StepState* ds, cudaStream_t st);
int launch_sweep_xcombine(const Grid& g, const Eos& q, int limiter, int k, bool pred, CState5 V, CState5 Dl, Fluxes fx, Stage sg, CState5 Ua, State5 out,
                          Source src, StepState* ds, cudaStream_t st);

// ---- conversions and reductions
int launch_prim2con(const Grid& g, const Eos& q, State5 U, cudaStream_t st);          // in place: (e,v,n) -> (E,M,R), Eq.4
int launch_con2prim(const Grid& g, const Eos& q, CState5 U, State5 P, cudaStream_t st); // Eq.23
int launch_totals(const Grid& g, CState5 U, double* partials /* 5*nblocks */, int nblocks, cudaStream_t st);
// reading A19: copy a state of n elements per component from double to float (to_f32, round to nearest even) or from float to double;
// the component pointers of src and dst are spaced for their own element type
int launch_state_convert(long long n, int to_f32, CState5 src, State5 dst, int num_sms, cudaStream_t st);

// ---- FP64 pipe micro-benchmarks (mf_probe_fp64; diagnostic, not on the hot path)
int probe_fp64(double out[8]);

} // namespace mf
