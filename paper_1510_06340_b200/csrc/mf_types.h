// mf_types.h — plain structs shared by the host API (mf_api.cu) and the kernels (mf_kernels.cu).
#pragma once
#include <cuda_runtime.h>
#include "mf_device.cuh"

namespace mf {

// Division of an unsigned 32-bit index by a divisor fixed at mf_create (Granlund-Montgomery round-up multiplier): q = n / d for
// every n < 2^32 in five integer instructions; the general '/' costs ~20 (32-bit) or ~100 (64-bit) on the GPU.
struct FastDiv {
    unsigned int d, mul;
    int sh1, sh2;
};
inline FastDiv make_fastdiv(unsigned int d)
{
    FastDiv f;
    int l = 0;
    while ((1ull << l) < d) ++l;                                   // ceil(log2 d)
    f.d = d;
    f.mul = (unsigned int)(((1ull << 32) * ((1ull << l) - d)) / d + 1);
    f.sh1 = l < 1 ? l : 1;
    f.sh2 = l > 1 ? l - 1 : 0;
    return f;
}

// Grid geometry, passed to kernels by value.
struct Grid {
    int n[3];          // interior extents (x, y, z)
    int h[3];          // 1 on active axes, else 0: the ghost layer the face states are needed on
    int e[3];          // n + 2h: extents of the "extended" layout that holds face states and fluxes
    int act[3];
    int periodic;
    long long ncell;   // n0*n1*n2
    long long next;    // e0*e1*e2
    long long ns[3];   // strides of the interior layout
    long long es[3];   // strides of the extended layout
    double dx;
    double inv_dx;     // 1/dx: the product build multiplies, the strict build divides like the oracle
    int nev;           // events in the batch (mf_create_batch; 1 otherwise): blockIdx.y of every staged kernel is the event, whose cells
                       // sit at offset event*ncell (interior layout) / event*next (extended layout) inside each component array
    FastDiv dv[2][3];  // dv[a][m]: division by n[a] + m, a = x, y, m = 0, 1, 2: every row length an index space of this grid has
    int cslot;         // first of this context's nev slots in the constant-memory copy of the step scalars, or -1: read them from StepState
    int state32;       // 1: the state registers hold single-precision values (mf_set_state_precision, reading A19)
};

// Per-step scalars that live in device memory so that a step never needs the host (A10).
struct StepState {
    double t;                       // simulation time at the start of the current step
    double dt;                      // this step's dt (same in every RK stage, A4)
    double lam;                     // dt/dx
    double hl;                      // 0.5*lam               (Eq.13)
    double c_lw;                    // 0.5*alpha*lam         (Eq.10)
    double c_lf;                    // 0.5/(alpha*lam)       (Eq.11)
    unsigned long long smax_bits;   // atomicMax target: bit image of a non-negative double
    int status;                     // sticky: 1 = bad state seen by a CFL reduction
    int pad;
    long long steps;
};

// The scalars of a step that the hot kernels multiply with, also kept in CONSTANT memory (mf_stepconst.cuh): a constant-bank or
// uniform-register operand is not read from the register file, and a DFMA with three distinct REGISTER operands occupies the FP64 pipe
// for 3 cycles instead of 2 on B200 (measured: mf_probe_fp64, profiles/).  Negated forms are stored so that no operand needs a sign flip.
struct StepConst {
    double dt, lam, hl, c_lw, c_lf;     // as in StepState
    double nc_lw;                       // -c_lw          (Eq.10 on the mean/half-jump form)
    double nc2_lf;                      // -2 c_lf        (Eq.11)
    double nhlam;                       // -lam/2         (Eq.8)
};
constexpr int MF_CSLOTS = 512;          // events (of all live contexts together) whose step scalars fit the constant bank: 32 KB

// stage coefficients straight from the StepState in global memory (kernels without a constant-memory variant)
__device__ __forceinline__ MustaCoef musta_coef_of(const StepState* ds)
{
    MustaCoef m;
    m.lam = ds->lam; m.c_lw = ds->c_lw; m.c_lf = ds->c_lf; m.nc_lw = -m.c_lw; m.nc2_lf = -2.0 * m.c_lf; m.nhlam = -0.5 * m.lam;
    return m;
}

struct Source {
    double dEdx, norm, inv_two_s2, x0, y0, z0;   // S = dEdx*norm*exp(-r^2*inv_two_s2)
    int on;
};

// One conserved state: five component arrays
struct State5 {
    double* q[5];
};
struct CState5 {
    const double* q[5];
};

// Face states of the staged path: [d][side][component] arrays in the extended layout, and interface fluxes [d][component]
struct Faces {
    double* f[3][2][5];
};
struct Fluxes {
    double* f[3][5];
};

// RK stage description (Eq.6 / Eq.7): out = form(Ua, Ub, L + S(t + ts*dt))
struct Stage {
    int form;        // 0: Ua + dt*L   1: 0.5*(Ua + Ub + dt*L)   2: ca*Ua + cb*Ub + (cdt*dt)*L
    double ca, cb, cdt, ts;
    int cfl;         // 1: this is the step's last stage: also reduce S_max / status of the new state for the next step (a2)
};

} // namespace mf
