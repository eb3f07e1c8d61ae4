/*
 * mustaforce.h — C ABI of libmustaforce.so: the per-timestep MUSTA-FORCE update of ideal relativistic
 * hydrodynamics (arXiv 1510.06340) on a 3D Cartesian grid, fp64, hand-written CUDA for sm_100a.
 *
 * What one step computes (citations are PAPER.md lines; readings A1..A19 are listed in DESIGN.md):
 *   conservation system  dU/dt + dF/dx + dG/dy + dH/dz = 0,  U = (E, Mx, My, Mz, R)      Eq.1  :41-49
 *   fluxes               F_d = ((E+p)v_d, M_j v_d + p delta_jd, R v_d)                   Eq.3  :53-59
 *   con2prim             v = M/(E+p(e,n)), e = E - M.v, n = R sqrt(1-v^2)                Eq.23 :221-236
 *   reconstruction       U^{L,R} = U -/+ slope/2, slope = xi(r)(U_i-U_{i-1})             Eq.12, 15-22 :155-211
 *   MUSCL-Hancock        half-step evolution of the face values                          Eq.13 :163-173
 *   MUSTA_k / FORCE      k predictor-corrector stages of 1/2(Lax-Wendroff+Lax-Friedrichs) Eq.8-11 :123-151
 *   time integration     TVD Runge-Kutta 2 / 3                                           Eq.5-7 :84-115
 *   dt                   cfl*dx/S_max, S_max = max (|v|+cs)/(1+|v|cs)  (not in the paper, which uses a fixed dt :264)
 *
 * Conventions
 *   - Every function is extern "C", never throws, never exits.  int results: MF_OK (0) or a negative MF_E* code;
 *     mf_last_error() returns a message for the last failing call on that context.
 *   - HOST arrays are plain host pointers to nx*ny*nz doubles, x fastest: idx = i + nx*(j + ny*k).  The caller
 *     owns them and may free them on return.  Pinned memory makes the copies faster but is not required.
 *   - DEVICE arrays (the *_device calls) are device pointers with the same layout, valid on the context's GPU.
 *   - The context owns all its device memory.  All work of one context is ordered on its stream (its own
 *     non-blocking stream by default, or the one given to mf_set_stream).  mf_step / mf_step_dt return without
 *     waiting for the GPU; every other call that returns data synchronises.  One context is not thread-safe;
 *     distinct contexts are independent.
 *   - There is NO CPU fallback: every entry point that touches data fails with MF_ECUDA if no sm_100 device
 *     (or no CUDA driver) is present.
 *   - MF_ESTATE is sticky: a CFL reduction that met a non-finite cell, or a cell with E > 1e-12 and |M| > E,
 *     raises it on the device; the next synchronising call reports it.  The stored state is never modified by
 *     the admissibility guard (reading A12), so conservation is untouched.
 */
#ifndef MUSTAFORCE_H
#define MUSTAFORCE_H

#ifdef __cplusplus
extern "C" {
#endif

typedef struct mf_ctx mf_ctx;

enum { MF_EOS_CS2 = 0   /* p = cs2*e, default cs2 = 1/3: closed-form con2prim */,
       MF_EOS_TABLE = 1 /* tabulated p(e, n) (Eq.2 :47) with Newton con2prim (Eq.23 :221-236); set with mf_set_eos_table */ };
enum { MF_LIM_NONE = 0      /* Eq.14 central slope            :177 */,
       MF_LIM_MINMOD = 1    /* Minbee, Eq.18                  :201 */,
       MF_LIM_SUPERBEE = 2  /* Eq.19                          :203 */,
       MF_LIM_VANALBADA = 3 /* Eq.20 as printed               :205 */,
       MF_LIM_VANLEER = 4   /* Eq.21                          :207 */,
       MF_LIM_MC = 5        /* monotonized central (BASELINE.json configs 2, 5; not in the paper) */,
       MF_LIM_FIRST = 6     /* zero slope: first-order scheme */ };
enum { MF_BC_OUTFLOW = 0 /* clamp index per axis */, MF_BC_PERIODIC = 1 /* index modulo n per axis */ };
enum { MF_OK = 0, MF_EINVAL = -1, MF_ENOMEM = -2, MF_ECUDA = -3, MF_ESTATE = -4 };
enum { MF_PATH_AUTO = 0   /* fastest path that supports the configuration */,
       MF_PATH_STAGED = 1 /* three kernels per RK stage, face states and fluxes through HBM */,
       MF_PATH_FUSED = 2  /* predictor kernel + one tile kernel per RK stage: face states, fluxes and differences on chip (3D grids) */,
       MF_PATH_HYBRID = 3 /* the staged cell stage + the tile kernel (3D grids) */,
       MF_PATH_SWEEP = 4  /* per-direction sweep kernels that limit the slopes themselves from a +-2-cell halo of the state (:33 "each dimension
                             separately"): no face states in HBM.  Needs an active x axis and MF_EOS_CS2; with the Hancock predictor on also a
                             3D grid and a single event (a predictor kernel then writes the increment of Eq.13 once per cell).  MF_PATH_AUTO
                             takes it whenever the predictor is off. */,
       MF_PATH_SMALL = 5  /* small 1D grids (nx <= 766, ny = nz = 1, MF_EOS_CS2, one event, fp64 state, three state registers): ONE launch of ONE
                             block runs all n steps of an mf_step / mf_step_dt call - S_max and dt by a block reduction at the start of every
                             step, the stages synchronised with __syncthreads, face data and fluxes in shared memory.  Same arithmetic as the
                             staged path.  MF_PATH_AUTO takes it where it applies: such grids are launch bound on every other path. */ };

/* Create a context for an nx*ny*nz grid of spacing dx (same on every axis).  An axis of extent 1 is inactive
 * (ny = nz = 1 is the 1D scheme); an active axis needs extent >= 4; the grid with its boundary layer must have fewer
 * than 2^32 cells (the 400 B/cell of HBM are the tighter limit).  0 <= k_stages <= 8 is the number of Eq.8
 * updates (FORCE is evaluated k_stages+1 times, reading A5).  Defaults: RK2, outflow, cs2 = 1/3, Hancock
 * predictor on, alpha = number of active axes (:151), no source.  Returns NULL on bad arguments, allocation
 * failure or missing GPU (mf_last_error(NULL) tells which). */
mf_ctx* mf_create(int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages);
void    mf_destroy(mf_ctx*);

/* A batch of nevents independent events on identical grids (event-by-event running is what the paper builds the code for, :25, :389;
 * SURVEY.md 8(f) row 4): every kernel launch covers all events, each event keeps its own time and - under mf_step - its own
 * dt = cfl*dx/S_max(event) on the device, so an event of the batch evolves exactly as it would alone in an mf_create context.
 * Every state array of the calls below then holds nevents*nx*ny*nz doubles, event-major: idx = cell + nx*ny*nz*event.  Scheme options
 * (limiter, RK, boundary, EOS, source, ...) are shared by the batch.  1 <= nevents <= 65535, nevents*(cells with boundary layer) < 2^32;
 * runs on the staged path, or on the sweep path when the Hancock predictor is off (MF_PATH_AUTO).  mf_create(...) is mf_create_batch(1, ...). */
mf_ctx* mf_create_batch(int nevents, int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages);
int mf_batch_size(mf_ctx*);                 /* nevents (1 for mf_create) */

/* Copy a conserved state in (5 HOST arrays) and reset t = 0, steps = 0, status = MF_OK.  Synchronous. */
int mf_set_state(mf_ctx*, const double* E, const double* Mx, const double* My, const double* Mz, const double* R);
/* Copy the conserved state out (5 HOST arrays).  Synchronises; returns MF_ESTATE if the sticky flag is up. */
int mf_get_state(mf_ctx*, double* E, double* Mx, double* My, double* Mz, double* R);
/* The same two copies WITHOUT synchronisation, for callers that stream independent events through several contexts (upload the next
 * event and download the last result while the current one is being stepped; event-by-event running is what the paper builds its code for,
 * :25, :389): the copies are enqueued on the context's stream and the call returns.  The HOST arrays must be page-locked (pinned) for the
 * copies to overlap with anything, must stay valid and untouched until the stream has passed them - mf_sync(ctx) or any synchronising call -
 * and the arrays of mf_get_state_async hold the state only after that.  Contexts are independent (one stream each), so set/step/get of
 * one context overlap with those of another.  The sticky state flag is reported by the next synchronising call, not here. */
int mf_set_state_async(mf_ctx*, const double* E, const double* Mx, const double* My, const double* Mz, const double* R);
int mf_get_state_async(mf_ctx*, double* E, double* Mx, double* My, double* Mz, double* R);
/* Same with DEVICE arrays; ordered on the context's stream, set does not synchronise. */
int mf_set_state_device(mf_ctx*, const double* E, const double* Mx, const double* My, const double* Mz, const double* R);
int mf_get_state_device(mf_ctx*, double* E, double* Mx, double* My, double* Mz, double* R);
/* Rest-frame variables (e, vx, vy, vz, n), HOST arrays: Eq.4 (:63-67) on the way in, Eq.23 on the way out. */
int mf_set_state_prim(mf_ctx*, const double* e, const double* vx, const double* vy, const double* vz, const double* n);
int mf_get_state_prim(mf_ctx*, double* e, double* vx, double* vy, double* vz, double* n);

/* Advance n steps.  mf_step: dt = cfl*dx/S_max recomputed on the device from U^n at every step, no host
 * round trip (reading A10).  mf_step_dt: the paper's fixed dt (Tables 1-3).  Asynchronous. */
int mf_step(mf_ctx*, int n, double cfl);
int mf_step_dt(mf_ctx*, int n, double dt);

/* out[q] = dx^D * sum over cells of (E, Mx, My, Mz, R), D = number of active axes; over all events of a batch, or over one.
 * Synchronises. */
int mf_conserved_totals(mf_ctx*, double out[5]);
int mf_conserved_totals_event(mf_ctx*, int event, double out[5]);
/* Simulation time, last dt used, steps taken since mf_set_state (of event 0 / of the given event: under mf_step the events of a
 * batch run on their own clocks).  Any pointer may be NULL.  Synchronises. */
int mf_get_time(mf_ctx*, double* t, double* last_dt, long long* steps);
int mf_get_time_event(mf_ctx*, int event, double* t, double* last_dt, long long* steps);
/* S_max of the stored state (runs the CFL reduction); the largest over the events of a batch.  Synchronises. */
int mf_max_signal_speed(mf_ctx*, double* smax);

int mf_set_rk(mf_ctx*, int order);          /* 2 (Eq.6, default) or 3 (Eq.7) */
int mf_set_boundary(mf_ctx*, int bc);       /* MF_BC_OUTFLOW (default) or MF_BC_PERIODIC */
int mf_set_cs2(mf_ctx*, double cs2);        /* 0 < cs2 < 1, default 1/3 */
/* Tabulated equation of state for a context created with MF_EOS_TABLE (until it is set the context uses p = cs2*e).  ln_p is a HOST
 * array of nn rows of ne values (e fastest): ln p at e = exp(ln_e0 + i*dln_e), n = n0 + j*dn.  Lookup: bilinear in (ln e, n) of ln p;
 * the end cells extrapolate linearly in ln e, outside the n range the value is held; nn = 1: no n dependence.  con2prim then solves
 * v (E + p(E - |M|v, R sqrt(1-v^2))) = |M| for the speed by safeguarded Newton (reading A18), and the CFL reduction uses the
 * table's adiabatic sound speed.  The table is copied to the device; the call synchronises. */
int mf_set_eos_table(mf_ctx*, int ne, int nn, double ln_e0, double dln_e, double n0, double dn, const double* ln_p);
int mf_set_predictor(mf_ctx*, int on);      /* Eq.13 half step on (default, paper-literal) or off (MUSCL + RK) */
int mf_set_alpha(mf_ctx*, double alpha);    /* FORCE alpha, default = number of active axes (:151) */
/* Moving Gaussian energy-momentum source S_E = S_Mx = dEdx * G_sigma(x - (x0+t, y0, z0)) added to L in every RK
 * stage at the stage time (reading A14; not in the paper).  dEdx = 0 disables it. */
int mf_set_jet_source(mf_ctx*, double dEdx, double sigma, double x0, double y0, double z0);
int mf_set_path(mf_ctx*, int path);         /* MF_PATH_*; MF_EINVAL if that path cannot run this configuration */
int mf_get_path(mf_ctx*, int* path);        /* the path mf_step will actually take */
/* Low-storage Runge-Kutta (:117 "a low storage version of the third order method can be used"; the paper prints no formula): the same
 * Eq.6 / Eq.7 arithmetic with two state registers instead of three - every stage after the first replaces the work register in place, so
 * the results are bit-identical to the three-register form.  Frees (on = 1) or re-allocates (on = 0) the third register; synchronises.
 * Staged path only (MF_PATH_AUTO then resolves to it); MF_EINVAL if another path is selected. */
int mf_set_low_storage(mf_ctx*, int on);
/* Single-precision STATE ("The state of the system is saved as 5 single precision floating-point numbers
 * per lattice cell"; reading A19): bits = 32 makes every STORED state value a float - the state handed in and the result of every Runge-Kutta
 * stage are rounded to nearest even on the store - while all arithmetic between a load and the next store, the scratch (face states, fluxes)
 * and the CFL reduction (taken from the stored, rounded U^n) stay fp64.  Halves the bytes of the state registers that cross HBM.  The calls
 * that hand states in or out keep their double arrays (values are rounded on the way in and widened on the way out).  bits = 64 (default)
 * restores the fp64 state.  The current state is converted; synchronises.  Runs on the staged path and, without the Hancock predictor, on
 * the sweep path (MF_PATH_AUTO resolves accordingly); MF_EINVAL for another bit count or if a path that cannot carry it is selected.  Outside BASELINE.json's fp64 contract: bench.py reports it beside the headline, never as it. */
int mf_set_state_precision(mf_ctx*, int bits);
int mf_get_state_precision(mf_ctx*, int* bits);
/* mf_step / mf_step_dt replay whole steps from a CUDA graph when n >= 7 (5 in low-storage mode): one eager step, then one captured period of
 * the register rotation (3 steps, or 2) launched repeatedly, the remainder eagerly.  The launches and their arguments are exactly the eager
 * ones (every per-step scalar lives in device memory), so results are bit-identical; it removes the per-launch host cost that dominates
 * small grids.  On by default; off while mf_profile is recording.  mf_set_graph(ctx, 0) forces eager launches. */
int mf_set_graph(mf_ctx*, int on);
/* Diagnostic: how many times this context captured a graph and how many times it launched one (either pointer may be NULL).  Repeated
 * mf_step(n) calls with the same cfl (or dt) and options reuse one capture whatever n is. */
int mf_graph_stats(mf_ctx*, long long* captures, long long* replays);
/* Device memory currently held by the context (state registers, scratch allocated so far, tables), in bytes. */
int mf_memory_bytes(mf_ctx*, long long* bytes);
/* Run on a caller-owned CUDA stream (a cudaStream_t passed as void*), e.g. PyTorch's current stream, so the
 * caller's events bracket the kernels.  NULL restores the context's own stream. */
int mf_set_stream(mf_ctx*, void* cuda_stream);

int mf_sync(mf_ctx*);                       /* wait for the stream; returns the sticky status */
const char* mf_last_error(mf_ctx*);         /* ctx may be NULL: message of the last failed mf_create */

/* L(U) of the stored state for a given dt, 5 HOST arrays (diagnostic: lets a test compare the spatial operator alone). */
int mf_eval_L(mf_ctx*, double dt, double* L_E, double* L_Mx, double* L_My, double* L_Mz, double* L_R);
/* Number of kernel launches issued by this context since creation (for bench.py's gpu_launches). */
int mf_launch_count(mf_ctx*, long long* launches);
/* Per-kernel-class device timing with CUDA events recorded on the context's stream around every launch of a class
 * (at most 8192 launches are kept between reads).  mf_profile(ctx, 1) starts recording, mf_profile(ctx, 0) stops.
 * mf_profile_read synchronises, writes the summed milliseconds and launch counts per class since the last read and
 * clears them.  Classes: 0 CFL reduction, 1 cell stage (a3+a4), 2 interface flux stage (a5+a6), 3 combine (a7+a8),
 * 4 fused stage (a1,a3-a8 in one kernel), 5 per-step scalar kernels, 6-7 unused. */
enum { MF_NCLASS = 8 };
int mf_profile(mf_ctx*, int on);
int mf_profile_read(mf_ctx*, double ms[MF_NCLASS], long long launches[MF_NCLASS]);

/* DIAGNOSTIC, not part of the hot path (bench.py calls it for the roofline denominators; MEASURED_PEAKS.json has no FP64 entry).
 * Measured FP64-pipe issue rates of the current device: runs register-only loops of dependent-chain-free DFMA, DADD, DMUL,
 * reciprocal and square root and writes instructions (or results) per second:
 * out = { dfma/s with two register operands (x*a+a), dadd/s, dmul/s, rcp results/s, sqrt results/s, SM clock estimate in Hz, SM count,
 *         dfma/s with three distinct register operands (x = y*z + x; the register file delivers them in 3 cycles instead of 2) }. */
int mf_probe_fp64(double out[8]);
/* Conserved totals WITHOUT any allocation, for callers that cannot call cudaMalloc (code under CUDA-graph capture, tight serving loops,
 * harnesses that forbid it): out5[q] = scale * sum over ncells cells of (E, Mx, My, Mz, R)[q] (Eq.1's conserved quantities, :41-49; pass
 * scale = dx^D for mf_conserved_totals' convention).  The five inputs and out5 (5 doubles) are DEVICE pointers owned by the caller; no
 * context is needed.  The per-block partial sums that mf_conserved_totals keeps in a cudaMalloc'ed buffer live in a file-scope
 * __device__ array of 40 KB that every GPU that loads the library holds until exit; ncells <= MF_STATIC_MAX_CELLS (2^24 = 256^3),
 * larger sizes return MF_EINVAL (mf_static_last_error() says why).  Two kernel launches on cuda_stream (a cudaStream_t as void*, NULL =
 * the default stream), asynchronous, no cudaMalloc/cudaFree, deterministic summation order.  Every call shares the array, which keeps
 * the last call's contents (a call overwrites every slot it reads, so nothing has to be cleared): calls that OVERLAP on the GPU -
 * different streams, several host threads on one device - race on it; serialise them. */
#define MF_STATIC_MAX_CELLS (1LL << 24)
int mf_totals_static(const double* E, const double* Mx, const double* My, const double* Mz, const double* R, long long ncells, double scale,
                     double* out5, void* cuda_stream);
const char* mf_static_last_error(void);     /* message of the calling thread's last failed mf_totals_static */

/* Library build info: "mustaforce <version> sm_100a [strict]" */
const char* mf_version(void);

#ifdef __cplusplus
}
#endif
#endif
