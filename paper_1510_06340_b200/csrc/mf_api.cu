// mf_api.cu — the C ABI declared in include/mustaforce.h: context, device buffers, the RK stage driver.
// Host logic only; every arithmetic step of the path runs in the kernels (mf_kernels.cu / mf_fused.cu).
#include "../../include/mustaforce.h"
#include "mf_kernels.h"

#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <string>
#include <vector>

using namespace mf;

#ifdef MF_STRICT
#define MF_VERSION_STR "mustaforce 0.1 sm_100a strict"
#else
#define MF_VERSION_STR "mustaforce 0.1 sm_100a"
#endif

struct mf_ctx {
    Grid g;
    Eos q;
    int limiter, k, rk, predictor, nact;
    double alpha;
    Source src;
    int path_req, path;
    int dev, num_sms;
    cudaStream_t own_stream, stream;
    int nev;                 // events in the batch (1 unless mf_create_batch)
    long long nst, nxt;      // nev*ncell, nev*next: the length of one component array in the interior / extended layout
    double* U[3];            // three state registers, 5*nst doubles each (U^n, U_(1), U_(2)), component-major, [component][event][cell]
    int nreg;                // 3, or 2 in low-storage mode (mf_set_low_storage): U[2] is then not allocated
    int cur;                 // which register holds U^n
    double* faces;           // staged path: 2*5*nact*next doubles
    double* fluxes;          // staged path: 5*nact*next doubles
    double* delta;           // fused path: Hancock increment, 5*next doubles
    int eos;                 // MF_EOS_*
    double* table;           // tabulated EOS: ln p, device copy
    int smax_valid;          // the device-side S_max accumulator already holds the reduction of the current U^n (fused into the last combine)
    StepState* ds;           // one per event
    StepConst* dsc;          // the step's multipliers per event: source of the constant-memory copy (mf_stepconst.cuh)
    StepState* h_ds;         // pinned mirror
    double* partials;        // totals: 5*nblocks doubles
    double* h_partials;
    int nblocks_tot;
    long long launches;
    std::string err;
    // per-class CUDA-event timing (mf_profile)
    // CUDA-graph replay of whole steps (launch-bound grids): one captured period of the register rotation, keyed by what is baked into it
    int graph_on;                          // mf_set_graph
    unsigned long long epoch;              // bumped by every call that changes what a captured step would launch
    cudaGraphExec_t graph_exec;
    unsigned long long graph_epoch;
    int graph_cur, graph_mode, graph_steps;
    double graph_value;
    long long graph_launches;
    long long graph_captures, graph_replays;   // diagnostics (mf_graph_stats)
    int prof_on;
    std::vector<cudaEvent_t> prof_ev;     // pairs: [2i] start, [2i+1] stop
    std::vector<int> prof_cls;            // class of pair i
    size_t prof_used;
};

namespace {

thread_local std::string g_create_err;

// Constant-memory slots for the step scalars (MF_CSLOTS events over all live contexts): first fit over a bitmap; -1 when nothing fits,
// the context then reads the scalars from global memory.
std::mutex g_slot_mutex;
bool g_slot_used[MF_CSLOTS];
int slots_acquire(int n)
{
    if (n > MF_CSLOTS) return -1;
    std::lock_guard<std::mutex> lock(g_slot_mutex);
    for (int b = 0; b + n <= MF_CSLOTS; ++b) {
        int i = 0;
        while (i < n && !g_slot_used[b + i]) ++i;
        if (i == n) { for (i = 0; i < n; ++i) g_slot_used[b + i] = true; return b; }
        b += i;
    }
    return -1;
}
void slots_release(int b, int n)
{
    if (b < 0) return;
    std::lock_guard<std::mutex> lock(g_slot_mutex);
    for (int i = 0; i < n; ++i) g_slot_used[b + i] = false;
}

int fail(mf_ctx* c, int code, const std::string& msg) { if (c) c->err = msg; else g_create_err = msg; return code; }

int cuda_fail(mf_ctx* c, cudaError_t e, const char* what)
{
    return fail(c, MF_ECUDA, std::string(what) + ": " + cudaGetErrorString(e));
}

#define MF_CUDA(c, call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail((c), e_, #call); } while (0)

CState5 cstate(const double* base, long long n) { CState5 s; for (int v = 0; v < 5; ++v) s.q[v] = base + v * n; return s; }
State5 state(double* base, long long n) { State5 s; for (int v = 0; v < 5; ++v) s.q[v] = base + v * n; return s; }

// Component pointers of a STATE REGISTER: nst elements per component of the context's state element type (double, or float in 32-bit state
// mode, reading A19).  The structs carry double pointers either way; the kernels of the staged path cast them back (ld_state / st_state).
CState5 creg_as(const mf_ctx* c, const double* base, bool f32, long long first = 0)
{
    CState5 s;
    for (int v = 0; v < 5; ++v)
        s.q[v] = f32 ? reinterpret_cast<const double*>(reinterpret_cast<const float*>(base) + v * c->nst + first) : base + v * c->nst + first;
    return s;
}
State5 reg_as(const mf_ctx* c, double* base, bool f32)
{
    State5 s;
    for (int v = 0; v < 5; ++v) s.q[v] = f32 ? reinterpret_cast<double*>(reinterpret_cast<float*>(base) + v * c->nst) : base + v * c->nst;
    return s;
}
CState5 creg(const mf_ctx* c, const double* base, long long first = 0) { return creg_as(c, base, c->g.state32 != 0, first); }
State5 reg(const mf_ctx* c, double* base) { return reg_as(c, base, c->g.state32 != 0); }

Faces faces_of(mf_ctx* c)
{
    Faces f; memset(&f, 0, sizeof(f));
    long long slot = 0;
    for (int d = 0; d < 3; ++d) {
        if (!c->g.act[d]) continue;
        for (int s = 0; s < 2; ++s) for (int v = 0; v < 5; ++v) f.f[d][s][v] = c->faces + (slot++) * c->nxt;
    }
    return f;
}

Fluxes fluxes_of(mf_ctx* c)
{
    Fluxes f; memset(&f, 0, sizeof(f));
    long long slot = 0;
    for (int d = 0; d < 3; ++d) {
        if (!c->g.act[d]) continue;
        for (int v = 0; v < 5; ++v) f.f[d][v] = c->fluxes + (slot++) * c->nxt;
    }
    return f;
}

void set_eos(Eos& q, double cs2)
{
    q.cs2 = cs2;
    q.c1 = 1.0 + cs2;
    q.c1sq = q.c1 * q.c1;
    q.four_cs2 = 4.0 * cs2;
    q.cs = std::sqrt(cs2);
    q.qc1sq = 0.25 * q.c1sq;
    q.hc1 = 0.5 * q.c1;
    q.vcap2 = V_CAP * V_CAP;
}

void clear_table(Eos& q)
{
    q.kind = 0; q.ne = q.nn = 0; q.pad = 0; q.ln_e0 = q.dln_e = q.n0 = q.dn = 0.0; q.lnp = nullptr;
    q.inv_dln_e = q.inv_dn = 0.0; q.lnpf = nullptr;
}

int resolve_path(mf_ctx* c)
{
    if (c->g.state32) {
        // single-precision state: the kernels of the staged path and, without the Hancock step, of the sweep path carry the state element
        // type (k_delta_stage and the tile kernels read doubles)
        const bool sweep_ok = !c->predictor && c->nreg == 3 && sweep_supported(c->g, c->q.kind || c->eos != MF_EOS_CS2, 0);
        if (c->path_req == MF_PATH_SWEEP) { if (!sweep_ok) return MF_EINVAL; c->path = MF_PATH_SWEEP; return MF_OK; }
        if (c->path_req != MF_PATH_AUTO && c->path_req != MF_PATH_STAGED) return MF_EINVAL;
        c->path = (c->path_req == MF_PATH_AUTO && sweep_ok) ? MF_PATH_SWEEP : MF_PATH_STAGED;
        return MF_OK;
    }
    if (c->nreg == 2) {
        // low storage: an RK stage writes its result over the register it read, which only the staged path's last kernel allows (it touches
        // the state at the thread's own cell only; the sweep and tile kernels read neighbours of the state they are replacing)
        if (c->path_req != MF_PATH_AUTO && c->path_req != MF_PATH_STAGED) return MF_EINVAL;
        c->path = MF_PATH_STAGED;
        return MF_OK;
    }
    if (c->path_req == MF_PATH_FUSED || c->path_req == MF_PATH_HYBRID) {
        if (!fused_supported(c->g) || c->eos != MF_EOS_CS2 || c->nev > 1) return MF_EINVAL;      // the tile kernel is built for p = cs2*e and three active axes
        c->path = c->path_req;
    }
    else if (c->path_req == MF_PATH_SWEEP) {
        if (!sweep_supported(c->g, c->q.kind || c->eos != MF_EOS_CS2, c->predictor)) return MF_EINVAL;
        c->path = MF_PATH_SWEEP;
    }
    else if (c->path_req == MF_PATH_SMALL) {
        if (!small_supported(c->g, c->q.kind || c->eos != MF_EOS_CS2)) return MF_EINVAL;
        c->path = MF_PATH_SMALL;
    }
    else if (c->path_req == MF_PATH_STAGED) c->path = MF_PATH_STAGED;
    else if (small_supported(c->g, c->q.kind || c->eos != MF_EOS_CS2)) c->path = MF_PATH_SMALL;      // AUTO: launch-bound grids
    else {
        // AUTO.  Predictor on: the staged path measured faster than the fused path on B200 (profiles/).  Predictor off: the sweep kernels
        // need no cell stage and no face-state scratch.
        c->path = (!c->predictor && sweep_supported(c->g, c->q.kind || c->eos != MF_EOS_CS2, 0)) ? MF_PATH_SWEEP : MF_PATH_STAGED;
    }
    return MF_OK;
}

// RAII-free scope: record an event pair around the launches of one kernel class when profiling is on
constexpr size_t PROF_MAX = 8192;
int prof_begin(mf_ctx* c, int cls)
{
    if (!c->prof_on || c->prof_used >= PROF_MAX) return -1;
    size_t i = c->prof_used;
    if (c->prof_ev.size() < 2 * (i + 1)) {
        cudaEvent_t a, b;
        if (cudaEventCreate(&a) != cudaSuccess || cudaEventCreate(&b) != cudaSuccess) { cudaGetLastError(); return -1; }
        c->prof_ev.push_back(a); c->prof_ev.push_back(b); c->prof_cls.push_back(cls);
    }
    c->prof_cls[i] = cls;
    cudaEventRecord(c->prof_ev[2 * i], c->stream);
    return (int)i;
}
void prof_end(mf_ctx* c, int slot)
{
    if (slot < 0) return;
    cudaEventRecord(c->prof_ev[2 * slot + 1], c->stream);
    c->prof_used = (size_t)slot + 1;
}

// scratch is allocated on first use, so that a path only pays for what it needs (fused: delta; sweep: fluxes (+ delta); staged: faces + fluxes)
int ensure_flux_buffer(mf_ctx* c)
{
    if (c->fluxes) return MF_OK;
    size_t nx = (size_t)5 * c->nact * c->nxt;
    if (cudaMalloc(&c->fluxes, nx * sizeof(double)) != cudaSuccess) { cudaGetLastError(); c->fluxes = nullptr; return fail(c, MF_ENOMEM, "cudaMalloc(fluxes) failed"); }
    return MF_OK;
}

int ensure_delta_buffer(mf_ctx* c)
{
    if (c->delta) return MF_OK;
    if (cudaMalloc(&c->delta, sizeof(double) * 5 * c->g.next) != cudaSuccess) { cudaGetLastError(); c->delta = nullptr; return fail(c, MF_ENOMEM, "cudaMalloc(delta) failed"); }
    return MF_OK;
}

int ensure_staged_buffers(mf_ctx* c)
{
    int rc = ensure_flux_buffer(c);
    if (rc != MF_OK || c->faces) return rc;
    size_t nf = (size_t)10 * c->nact * c->nxt;
    if (cudaMalloc(&c->faces, nf * sizeof(double)) != cudaSuccess) { cudaGetLastError(); c->faces = nullptr; return fail(c, MF_ENOMEM, "cudaMalloc(face states) failed"); }
    return MF_OK;
}

// One evaluation of  out = form(Ua, V, L(V) + S)  on the selected path.
int run_stage(mf_ctx* c, const double* V, const Stage& sg, const double* Ua, double* out)
{
    const long long n = c->nst;
    if (c->path == MF_PATH_FUSED || c->path == MF_PATH_HYBRID) {
        if (c->path == MF_PATH_HYBRID) {                           // the staged path's cell stage + the tile kernel
            int rc = ensure_staged_buffers(c);
            if (rc != MF_OK) return rc;
            Faces fc = faces_of(c);
            int ps = prof_begin(c, 1);
            c->launches += launch_cell_stage(c->g, c->q, c->limiter, c->predictor, cstate(V, n), fc, c->ds, c->stream);
            prof_end(c, ps);
            ps = prof_begin(c, 4);
            c->launches += launch_tile_stage_pre(c->g, c->q, c->k, fc, cstate(V, n), sg, cstate(Ua, n), state(out, n), c->src, c->ds, c->num_sms, c->stream);
            prof_end(c, ps);
            return MF_OK;
        }
        int rc = ensure_delta_buffer(c);
        if (rc != MF_OK) return rc;
        int ps;
        if (c->predictor) {
            ps = prof_begin(c, 1);
            c->launches += launch_delta_stage(c->g, c->q, c->limiter, cstate(V, n), state(c->delta, c->g.next), c->ds, c->stream);
            prof_end(c, ps);
        }
        ps = prof_begin(c, 4);
        c->launches += launch_fused_stage(c->g, c->q, c->limiter, c->predictor, c->k, cstate(V, n), cstate(c->delta, c->g.next), sg, cstate(Ua, n),
                                          state(out, n), c->src, c->ds, c->num_sms, 0, c->stream);
        prof_end(c, ps);
    } else if (c->path == MF_PATH_SWEEP) {
        if (!sweep_supported(c->g, c->q.kind, c->predictor)) return fail(c, MF_EINVAL, "the sweep path does not support this configuration");
        int rc = ensure_flux_buffer(c);
        if (rc == MF_OK && c->predictor) rc = ensure_delta_buffer(c);
        if (rc != MF_OK) return rc;
        Fluxes fx = fluxes_of(c);
        const bool pred = c->predictor != 0;
        const CState5 Vs = creg(c, V), Uas = creg(c, Ua);
        const State5 outs = sg.form == 3 ? state(out, n) : reg(c, out);
        CState5 Dl = pred ? cstate(c->delta, c->g.next) : Vs;
        int ps;
        if (pred) {
            ps = prof_begin(c, 1);
            c->launches += launch_delta_stage(c->g, c->q, c->limiter, cstate(V, n), state(c->delta, c->g.next), c->ds, c->stream);
            prof_end(c, ps);
        }
        if (c->g.act[1] || c->g.act[2]) {
            ps = prof_begin(c, 2);
            c->launches += launch_sweep_flux(c->g, c->q, c->limiter, c->k, pred, Vs, Dl, fx, c->ds, c->stream);
            prof_end(c, ps);
        }
        ps = prof_begin(c, 3);
        c->launches += launch_sweep_xcombine(c->g, c->q, c->limiter, c->k, pred, Vs, Dl, fx, sg, Uas, outs, c->src, c->ds, c->stream);
        prof_end(c, ps);
    } else {
        int rc = ensure_staged_buffers(c);
        if (rc != MF_OK) return rc;
        Faces fc = faces_of(c);
        Fluxes fx = fluxes_of(c);
        // state registers in the context's state element type (reading A19); the result of form 3 (mf_eval_L) is L itself, always double
        const CState5 Vs = creg(c, V), Uas = creg(c, Ua);
        const State5 outs = sg.form == 3 ? state(out, n) : reg(c, out);
        int ps = prof_begin(c, 1);
        c->launches += launch_cell_stage(c->g, c->q, c->limiter, c->predictor, Vs, fc, c->ds, c->stream);
        prof_end(c, ps);
        if (c->g.act[0]) {
            // y and z fluxes to HBM, then the x fluxes fused with divergence + source + RK combine (F_x stays on chip)
            ps = prof_begin(c, 2);
            c->launches += launch_flux_stage(c->g, c->q, c->k, 6, fc, fx, c->ds, c->stream);
            prof_end(c, ps);
            ps = prof_begin(c, 3);
            c->launches += launch_xflux_combine(c->g, c->q, c->k, fc, fx, sg, Uas, Vs, outs, c->src, c->ds, c->stream);
            prof_end(c, ps);
        } else {
            ps = prof_begin(c, 2);
            c->launches += launch_flux_stage(c->g, c->q, c->k, 7, fc, fx, c->ds, c->stream);
            prof_end(c, ps);
            ps = prof_begin(c, 3);
            c->launches += launch_combine(c->g, c->q, fx, sg, Uas, Vs, outs, c->src, c->ds, c->stream);
            prof_end(c, ps);
        }
    }
    return MF_OK;
}

// does the last kernel of a step also reduce S_max of the new state (a2) for the next step's dt?
bool last_stage_reduces_cfl(const mf_ctx* c)
{
    return c->path == MF_PATH_STAGED || c->path == MF_PATH_SWEEP || (c->path == MF_PATH_HYBRID && tile_reduces_cfl());
}

// RK2 (Eq.6 :103-105) / RK3 (Eq.7 :110-114); per-step scalars are already in c->ds.
int run_step(mf_ctx* c)
{
    double* Un = c->U[c->cur];
    int rc;
    if (c->nreg == 2) {
        // Low-storage form (:117): the same Eq.6 / Eq.7 arithmetic with ONE work register next to U^n; stages 2 and 3 replace the work
        // register in place (the x kernel reads U_(s) at its own cell before it stores there).
        double* Rw = c->U[1 - c->cur];
        Stage s1 = { 0, 1.0, 0.0, 1.0, 0.0 };
        if ((rc = run_stage(c, Un, s1, Un, Rw)) != MF_OK) return rc;
        if (c->rk == 2) {
            Stage s2 = { 1, 0.5, 0.5, 1.0, 1.0 };
            s2.cfl = 1;
            if ((rc = run_stage(c, Rw, s2, Un, Rw)) != MF_OK) return rc;
        } else {
            Stage s2 = { 2, 0.75, 0.25, 0.25, 1.0 };
            Stage s3 = { 2, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 0.5 };
            s3.cfl = 1;
            if ((rc = run_stage(c, Rw, s2, Un, Rw)) != MF_OK) return rc;
            if ((rc = run_stage(c, Rw, s3, Un, Rw)) != MF_OK) return rc;
        }
        c->cur = 1 - c->cur;
        c->launches += launch_end_step(c->ds, c->nev, c->stream);
        c->smax_valid = 1;
        return MF_OK;
    }
    double* Ra = c->U[(c->cur + 1) % 3];
    double* Rb = c->U[(c->cur + 2) % 3];
    if (c->rk == 2) {
        Stage s1 = { 0, 1.0, 0.0, 1.0, 0.0 };
        Stage s2 = { 1, 0.5, 0.5, 1.0, 1.0 };
        s2.cfl = last_stage_reduces_cfl(c);
        if ((rc = run_stage(c, Un, s1, Un, Ra)) != MF_OK) return rc;
        if ((rc = run_stage(c, Ra, s2, Un, Rb)) != MF_OK) return rc;
        c->cur = (c->cur + 2) % 3;
    } else {
        Stage s1 = { 0, 1.0, 0.0, 1.0, 0.0 };
        Stage s2 = { 2, 0.75, 0.25, 0.25, 1.0 };
        Stage s3 = { 2, 1.0 / 3.0, 2.0 / 3.0, 2.0 / 3.0, 0.5 };
        s3.cfl = last_stage_reduces_cfl(c);
        if ((rc = run_stage(c, Un, s1, Un, Ra)) != MF_OK) return rc;
        if ((rc = run_stage(c, Ra, s2, Un, Rb)) != MF_OK) return rc;
        if ((rc = run_stage(c, Rb, s3, Un, Ra)) != MF_OK) return rc;
        c->cur = (c->cur + 1) % 3;
    }
    c->launches += launch_end_step(c->ds, c->nev, c->stream);
    c->smax_valid = last_stage_reduces_cfl(c);
    return MF_OK;
}

int check_launch(mf_ctx* c)
{
    cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(c, e, "kernel launch");
    return MF_OK;
}

// synchronise and fetch the device-side step state into the pinned mirror
int fetch_step_state(mf_ctx* c)
{
    MF_CUDA(c, cudaMemcpyAsync(c->h_ds, c->ds, sizeof(StepState) * c->nev, cudaMemcpyDeviceToHost, c->stream));
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    int status = 0;
    for (int ev = 0; ev < c->nev; ++ev) status |= c->h_ds[ev].status;
    if (status) return fail(c, MF_ESTATE, "a CFL reduction met a non-finite or superluminal (|M| > E) cell");
    return MF_OK;
}

} // namespace

extern "C" {

const char* mf_version(void) { return MF_VERSION_STR; }

mf_ctx* mf_create(int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages)
{
    return mf_create_batch(1, nx, ny, nz, dx, eos, limiter, k_stages);
}

mf_ctx* mf_create_batch(int nevents, int nx, int ny, int nz, double dx, int eos, int limiter, int k_stages)
{
    const int n[3] = { nx, ny, nz };
    if (nevents < 1 || nevents > 65535) { fail(nullptr, MF_EINVAL, "the number of events must be in 1..65535"); return nullptr; }
    for (int a = 0; a < 3; ++a)
        if (n[a] < 1 || (n[a] > 1 && n[a] < 4)) { fail(nullptr, MF_EINVAL, "each extent must be 1 (inactive) or >= 4"); return nullptr; }
    if (!(dx > 0.0)) { fail(nullptr, MF_EINVAL, "dx must be > 0"); return nullptr; }
    if (eos != MF_EOS_CS2 && eos != MF_EOS_TABLE) { fail(nullptr, MF_EINVAL, "unknown eos"); return nullptr; }
    if (limiter < 0 || limiter > MF_LIM_FIRST) { fail(nullptr, MF_EINVAL, "unknown limiter"); return nullptr; }
    if (k_stages < 0 || k_stages > 8) { fail(nullptr, MF_EINVAL, "k_stages must be in 0..8"); return nullptr; }

    int ndev = 0;
    cudaError_t e = cudaGetDeviceCount(&ndev);
    if (e != cudaSuccess || ndev < 1) {
        cudaGetLastError();
        fail(nullptr, MF_ECUDA, std::string("no CUDA device (there is no CPU fallback): ") + cudaGetErrorString(e));
        return nullptr;
    }
    mf_ctx* c = new (std::nothrow) mf_ctx();
    if (!c) { fail(nullptr, MF_ENOMEM, "host allocation failed"); return nullptr; }
    memset(&c->g, 0, sizeof(c->g));
    c->g.cslot = -1;
    c->nev = 0;
    c->U[0] = c->U[1] = c->U[2] = nullptr; c->faces = c->fluxes = nullptr; c->delta = nullptr;
    c->ds = nullptr; c->h_ds = nullptr; c->dsc = nullptr;
    c->partials = nullptr; c->h_partials = nullptr; c->own_stream = nullptr; c->stream = nullptr;
    cudaGetDevice(&c->dev);
    cudaDeviceProp prop;
    if (cudaGetDeviceProperties(&prop, c->dev) != cudaSuccess || prop.major < 10) {
        cudaGetLastError();
        fail(nullptr, MF_ECUDA, "device is not sm_100 or newer (library is built for sm_100a only)");
        delete c; return nullptr;
    }
    c->num_sms = prop.multiProcessorCount;
    Grid& g = c->g;
    c->nact = 0;
    for (int a = 0; a < 3; ++a) {
        g.n[a] = n[a]; g.act[a] = n[a] > 1; g.h[a] = g.act[a] ? 1 : 0; g.e[a] = n[a] + 2 * g.h[a];
        c->nact += g.act[a];
    }
    g.periodic = 0;
    g.ncell = (long long)nx * ny * nz;
    g.next = (long long)g.e[0] * g.e[1] * g.e[2];
    g.nev = c->nev = nevents;
    c->nst = g.ncell * nevents; c->nxt = g.next * nevents;
    if (c->nxt >= (1LL << 32)) {                                    // the kernels index cells with unsigned 32-bit offsets
        fail(nullptr, MF_EINVAL, "grid has 2^32 or more cells");
        delete c; return nullptr;
    }
    g.ns[0] = 1; g.ns[1] = nx; g.ns[2] = (long long)nx * ny;
    g.es[0] = 1; g.es[1] = g.e[0]; g.es[2] = (long long)g.e[0] * g.e[1];
    g.dx = dx;
    g.inv_dx = 1.0 / dx;
    g.cslot = slots_acquire(nevents);
    for (int a = 0; a < 2; ++a) for (int m = 0; m < 3; ++m) g.dv[a][m] = make_fastdiv((unsigned int)(n[a] + m));
    set_eos(c->q, 1.0 / 3.0);
    clear_table(c->q);
    c->eos = eos; c->table = nullptr;
    c->limiter = limiter; c->k = k_stages; c->rk = 2; c->predictor = 1;
    c->alpha = c->nact > 0 ? (double)c->nact : 1.0;                 // A9
    memset(&c->src, 0, sizeof(c->src));
    c->path_req = MF_PATH_AUTO; c->cur = 0; c->nreg = 3; c->launches = 0;
    c->prof_on = 0; c->prof_used = 0; c->smax_valid = 0;
    c->graph_on = 1; c->epoch = 0; c->graph_exec = nullptr; c->graph_epoch = 0; c->graph_cur = -1; c->graph_mode = -1; c->graph_steps = 0;
    c->graph_value = 0.0; c->graph_launches = 0; c->graph_captures = 0; c->graph_replays = 0;
    resolve_path(c);
    c->nblocks_tot = c->num_sms * 4;

    bool ok = cudaStreamCreateWithFlags(&c->own_stream, cudaStreamNonBlocking) == cudaSuccess;
    c->stream = c->own_stream;
    for (int r = 0; ok && r < 3; ++r) ok = cudaMalloc(&c->U[r], sizeof(double) * 5 * c->nst) == cudaSuccess;
    ok = ok && cudaMalloc(&c->ds, sizeof(StepState) * nevents) == cudaSuccess;
    ok = ok && cudaMalloc(&c->dsc, sizeof(StepConst) * nevents) == cudaSuccess;
    ok = ok && cudaMallocHost(&c->h_ds, sizeof(StepState) * nevents) == cudaSuccess;
    ok = ok && cudaMalloc(&c->partials, sizeof(double) * 5 * c->nblocks_tot) == cudaSuccess;
    ok = ok && cudaMallocHost(&c->h_partials, sizeof(double) * 5 * c->nblocks_tot) == cudaSuccess;
    if (ok) {
        for (int r = 0; r < 3; ++r) cudaMemsetAsync(c->U[r], 0, sizeof(double) * 5 * c->nst, c->stream);
        c->launches += launch_reset(c->ds, c->nev, c->stream);
        ok = cudaStreamSynchronize(c->stream) == cudaSuccess;
    }
    if (!ok) {
        cudaError_t le = cudaGetLastError();
        fail(nullptr, MF_ENOMEM, std::string("device allocation failed: ") + cudaGetErrorString(le));
        mf_destroy(c);
        return nullptr;
    }
    return c;
}

void mf_destroy(mf_ctx* c)
{
    if (!c) return;
    if (c->stream) cudaStreamSynchronize(c->stream);
    for (int r = 0; r < 3; ++r) if (c->U[r]) cudaFree(c->U[r]);
    if (c->faces) cudaFree(c->faces);
    if (c->fluxes) cudaFree(c->fluxes);
    if (c->delta) cudaFree(c->delta);
    if (c->table) cudaFree(c->table);
    if (c->ds) cudaFree(c->ds);
    if (c->dsc) cudaFree(c->dsc);
    slots_release(c->g.cslot, c->nev);
    if (c->h_ds) cudaFreeHost(c->h_ds);
    if (c->partials) cudaFree(c->partials);
    if (c->h_partials) cudaFreeHost(c->h_partials);
    if (c->graph_exec) cudaGraphExecDestroy(c->graph_exec);
    if (c->own_stream) cudaStreamDestroy(c->own_stream);
    for (cudaEvent_t e : c->prof_ev) cudaEventDestroy(e);
    delete c;
}

const char* mf_last_error(mf_ctx* c) { return c ? c->err.c_str() : g_create_err.c_str(); }

int mf_set_stream(mf_ctx* c, void* cuda_stream)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    c->stream = cuda_stream ? (cudaStream_t)cuda_stream : c->own_stream;
    return MF_OK;
}

int mf_sync(mf_ctx* c)
{
    if (!c) return MF_EINVAL;
    return fetch_step_state(c);
}

int mf_launch_count(mf_ctx* c, long long* launches)
{
    if (!c || !launches) return MF_EINVAL;
    *launches = c->launches;
    return MF_OK;
}

int mf_profile(mf_ctx* c, int on)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    c->prof_on = on ? 1 : 0;
    return MF_OK;
}

int mf_profile_read(mf_ctx* c, double ms[MF_NCLASS], long long launches[MF_NCLASS])
{
    if (!c || !ms || !launches) return MF_EINVAL;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    for (int k = 0; k < MF_NCLASS; ++k) { ms[k] = 0.0; launches[k] = 0; }
    for (size_t i = 0; i < c->prof_used; ++i) {
        float t = 0.f;
        MF_CUDA(c, cudaEventElapsedTime(&t, c->prof_ev[2 * i], c->prof_ev[2 * i + 1]));
        ms[c->prof_cls[i]] += (double)t;
        launches[c->prof_cls[i]] += 1;
    }
    c->prof_used = 0;
    return MF_OK;
}

int mf_probe_fp64(double out[8])
{
    if (!out) return MF_EINVAL;
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev < 1) { cudaGetLastError(); return MF_ECUDA; }
    return probe_fp64(out) == 0 ? MF_OK : MF_ECUDA;
}

} // extern "C"

// ============================================================================ state in / out, stepping, options
namespace {

int reset_after_set(mf_ctx* c)
{
    c->smax_valid = 0;
    c->launches += launch_reset(c->ds, c->nev, c->stream);
    return check_launch(c);
}

// The caller's doubles land in register 0 as doubles (every register is allocated for doubles).  In 32-bit state mode finish_copy_in then
// rounds them into register 1 as floats, which becomes U^n (reading A19: the state handed in is rounded once).
int copy_in(mf_ctx* c, const double* const src[5], cudaMemcpyKind kind)
{
    c->cur = 0;
    for (int v = 0; v < 5; ++v)
        MF_CUDA(c, cudaMemcpyAsync(c->U[0] + v * c->nst, src[v], sizeof(double) * c->nst, kind, c->stream));
    return MF_OK;
}

int finish_copy_in(mf_ctx* c)
{
    if (!c->g.state32) return MF_OK;
    c->launches += launch_state_convert(c->nst, 1, cstate(c->U[0], c->nst), reg(c, c->U[1]), c->num_sms, c->stream);
    c->cur = 1;
    return MF_OK;
}

// `base` holds doubles, nst per component
int copy_out(mf_ctx* c, const double* base, double* const dst[5], cudaMemcpyKind kind)
{
    for (int v = 0; v < 5; ++v)
        MF_CUDA(c, cudaMemcpyAsync(dst[v], base + v * c->nst, sizeof(double) * c->nst, kind, c->stream));
    return MF_OK;
}

// U^n as doubles: the register itself, or in 32-bit state mode its widened copy in the next (free between steps) register
const double* state_as_doubles(mf_ctx* c)
{
    if (!c->g.state32) return c->U[c->cur];
    double* scratch = c->U[(c->cur + 1) % c->nreg];
    c->launches += launch_state_convert(c->nst, 0, creg(c, c->U[c->cur]), state(scratch, c->nst), c->num_sms, c->stream);
    return scratch;
}

} // namespace

extern "C" {

int mf_set_state(mf_ctx* c, const double* E, const double* Mx, const double* My, const double* Mz, const double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    const double* src[5] = { E, Mx, My, Mz, R };
    int rc = copy_in(c, src, cudaMemcpyHostToDevice);
    if (rc != MF_OK) return rc;
    finish_copy_in(c);
    if ((rc = reset_after_set(c)) != MF_OK) return rc;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    return MF_OK;
}

int mf_set_state_async(mf_ctx* c, const double* E, const double* Mx, const double* My, const double* Mz, const double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    const double* src[5] = { E, Mx, My, Mz, R };
    int rc = copy_in(c, src, cudaMemcpyHostToDevice);
    if (rc != MF_OK) return rc;
    finish_copy_in(c);
    return reset_after_set(c);                                     // no synchronisation: the host arrays stay in use until the stream has passed
}

int mf_get_state_async(mf_ctx* c, double* E, double* Mx, double* My, double* Mz, double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    double* dst[5] = { E, Mx, My, Mz, R };
    int rc = copy_out(c, state_as_doubles(c), dst, cudaMemcpyDeviceToHost);
    if (rc != MF_OK) return rc;
    return check_launch(c);                                        // the arrays are complete after the next mf_sync
}

int mf_set_state_device(mf_ctx* c, const double* E, const double* Mx, const double* My, const double* Mz, const double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    const double* src[5] = { E, Mx, My, Mz, R };
    int rc = copy_in(c, src, cudaMemcpyDeviceToDevice);
    if (rc != MF_OK) return rc;
    finish_copy_in(c);
    return reset_after_set(c);
}

int mf_get_state(mf_ctx* c, double* E, double* Mx, double* My, double* Mz, double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    double* dst[5] = { E, Mx, My, Mz, R };
    int rc = copy_out(c, state_as_doubles(c), dst, cudaMemcpyDeviceToHost);
    if (rc != MF_OK) return rc;
    return fetch_step_state(c);
}

int mf_get_state_device(mf_ctx* c, double* E, double* Mx, double* My, double* Mz, double* R)
{
    if (!c) return MF_EINVAL;
    if (!E || !Mx || !My || !Mz || !R) return fail(c, MF_EINVAL, "null pointer");
    double* dst[5] = { E, Mx, My, Mz, R };
    int rc = copy_out(c, state_as_doubles(c), dst, cudaMemcpyDeviceToDevice);
    if (rc != MF_OK) return rc;
    return fetch_step_state(c);
}

int mf_set_state_prim(mf_ctx* c, const double* e, const double* vx, const double* vy, const double* vz, const double* n)
{
    if (!c) return MF_EINVAL;
    if (!e || !vx || !vy || !vz || !n) return fail(c, MF_EINVAL, "null pointer");
    const double* src[5] = { e, vx, vy, vz, n };
    int rc = copy_in(c, src, cudaMemcpyHostToDevice);
    if (rc != MF_OK) return rc;
    c->launches += launch_prim2con(c->g, c->q, state(c->U[0], c->nst), c->stream);      // Eq.4 on the device
    finish_copy_in(c);
    if ((rc = reset_after_set(c)) != MF_OK) return rc;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    return MF_OK;
}

int mf_get_state_prim(mf_ctx* c, double* e, double* vx, double* vy, double* vz, double* n)
{
    if (!c) return MF_EINVAL;
    if (!e || !vx || !vy || !vz || !n) return fail(c, MF_EINVAL, "null pointer");
    double* scratch = c->U[(c->cur + 1) % c->nreg];
    c->launches += launch_con2prim(c->g, c->q, creg(c, c->U[c->cur]), state(scratch, c->nst), c->stream);
    int rc = check_launch(c);
    if (rc != MF_OK) return rc;
    double* dst[5] = { e, vx, vy, vz, n };
    if ((rc = copy_out(c, scratch, dst, cudaMemcpyDeviceToHost)) != MF_OK) return rc;
    return fetch_step_state(c);
}

// per-step scalars on the device, then their copy into the constant memory of the unit whose kernels run this path
static int begin_step(mf_ctx* c, int mode, double value)
{
    c->launches += launch_begin_step(c->ds, c->dsc, c->nev, mode, value, c->g.dx, c->alpha, c->stream);
    if (c->g.cslot >= 0 && (c->path == MF_PATH_STAGED || c->path == MF_PATH_HYBRID || c->path == MF_PATH_SMALL)) {   // (SMALL: mf_eval_L runs staged kernels)
        if (upload_step_const_staged(c->dsc, c->g.cslot, c->nev, c->stream) != 0) { cudaGetLastError(); return fail(c, MF_ECUDA, "copy of the step scalars to constant memory failed"); }
    }
    if (c->g.cslot >= 0 && c->path == MF_PATH_HYBRID) {
        if (upload_step_const_tile(c->dsc, c->g.cslot, c->nev, c->stream) != 0) { cudaGetLastError(); return fail(c, MF_ECUDA, "copy of the step scalars to constant memory failed"); }
    }
    return MF_OK;
}

// ---- stepping.  One step = (CFL reduction if the accumulator is stale) + per-step scalars + the RK stages; nothing in it needs the host.
// mode 0: dt = value*dx/S_max (value = cfl); mode 1: dt = value.
static int enqueue_step(mf_ctx* c, int mode, double value)
{
    if (mode == 0 && !c->smax_valid) {                            // otherwise the previous step's last combine already reduced U^n
        int ps = prof_begin(c, 0);
        c->launches += launch_cfl(c->g, c->q, creg(c, c->U[c->cur]), c->ds, c->num_sms, c->stream);   // a2, from U^n
        prof_end(c, ps);
    }
    int rc = begin_step(c, mode, value);
    if (rc != MF_OK) return rc;
    return run_step(c);
}

// Launch-bound grids (config 1: 400 cells, 8 launches of a few microseconds of work each): after one eager step - which allocates the
// scratch and brings the S_max accumulator into its steady state - a whole period of the register rotation (3 steps, 2 in low-storage
// mode) is captured into a CUDA graph once and replayed.  Every per-step scalar lives in device memory (StepState), so the replayed
// launches are exactly the eager ones; what IS baked into the graph (cfl or dt, the option set, the stream, the starting register) is its key.
static int run_steps(mf_ctx* c, int n, int mode, double value)
{
    int done = 0, rc;
    if (c->path == MF_PATH_SMALL && n > 0) {
        // the whole call is one launch: the kernel takes S_max of U^n itself at every step, rotates the registers like run_step and keeps the clock
        int ps = prof_begin(c, 4);
        c->launches += launch_small_steps(c->g, c->q, c->limiter, c->predictor, c->k, c->rk, c->alpha, mode, value, n, c->cur, c->U, c->src, c->ds, c->stream);
        prof_end(c, ps);
        c->cur = (c->cur + (long long)n * (c->rk == 2 ? 2 : 1)) % 3;
        c->smax_valid = 0;
        return check_launch(c);
    }
    const int period = c->nreg;                                   // cur returns to its value after this many steps (RK2 and RK3 alike)
    if (c->graph_on && !c->prof_on && n >= 1 + 2 * period) {
        if ((rc = enqueue_step(c, mode, value)) != MF_OK) return rc;
        if ((rc = check_launch(c)) != MF_OK) return rc;
        done = 1;
        const bool same_key = c->graph_exec && c->graph_epoch == c->epoch && c->graph_mode == mode && c->graph_value == value &&
                              c->graph_steps == period;
        // The captured period starts from one particular state register.  A call whose step count is not a multiple of the period leaves
        // U^n in another one: walk there with at most period - 1 eager steps instead of throwing the graph away.
        while (same_key && c->graph_cur != c->cur && n - done > period) {
            if ((rc = enqueue_step(c, mode, value)) != MF_OK) return rc;
            ++done;
        }
        const bool hit = same_key && c->graph_cur == c->cur;
        if (!hit) {
            c->graph_captures++;
            if (c->graph_exec) {                                   // the old graph may still be running on this stream
                MF_CUDA(c, cudaStreamSynchronize(c->stream));
                cudaGraphExecDestroy(c->graph_exec); c->graph_exec = nullptr;
            }
            const int cur0 = c->cur, smax0 = c->smax_valid;
            const long long l0 = c->launches;
            cudaGraph_t graph = nullptr;
            if (cudaStreamBeginCapture(c->stream, cudaStreamCaptureModeThreadLocal) == cudaSuccess) {
                rc = MF_OK;
                for (int s = 0; s < period && rc == MF_OK; ++s) rc = enqueue_step(c, mode, value);
                const cudaError_t e = cudaStreamEndCapture(c->stream, &graph);
                c->graph_launches = c->launches - l0;
                c->launches = l0;                                  // nothing ran yet: the capture only recorded
                c->cur = cur0; c->smax_valid = smax0;
                if (rc != MF_OK || e != cudaSuccess || !graph || cudaGraphInstantiate(&c->graph_exec, graph, 0) != cudaSuccess) {
                    cudaGetLastError();
                    c->graph_exec = nullptr;                       // fall back to eager launches below
                }
                if (graph) cudaGraphDestroy(graph);
            } else cudaGetLastError();
            if (c->graph_exec) {
                c->graph_epoch = c->epoch; c->graph_cur = c->cur; c->graph_mode = mode; c->graph_value = value; c->graph_steps = period;
            }
        }
        if (c->graph_exec) {
            while (n - done >= period) {
                MF_CUDA(c, cudaGraphLaunch(c->graph_exec, c->stream));
                c->graph_replays++;
                c->launches += c->graph_launches;
                done += period;                                    // cur and smax_valid are back where they were
            }
        }
    }
    for (; done < n; ++done)
        if ((rc = enqueue_step(c, mode, value)) != MF_OK) return rc;
    return check_launch(c);
}

int mf_step(mf_ctx* c, int n, double cfl)
{
    if (!c) return MF_EINVAL;
    if (n < 0 || !(cfl > 0.0)) return fail(c, MF_EINVAL, "bad n or cfl");
    return run_steps(c, n, 0, cfl);
}

int mf_step_dt(mf_ctx* c, int n, double dt)
{
    if (!c) return MF_EINVAL;
    if (n < 0 || !(dt > 0.0)) return fail(c, MF_EINVAL, "bad n or dt");
    return run_steps(c, n, 1, dt);
}

int mf_set_graph(mf_ctx* c, int on)
{
    if (!c) return MF_EINVAL;
    c->graph_on = on ? 1 : 0;
    return MF_OK;
}

int mf_graph_stats(mf_ctx* c, long long* captures, long long* replays)
{
    if (!c) return MF_EINVAL;
    if (captures) *captures = c->graph_captures;
    if (replays) *replays = c->graph_replays;
    return MF_OK;
}

int mf_eval_L(mf_ctx* c, double dt, double* L_E, double* L_Mx, double* L_My, double* L_Mz, double* L_R)
{
    if (!c) return MF_EINVAL;
    if (!(dt > 0.0) || !L_E || !L_Mx || !L_My || !L_Mz || !L_R) return fail(c, MF_EINVAL, "bad dt or null pointer");
    double* Un = c->U[c->cur];
    double* scratch = c->U[(c->cur + 1) % c->nreg];
    { int rb = begin_step(c, 1, dt); if (rb != MF_OK) return rb; }
    Stage sg = { 3, 0.0, 0.0, 0.0, 0.0 };
    c->smax_valid = 0;
    Source keep = c->src;
    c->src.on = 0;
    int rc = run_stage(c, Un, sg, Un, scratch);
    c->src = keep;
    if (rc != MF_OK) return rc;
    if ((rc = check_launch(c)) != MF_OK) return rc;
    double* dst[5] = { L_E, L_Mx, L_My, L_Mz, L_R };
    if ((rc = copy_out(c, scratch, dst, cudaMemcpyDeviceToHost)) != MF_OK) return rc;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    return MF_OK;
}

// event < 0: all events of the batch
static int totals_of(mf_ctx* c, int event, double out[5])
{
    Grid g = c->g;
    const CState5 U = creg(c, c->U[c->cur], event < 0 ? 0 : (long long)event * g.ncell);
    if (event < 0) g.ncell = c->nst;
    c->launches += launch_totals(g, U, c->partials, c->nblocks_tot, c->stream);
    int rc = check_launch(c);
    if (rc != MF_OK) return rc;
    MF_CUDA(c, cudaMemcpyAsync(c->h_partials, c->partials, sizeof(double) * 5 * c->nblocks_tot, cudaMemcpyDeviceToHost, c->stream));
    rc = fetch_step_state(c);
    double vol = 1.0;
    for (int a = 0; a < 3; ++a) if (c->g.act[a]) vol *= c->g.dx;
    for (int v = 0; v < 5; ++v) {
        long double acc = 0.0L;
        for (int b = 0; b < c->nblocks_tot; ++b) acc += (long double)c->h_partials[v * c->nblocks_tot + b];
        out[v] = (double)(acc * (long double)vol);
    }
    return rc;
}

int mf_conserved_totals(mf_ctx* c, double out[5])
{
    if (!c || !out) return MF_EINVAL;
    return totals_of(c, -1, out);
}

int mf_conserved_totals_event(mf_ctx* c, int event, double out[5])
{
    if (!c || !out) return MF_EINVAL;
    if (event < 0 || event >= c->nev) return fail(c, MF_EINVAL, "no such event");
    return totals_of(c, event, out);
}

int mf_batch_size(mf_ctx* c) { return c ? c->nev : MF_EINVAL; }

int mf_get_time_event(mf_ctx* c, int event, double* t, double* last_dt, long long* steps)
{
    if (!c) return MF_EINVAL;
    if (event < 0 || event >= c->nev) return fail(c, MF_EINVAL, "no such event");
    int rc = fetch_step_state(c);
    if (t) *t = c->h_ds[event].t;
    if (last_dt) *last_dt = c->h_ds[event].dt;
    if (steps) *steps = c->h_ds[event].steps;
    return rc;
}

int mf_get_time(mf_ctx* c, double* t, double* last_dt, long long* steps) { return mf_get_time_event(c, 0, t, last_dt, steps); }

int mf_max_signal_speed(mf_ctx* c, double* smax)
{
    if (!c || !smax) return MF_EINVAL;
    c->launches += launch_cfl(c->g, c->q, creg(c, c->U[c->cur]), c->ds, c->num_sms, c->stream);
    int rc = check_launch(c);
    if (rc != MF_OK) return rc;
    rc = fetch_step_state(c);
    unsigned long long bits = 0;                                   // non-negative doubles: bit order == value order
    for (int ev = 0; ev < c->nev; ++ev) if (c->h_ds[ev].smax_bits > bits) bits = c->h_ds[ev].smax_bits;
    memcpy(smax, &bits, sizeof(double));
    // leave the accumulators empty for the next reduction
    c->smax_valid = 0;
    cudaMemset2DAsync(&c->ds[0].smax_bits, sizeof(StepState), 0, sizeof(unsigned long long), (size_t)c->nev, c->stream);   // one strided memset for all events
    return rc;
}

int mf_set_rk(mf_ctx* c, int order)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (order != 2 && order != 3) return fail(c, MF_EINVAL, "rk order must be 2 or 3");
    c->rk = order; return MF_OK;
}
int mf_set_boundary(mf_ctx* c, int bc)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (bc != MF_BC_OUTFLOW && bc != MF_BC_PERIODIC) return fail(c, MF_EINVAL, "unknown boundary condition");
    c->g.periodic = bc == MF_BC_PERIODIC; return MF_OK;
}
int mf_set_cs2(mf_ctx* c, double cs2)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (!(cs2 > 0.0) || !(cs2 < 1.0)) return fail(c, MF_EINVAL, "cs2 must be in (0,1)");
    set_eos(c->q, cs2);
    c->smax_valid = 0;                                             // the accumulator holds S_max for the old sound speed
    return MF_OK;
}
int mf_set_eos_table(mf_ctx* c, int ne, int nn, double ln_e0, double dln_e, double n0, double dn, const double* ln_p)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (c->eos != MF_EOS_TABLE) return fail(c, MF_EINVAL, "context was not created with MF_EOS_TABLE");
    if (ne < 2 || nn < 1 || !(dln_e > 0.0) || (nn > 1 && !(dn > 0.0)) || !ln_p) return fail(c, MF_EINVAL, "bad table");
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    if (c->table) { cudaFree(c->table); c->table = nullptr; }
    const size_t count = (size_t)ne * nn, bytes = sizeof(double) * count;
    if (cudaMalloc(&c->table, bytes + sizeof(float) * count) != cudaSuccess) { cudaGetLastError(); c->table = nullptr; return fail(c, MF_ENOMEM, "cudaMalloc(EOS table) failed"); }
    MF_CUDA(c, cudaMemcpy(c->table, ln_p, bytes, cudaMemcpyHostToDevice));
    {                                                  // float copy behind the doubles: the fp32 seed of the speed solve reads it
        std::vector<float> lf(count);
        for (size_t i = 0; i < count; ++i) lf[i] = (float)ln_p[i];
        MF_CUDA(c, cudaMemcpy(c->table + count, lf.data(), sizeof(float) * count, cudaMemcpyHostToDevice));
    }
    c->q.kind = 1; c->q.ne = ne; c->q.nn = nn; c->q.ln_e0 = ln_e0; c->q.dln_e = dln_e; c->q.n0 = n0; c->q.dn = nn > 1 ? dn : 1.0;
    c->q.lnp = c->table;
    c->q.lnpf = reinterpret_cast<const float*>(c->table + count);
    c->q.inv_dln_e = 1.0 / c->q.dln_e; c->q.inv_dn = 1.0 / c->q.dn;
    c->smax_valid = 0;
    return MF_OK;
}
int mf_set_predictor(mf_ctx* c, int on)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    const int keep = c->predictor;
    c->predictor = on ? 1 : 0;
    if (resolve_path(c) != MF_OK) { c->predictor = keep; resolve_path(c); return fail(c, MF_EINVAL, "the selected path does not support this predictor setting: select another path first"); }
    return MF_OK;
}
int mf_set_alpha(mf_ctx* c, double alpha)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (!(alpha > 0.0)) return fail(c, MF_EINVAL, "alpha must be > 0");
    c->alpha = alpha; return MF_OK;
}
int mf_set_jet_source(mf_ctx* c, double dEdx, double sigma, double x0, double y0, double z0)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (dEdx != 0.0 && !(sigma > 0.0)) return fail(c, MF_EINVAL, "sigma must be > 0");
    const double PI = 3.14159265358979323846;
    double s2 = sigma > 0.0 ? sigma * sigma : 1.0;
    c->src.dEdx = dEdx;
    c->src.norm = 1.0 / std::pow(2.0 * PI * s2, 1.5);
    c->src.inv_two_s2 = 1.0 / (2.0 * s2);
    c->src.x0 = x0; c->src.y0 = y0; c->src.z0 = z0;
    c->src.on = dEdx != 0.0;
    return MF_OK;
}
int mf_set_path(mf_ctx* c, int path)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    if (path < MF_PATH_AUTO || path > MF_PATH_SMALL) return fail(c, MF_EINVAL, "unknown path");
    int keep = c->path_req;
    c->path_req = path;
    if (resolve_path(c) != MF_OK) { c->path_req = keep; resolve_path(c); return fail(c, MF_EINVAL, "this path does not support this configuration (fused/hybrid: three active axes, MF_EOS_CS2, one event; sweep: active x axis, MF_EOS_CS2, and with the predictor on a 3D grid and one event; small: 1D, nx <= 766, MF_EOS_CS2, one event; low storage: staged only)"); }
    return MF_OK;
}
int mf_set_low_storage(mf_ctx* c, int on)
{
    if (!c) return MF_EINVAL;
    c->epoch++;
    on = on ? 1 : 0;
    if (on == (c->nreg == 2)) return MF_OK;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    if (on) {
        c->nreg = 2;
        if (resolve_path(c) != MF_OK) { c->nreg = 3; resolve_path(c); return fail(c, MF_EINVAL, "low-storage Runge-Kutta runs on the staged path only: select MF_PATH_AUTO or MF_PATH_STAGED first"); }
        if (c->cur == 2) {                                         // bring U^n into one of the two registers that stay
            MF_CUDA(c, cudaMemcpy(c->U[0], c->U[2], sizeof(double) * 5 * c->nst, cudaMemcpyDeviceToDevice));
            c->cur = 0;
        }
        cudaFree(c->U[2]); c->U[2] = nullptr;
    } else {
        if (cudaMalloc(&c->U[2], sizeof(double) * 5 * c->nst) != cudaSuccess) { cudaGetLastError(); c->U[2] = nullptr; return fail(c, MF_ENOMEM, "cudaMalloc(third state register) failed"); }
        c->nreg = 3;
        resolve_path(c);
    }
    return MF_OK;
}

int mf_set_state_precision(mf_ctx* c, int bits)
{
    if (!c) return MF_EINVAL;
    if (bits != 32 && bits != 64) return fail(c, MF_EINVAL, "state precision must be 32 or 64 bits");
    const int on = bits == 32;
    if (on == c->g.state32) return MF_OK;
    c->epoch++;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    const int keep = c->g.state32;
    c->g.state32 = on;
    if (resolve_path(c) != MF_OK) {
        c->g.state32 = keep; resolve_path(c);
        return fail(c, MF_EINVAL, "the single-precision state runs on the staged path and, without the Hancock step, on the sweep path: select MF_PATH_AUTO or MF_PATH_STAGED first");
    }
    // the stored state changes its element type: U^n is converted into the next register (free between steps), which becomes U^n
    const int next = (c->cur + 1) % c->nreg;
    c->launches += launch_state_convert(c->nst, on, creg_as(c, c->U[c->cur], keep != 0), reg_as(c, c->U[next], on != 0), c->num_sms, c->stream);
    c->cur = next;
    c->smax_valid = 0;                                             // S_max is taken from the stored (rounded) state
    int rc = check_launch(c);
    if (rc != MF_OK) return rc;
    MF_CUDA(c, cudaStreamSynchronize(c->stream));
    return MF_OK;
}

int mf_get_state_precision(mf_ctx* c, int* bits) { if (!c || !bits) return MF_EINVAL; *bits = c->g.state32 ? 32 : 64; return MF_OK; }

int mf_memory_bytes(mf_ctx* c, long long* bytes)
{
    if (!c || !bytes) return MF_EINVAL;
    long long b = (long long)sizeof(double) * 5 * c->nst * c->nreg;
    if (c->faces) b += (long long)sizeof(double) * 10 * c->nact * c->nxt;
    if (c->fluxes) b += (long long)sizeof(double) * 5 * c->nact * c->nxt;
    if (c->delta) b += (long long)sizeof(double) * 5 * c->g.next;
    if (c->table) b += (long long)(sizeof(double) + sizeof(float)) * c->q.ne * c->q.nn;
    b += (long long)sizeof(StepState) * c->nev + (long long)sizeof(double) * 5 * c->nblocks_tot;
    *bytes = b;
    return MF_OK;
}

int mf_get_path(mf_ctx* c, int* path) { if (!c || !path) return MF_EINVAL; *path = c->path; return MF_OK; }

} // extern "C"
