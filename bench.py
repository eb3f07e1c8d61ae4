#!/usr/bin/env python
"""bench.py — fp64 cell-updates/s of the MUSTA-FORCE step (BASELINE.json metric) on N GPUs of one node.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3] [--grid nz,ny,nx] [--path auto]

A "step" is one pass of the whole hot path (CFL reduction, all RK stages: ghost handling, limited reconstruction,
Hancock predictor, MUSTA/FORCE fluxes with con2prim, flux divergence, RK combine) over one synthetic grid.
Default workload: BASELINE.json config 3 (the one the metric is quoted on): 256^3 periodic Gaussian hot spot,
dx 0.05, k=3, superbee, RK3, cfl 0.3.  N > 1 runs N independent replicas (the path does not shard in this build,
DESIGN.md "Multi-GPU"): weak scaling, no data-path collective.

One JSON line on stdout (rank 0).  --impl reference times the CPU oracle (oracle/) on a bounded sample instead.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1510_06340_b200 import workloads  # noqa: E402
from paper_1510_06340_b200.replicas import Replicas  # noqa: E402

METRIC = "fp64 cell-updates/s, MUSTA-FORCE step"
UNIT = "cell-updates/s"

# ----------------------------------------------------------------------------------------------------------------
# Algorithmic work per cell-update.  FP64-pipe issue SLOTS:
# add/sub/mul/fma/compare/min/max = 1, abs/neg/select = 0, and two conventions for the divide and the square root:
#   "survey"  (the frozen round-1 denominator): divide = 8, square root = 8, one flux evaluation 16 + 8 + 8 = 32;
#   "minimal" (what the product code demonstrates, mf_device.cuh flux_fast: Newton reciprocal 3, Newton root 6, F_E = M_d): flux = 24.
# The survey count is ABOVE the instructions the kernels issue (644 slots against ~485 FP64 instructions per MUSTA interface, k = 3), so
# a fraction of it flatters the FP64 pipe; bench.py reports both, and the minimal one is the figure to compare with pipe utilisation.
DIV, SQRT = 8, 8
FLUX = 16 + DIV + SQRT                    # a6: one flux evaluation with con2prim             = 32
DIV_MIN, SQRT_MIN, FLUX_MIN = 3, 6, 24
SLOPE = {"none": 2, "first": 0, "minmod": 3, "superbee": 7, "mc": 8, "vanleer": 4 + DIV, "vanalbada": 6 + DIV}
# Tabulated EOS (8(f) row 1): a flux evaluation is the 16 slots of the flux arithmetic plus one speed solve.  Measured on this workload with the
# counting build (-DMF_COUNT_EVALS: 1.84e9 solves at 128^3, one full table evaluation and 0.00 incremental ones per solve, no fallback): the
# fp32-seeded Newton reaches its stopping rule after ONE fp64 evaluation, ~185 FP64 instructions per solve (root 6, three reciprocals 9, log ~20,
# exp ~20, bilinear lookup with derivatives ~25, Newton step and the first-order pressure update ~20, admissibility and cell test ~20, the rest
# in the guard), so the algorithmic count is 16 + 185 = 201 slots in both conventions (its root and reciprocals are already the minimal ones).
FLUX_TABLE = 16 + 185
SLOPE_MIN = {"none": 2, "first": 0, "minmod": 3, "superbee": 7, "mc": 8, "vanleer": 4 + DIV_MIN, "vanalbada": 6 + DIV_MIN}


def alg_slots(limiter, k, rk, ndim, predictor=True, minimal=False, table=False):
    """(slots per cell-update, slots per L-evaluation, slots of the MUSTA fluxes per L-evaluation)."""
    flux, div, sqrt, slope = (FLUX_MIN, DIV_MIN, SQRT_MIN, SLOPE_MIN) if minimal else (FLUX, DIV, SQRT, SLOPE)
    if table:
        flux = FLUX_TABLE
    recon = 5 * ndim * (4 + slope[limiter])                         # a3: a, b, slope, two face values
    pred = (2 * ndim * flux + 5 * 4 * ndim) if predictor else 0     # a4: 2D flux evaluations + delta + 2D face updates
    force = 3 * flux + 50                                           # Eq.9-11: three fluxes + 10 per component
    musta = (k + 1) * force + 20 * k                                # a5: k Eq.8 updates
    comb = 5 * (2 * ndim + 5)                                       # a7: divergence + RK form
    cfl = ((FLUX_TABLE + 60) if table else (16 + div + sqrt)) + (3 + sqrt) + (2 + div) + 1     # a2 (table: one more lookup for the sound speed)
    per_L = recon + pred + ndim * musta + comb
    return rk * per_L + cfl, per_L, ndim * musta


def class_work(path, limiter, k, ndim, x_active, predictor=True, state_bytes=8, table=False):
    """Algorithmic (FP64 slots, HBM bytes) per cell of one launch group of each kernel class, for one RK stage.
    Bytes are what that kernel must read and write given the data layout of DESIGN.md section 4; `state_bytes` is the size of a stored
    state element (8, or 4 in single-precision state mode, staged path only: the scratch stays fp64)."""
    sb = 5 * state_bytes                                                       # one state, per cell
    fl = FLUX_TABLE if table else FLUX
    recon = 5 * ndim * (4 + SLOPE[limiter])
    pred = (2 * ndim * fl + 5 * 4 * ndim) if predictor else 0
    musta = (k + 1) * (3 * fl + 50) + 20 * k
    comb = 5 * (2 * ndim + 5)
    if path == "staged":
        nflux = ndim - 1 if x_active else ndim
        out = {"cell_stage": (recon + pred, sb + 40 * (1 + ndim)),            # U in; W and the half slopes H_d out
               "flux_stage": (nflux * musta, nflux * 120)}                    # W, H_d in, F_d out, per direction
        if x_active:
            out["combine"] = (musta + comb, 80 + 40 * (ndim - 1) + 2 * sb + sb)   # W, H_x, F_y, F_z, U^n, U_(s) in; new state out
        else:
            out["combine"] = (comb, 40 * ndim + 2 * sb + sb)
        return out
    if path == "sweep":
        # the sweep kernels limit their own slopes (one direction's share of the reconstruction each) from U; with the predictor on a
        # separate kernel writes delta (the reconstruction is then counted once more there: it is needed for Eq.13)
        rdir = recon // ndim
        dl = 40 if predictor else 0
        out = {"flux_stage": ((ndim - 1) * (musta + rdir), (ndim - 1) * (sb + dl + 40)),          # U (+ delta) in, F_d out
               "combine": (musta + rdir + comb, sb + dl + 40 * (ndim - 1) + sb + sb)}            # U (+ delta), F_y, F_z, U^n in; new state out
        if predictor:
            out["cell_stage"] = (recon + pred, 80)                                                 # U in, delta out
        return out
    if path == "hybrid":
        return {"cell_stage": (recon + pred, 40 + 40 * (1 + ndim)), "fused_stage": (ndim * musta + comb, 40 + 40 * ndim + 80 + 40)}
    return {"cell_stage": (recon + pred, 80), "fused_stage": (recon + ndim * musta + comb, 80 + 80 + 40)}   # fused: delta kernel + tile kernel


def alg_bytes(rk, state_bytes=8):
    """Minimum HBM bytes per cell-update: stage 1 reads U^n writes U1 (80 B), later stages read U_s and U^n, write (120 B); CFL +32 B
    (halved with a single-precision state)."""
    return (80 + 120 * (rk - 1) + 32) * state_bytes // 8


# DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum per launch group, GB) of the kernels of THIS workload and path, from the ncu
# --set full captures committed under profiles/ - measured once under ncu, not during this run: the JSON line names the file
# ("traffic_source"), and nothing is reported for a workload, path or state precision without a committed capture.
NCU_TRAFFIC_256 = {
    ("staged", True): ("profiles/r02_ncu_full_staged_256.md", {"cell_stage": 3.396, "flux_stage": 3.409, "combine": 4.716}),
    ("hybrid", True): ("profiles/r02_ncu_hybrid_tile3_256.md", {"fused_stage": 5.602}),
    ("sweep", False): ("profiles/r01_ncu_full_sweep_256.md", {"flux_stage": 2.664, "combine": 3.359}),
}

FP64_LANES_PER_SM = 64       # B200 (sm_100): 4 SMSPs x 16 FP64 lanes; mf_probe_fp64 measures it


def peaks():
    mp = {}
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        mp = json.load(open(path))
    hbm = mp.get("hbm_gbs", 6650.0)
    return dict(hbm_gbs=hbm, hbm_source="measured (MEASURED_PEAKS.json)" if "hbm_gbs" in mp else "fallback (B200_PROFILING.md)",
                sm_max_mhz=mp.get("sm_max_mhz", 1965.0))


# ----------------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi samples of SM clock and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = "clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "--id=%d" % self.index, "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                          "-lms", "20"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def wait_first(self, timeout_s):
        t_end = time.perf_counter() + timeout_s
        while self.proc is not None and not self.lines and time.perf_counter() < t_end:
            time.sleep(0.01)

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0=None, t1=None):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        clocks, maxc, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ts, line in self.lines:
            if t0 is not None and not (t0 <= ts <= t1 + 0.1):
                continue
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                clocks.append(float(f[0])); maxc.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for nme, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nme)
        if not clocks:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples in the timed region"], "samples": 0}
        return {"sm_mhz": float(np.median(clocks)), "sm_max_mhz": float(max(maxc)), "reasons": sorted(reasons),
                "samples": len(clocks), "power_w_max": max(power)}


def make_workload(args):
    shape = tuple(int(x) for x in args.grid.split(",")) if args.grid else None
    st = workloads.gaussian_hot_spot() if (args.config == 3 and shape is None) else workloads.config(args.config, scale=shape)
    if args.predictor == "off":
        st["scheme"] = dict(st["scheme"], predictor=False)
    over = {}
    if args.k is not None:
        over["k_stages"] = args.k
    if args.limiter is not None:
        over["limiter"] = args.limiter
    if args.rk is not None:
        over["rk"] = args.rk
    if over:                                                   # not a BASELINE.json config any more: say so in the workload name
        st["scheme"] = dict(st["scheme"], **over)
        st["name"] = st["name"] + " (scheme overridden: %s)" % ", ".join("%s=%s" % kv for kv in sorted(over.items()))
    return st


def batch_fields(args, st):
    """The state arrays of the run: one event, or --batch B events stacked event-major for mf_create_batch (config 4: the seeded events
    0..B-1 of the 32; any other config: B copies of its state)."""
    fields = ("E", "Mx", "My", "Mz", "R")
    if args.batch <= 1:
        return [np.ascontiguousarray(st[f]) for f in fields]
    if args.config == 4:
        shape = tuple(int(x) for x in args.grid.split(",")) if args.grid else None
        events = [st] + [workloads.lumpy_event(event=ev, shape=shape) for ev in range(1, args.batch)]
    else:
        events = [st] * args.batch
    return [np.ascontiguousarray(np.stack([ev[f] for ev in events])) for f in fields]


def describe(st, extra=None):
    nz, ny, nx = st["shape"]
    cfg = {"workload": "%s %dx%dx%d dx=%g %s k=%d RK%d %s cfl=%g" % (
        st["name"], nx, ny, nz, st["dx"], st["scheme"]["limiter"], st["scheme"]["k_stages"], st["scheme"]["rk"],
        st["scheme"]["bc"], st["cfl"]), "cells": nx * ny * nz,
        "predictor": "on (paper-literal Eq.13)" if st["scheme"].get("predictor", True) else "off (MUSCL + RK, reading A4)"}
    if extra:
        cfg.update(extra)
    return cfg


# ----------------------------------------------------------------------------------------------------------------
def centre_crop(st, m):
    """A centred m^3 (or smaller) sub-box of the workload: the bounded sample the CPU oracle is timed on."""
    nz, ny, nx = st["shape"]
    cz, cy, cx = min(m, nz), min(m, ny), min(m, nx)
    z0, y0, x0 = (nz - cz) // 2, (ny - cy) // 2, (nx - cx) // 2
    out = dict(st)
    for key in ("E", "Mx", "My", "Mz", "R"):
        out[key] = np.ascontiguousarray(st[key][z0:z0 + cz, y0:y0 + cy, x0:x0 + cx])
    out["shape"] = (cz, cy, cx)
    return out


class OracleSample:
    """The CPU oracle as it stands (oracle/libmfo.so, one thread, never tuned for this) on a centred crop."""

    def __init__(self, st, crop):
        from oracle.mfo import Oracle, num_threads
        self.st = centre_crop(st, crop)
        nz, ny, nx = self.st["shape"]
        self.cells = nx * ny * nz
        self.o = Oracle(nx, ny, nz, dx=st["dx"], omp=False, **st["scheme"])
        self.o.set_state(self.st["E"], self.st["Mx"], self.st["My"], self.st["Mz"], self.st["R"])
        if "jet" in st:
            j = st["jet"]
            self.o.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
        self.cores = num_threads(False)
        self.cfl = st["cfl"]
        self.sample = "centred %dx%dx%d crop of the workload's initial state, same scheme" % (nx, ny, nz)

    def time_steps(self, steps):
        t0 = time.perf_counter()
        self.o.step(steps, self.cfl)
        return time.perf_counter() - t0


def cpu_baseline(st, budget_s=12.0, crop=64):
    s = OracleSample(st, crop)
    one = s.time_steps(1)                                     # also the warm-up
    n = max(1, min(50, int(budget_s / max(one, 1e-6))))
    dt = s.time_steps(n)
    return {"value": s.cells * n / dt, "unit": UNIT, "cores": s.cores, "kind": "oracle",
            "sample": "%s, %d steps in %.1f s" % (s.sample, n, dt)}


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, K timed steps after W warm-up steps of a bounded sample."""
    if int(os.environ.get("RANK", "0")) != 0:        # under torchrun rank 0 alone runs it; no process group is needed
        return
    st = make_workload(args)
    s = OracleSample(st, args.ref_crop)
    s.time_steps(max(args.warmup, 1))
    dt = s.time_steps(args.steps)
    value = s.cells * args.steps / dt
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": describe(st, {"sample": s.sample}),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": s.cores, "kind": "oracle", "sample": s.sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ----------------------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    from paper_1510_06340_b200 import binding
    from paper_1510_06340_b200.binding import MustaForce

    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU fallback (use --impl reference for the oracle)")
    rank, local_rank, world = int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))
    torch.cuda.set_device(local_rank)
    rep = Replicas(backend="nccl", device=torch.device("cuda", local_rank))
    st = make_workload(args)
    nz, ny, nx = st["shape"]
    nbatch = max(1, args.batch)
    cells = nx * ny * nz * nbatch
    sch = st["scheme"]
    ndim = sum(1 for n in (nx, ny, nz) if n > 1)
    arrays = batch_fields(args, st)

    stream = torch.cuda.Stream()
    with torch.cuda.stream(stream):
        eos_table = workloads.crossover_eos_table() if args.eos == "table" else None     # 8(f) row 1; not the metric's workload
        g = MustaForce(nx, ny, nz, dx=st["dx"], path=args.path, stream=stream.cuda_stream, eos_table=eos_table,
                       batch=nbatch if nbatch > 1 else None, state_bits=32 if args.state == "f32" else 64, **sch)
        if "jet" in st:
            j = st["jet"]
            g.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
        fields = ("E", "Mx", "My", "Mz", "R")
        # device-resident inputs for the kernel-throughput leg
        dev = [torch.from_numpy(a).to("cuda", non_blocking=False) for a in arrays]
        stream.synchronize()
        g.set_state_device([t.data_ptr() for t in dev])
        sampler = ClockSampler(local_rank)                        # started before the warm-up: nvidia-smi needs ~0.2 s to deliver its first line
        sampler.start()
        sampler.wait_first(3.0)
        g.step(args.warmup, st["cfl"])
        g.sync()
        rep.barrier()
        torch.cuda.synchronize()
        l0 = g.launch_count()
        g.profile(not args.no_kernel_times)      # per-class event pairs; while they record, mf_step launches eagerly (no CUDA-graph replay)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0 = time.perf_counter()
        e0.record(stream)
        g.step(args.steps, st["cfl"])
        e1.record(stream)
        stream.synchronize()
        rep.barrier()
        torch.cuda.synchronize()
        t1 = time.perf_counter()
        clocks = sampler.stop(t0, t1)
        g.profile(False)
        prof = g.profile_read()
        launches = g.launch_count() - l0
        elapsed_ms = rep.max(e0.elapsed_time(e1))
        status = g.sync()
        value = rep.sum(cells * args.steps) / (elapsed_ms * 1e-3)

        # ---- end to end through the C ABI with HOST buffers: H2D of the step's input and D2H of its result inside the timed region
        pin_in = [torch.from_numpy(a).pin_memory() for a in arrays]
        pin_out = [torch.empty_like(t).pin_memory() for t in pin_in]
        np_in = [t.numpy() for t in pin_in]
        np_out = [t.numpy() for t in pin_out]
        e2e_steps = max(1, min(args.steps, args.e2e_steps))
        for _ in range(2):
            g.set_state(*np_in); g.step(1, st["cfl"]); g.get_state(out=np_out)
        rep.barrier()
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        for _ in range(e2e_steps):
            g.set_state(*np_in)
            g.step(1, st["cfl"])
            g.get_state(out=np_out)
        torch.cuda.synchronize()
        e2e_s = rep.max(time.perf_counter() - w0)
        e2e_value = rep.sum(cells * e2e_steps) / e2e_s

        # ---- the same end-to-end work streamed through three contexts (mf_set_state_async / mf_step / mf_get_state_async, one stream each):
        # every step still uploads its input and downloads its result inside the timed region, but the upload of step i+1, the kernels of
        # step i and the download of step i-1 overlap (PCIe is full duplex) - the event-by-event use the paper builds its code for.
        e2e_pipe = None
        if not args.no_e2e_pipeline and 3 * g.memory_bytes() < 120e9:
            ctxs = [g]
            for _ in range(2):
                c2 = MustaForce(nx, ny, nz, dx=st["dx"], path=args.path, eos_table=eos_table, batch=nbatch if nbatch > 1 else None,
                                state_bits=32 if args.state == "f32" else 64, **sch)
                if "jet" in st:
                    c2.set_jet_source(j["dEdx"], j["sigma"], j["x0"], j["y0"], j["z0"])
                ctxs.append(c2)
            g.set_stream(None)                                            # back to its own stream: three contexts, three streams
            outs = [np_out] + [[torch.empty_like(t).pin_memory().numpy() for t in pin_in] for _ in range(2)]
            n_pipe = max(6, 3 * e2e_steps)
            for i in range(3):                                            # warm-up: allocates each context's scratch
                ctxs[i].set_state_async(*np_in); ctxs[i].step(1, st["cfl"]); ctxs[i].get_state_async(outs[i])
            for c2 in ctxs:
                c2.sync()
            rep.barrier()
            torch.cuda.synchronize()
            w0 = time.perf_counter()
            for i in range(n_pipe):
                c2 = ctxs[i % 3]
                c2.sync()                                                 # its previous result is complete; its buffers are free again
                c2.set_state_async(*np_in)
                c2.step(1, st["cfl"])
                c2.get_state_async(outs[i % 3])
            for c2 in ctxs:
                c2.sync()
            torch.cuda.synchronize()
            pipe_s = rep.max(time.perf_counter() - w0)
            same = all(np.array_equal(a, b) for a, b in zip(outs[0], outs[1])) and all(np.array_equal(a, b) for a, b in zip(outs[0], outs[2]))
            e2e_pipe = {"value": rep.sum(cells * n_pipe) / pipe_s, "unit": UNIT, "steps": n_pipe, "contexts": 3, "results_identical": bool(same),
                        "note": "mf_set_state_async + mf_step(1) + mf_get_state_async per step, round-robin over three contexts on their own streams: "
                                "upload, kernels and download of consecutive steps overlap; same bytes per step as the sequential figure"}
            for c2 in ctxs[1:]:
                c2.close()

    if rank != 0:
        rep.close()
        return

    pk = peaks()
    pred_on = sch.get("predictor", True)
    state_bytes = 4 if args.state == "f32" else 8
    table = args.eos == "table"
    slots_cu, slots_L, slots_musta = alg_slots(sch["limiter"], sch["k_stages"], sch["rk"], ndim, pred_on, table=table)
    slots_cu_min = alg_slots(sch["limiter"], sch["k_stages"], sch["rk"], ndim, pred_on, minimal=True, table=table)[0]
    alu_peak_slots = 148 * FP64_LANES_PER_SM * pk["sm_max_mhz"] * 1e6          # FP64 instructions/s, all SMs
    # dominant kernel, from the event pairs recorded around every launch inside the timed region
    work = class_work(g.path(), sch["limiter"], sch["k_stages"], ndim, nx > 1, pred_on, state_bytes, table)
    kernels = {}
    for name, (ms, groups) in prof.items():
        if name not in work or groups == 0:
            continue
        slots, nbytes = work[name]
        t = ms / groups * 1e-3                                              # one launch group = this class's launches of one RK stage
        t_alu, t_hbm = slots * cells / alu_peak_slots, nbytes * cells / (pk["hbm_gbs"] * 1e9)
        if t_alu >= t_hbm:
            ach, peak, unit, bound = 2.0 * slots * cells / t / 1e12, 2.0 * alu_peak_slots / 1e12, "TFLOP/s", "alu"
        else:
            ach, peak, unit, bound = nbytes * cells / t / 1e9, pk["hbm_gbs"], "GB/s", "hbm"
        kernels[name] = {"bound": bound, "achieved": ach, "peak": peak, "unit": unit, "frac": ach / peak, "traffic": None,
                         "kernel": name, "launch_ms": ms / groups, "share_of_step": ms / elapsed_ms,
                         "alg_slots_per_cell": slots, "alg_bytes_per_cell": nbytes}
    # DRAM traffic per launch group: only from a committed ncu --set full capture of this same workload, path and state precision
    dram_step = None
    if (nx, ny, nz) == (256, 256, 256) and sch["k_stages"] == 3 and sch["rk"] == 3 and nbatch == 1 and args.eos == "cs2" and \
            state_bytes == 8 and (g.path(), bool(pred_on)) in NCU_TRAFFIC_256:
        source, table = NCU_TRAFFIC_256[(g.path(), bool(pred_on))]
        for name, gb in table.items():
            if name in kernels:
                kernels[name]["traffic"] = gb * 1e9
                kernels[name]["traffic_source"] = source + " (one ncu --set full capture of this workload and path; not measured in this run)"
        if all(name in kernels or name == "cfl" for name in prof if prof[name][1]) and all(k_ in table for k_ in kernels):
            dram_step = sch["rk"] * sum(table.values()) * 1e9
    # the dominant kernel class = the one with the largest share of the timed region
    roof = max(kernels.values(), key=lambda r: r["share_of_step"]) if kernels else None
    if roof:
        roof = dict(roof, note="alu: FMA-equivalent flops = 2 x algorithmic FP64 issue slots (div = sqrt = 8 slots), peak = 2 x 148 SM x 64 "
                               "lanes x clocks.max.sm; hbm: algorithmic bytes of that kernel / measured copy bandwidth; launch_ms is one "
                               "launch group (the class's launches of one RK stage) from CUDA-event pairs on the library's stream")
    step_frac_alu = (slots_cu * cells * args.steps / (elapsed_ms * 1e-3)) / alu_peak_slots
    step_frac_alu_min = (slots_cu_min * cells * args.steps / (elapsed_ms * 1e-3)) / alu_peak_slots
    step_frac_hbm = (alg_bytes(sch["rk"], state_bytes) * cells * args.steps / (elapsed_ms * 1e-3)) / (pk["hbm_gbs"] * 1e9)
    probe = binding.probe_fp64()
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic",
            "config": describe(st, {"path": g.path(), "l2": "state registers (%.0f MB each) exceed the 126 MB L2" % (40e-6 * cells)
                                    if 40 * cells > 126e6 else "state fits in L2 (small grid)", "parallelism": "replicas x%d" % world,
                                    "batch": "%d events per launch (mf_create_batch), each on its own dt" % nbatch if nbatch > 1 else "single event",
                                    "state": "fp64 state registers" if state_bytes == 8 else
                                    "single-precision STATE (PAPER.md:250, reading A19; arithmetic and scratch stay fp64) - outside "
                                    "BASELINE.json's fp64 contract, reported beside the headline, never as it",
                                    "status": status, "eos": "p = e/3 (closed-form con2prim)" if args.eos == "cs2" else
                                    "tabulated crossover p(e,n), Newton con2prim (roofline: 201 slots per flux evaluation = 16 + one speed solve of ~185 FP64 "
                                    "instructions, one full table evaluation per solve measured with the counting build; the kernels are bound by "
                                    "instruction issue - fp32 seed, table addressing, call overhead - not by the FP64 pipe)"}),
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": 40 * cells, "d2h_bytes_per_step": 40 * cells,
                    "steps": e2e_steps, "note": "mf_set_state(host) + mf_step(1) + mf_get_state(host) per step, pinned host buffers, strictly one "
                    "after the other (the conservative figure)", "pipelined": e2e_pipe},
            "gpu_launches": launches,
            "roofline": roof,
            "roofline_kernels": kernels,
            "roofline_step": {"alg_slots_per_cell_update": slots_cu, "alg_bytes_per_cell_update": alg_bytes(sch["rk"], state_bytes),
                              "frac_alu": step_frac_alu, "frac_hbm": step_frac_hbm, "hbm_peak": pk["hbm_source"],
                              "alg_slots_minimal_per_cell_update": slots_cu_min, "frac_alu_minimal": step_frac_alu_min,
                              "slots_note": "frac_alu counts divide = square root = 8 slots and 32 per flux evaluation (SURVEY.md 8(d), the "
                                            "frozen denominator); frac_alu_minimal counts the sequences the product code issues (reciprocal 3, "
                                            "root 6, flux 24) and is the figure to read as FP64-pipe utilisation of useful work",
                              "dram_bytes_per_step": dram_step,
                              "dram_over_alg_bytes": (dram_step / (alg_bytes(sch["rk"], state_bytes) * cells)) if dram_step else None,
                              "measured_dfma_per_s": probe["dfma_per_s"], "measured_rcp_slots": probe["dfma_per_s"] / probe["rcp_per_s"],
                              "measured_sqrt_slots": probe["dfma_per_s"] / probe["sqrt_per_s"]},
            "kernels_ms": {k: {"ms_total": v[0], "groups": v[1]} for k, v in prof.items()}}
    if not args.no_cpu_baseline and world == 1:
        line["cpu_baseline"] = cpu_baseline(st, crop=args.ref_crop)
    print(json.dumps(line), flush=True)
    rep.close()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3, help="BASELINE.json config 1..5 (default 3 = the 256^3 metric workload)")
    ap.add_argument("--grid", default=None, help="nz,ny,nx override (parity/debug sizes)")
    ap.add_argument("--path", default="auto", choices=["auto", "staged", "fused", "hybrid", "sweep", "small"])
    ap.add_argument("--eos", default="cs2", choices=["cs2", "table"], help="table: synthetic crossover p(e,n) table with Newton con2prim")
    ap.add_argument("--predictor", default="on", choices=["on", "off"], help="off: without the Hancock half step (reading A4), reported beside the default")
    ap.add_argument("--k", type=int, default=None, help="override the number of MUSTA stages (e.g. 4: the paper's own setting, PAPER.md:256)")
    ap.add_argument("--limiter", default=None, choices=["none", "minmod", "superbee", "vanalbada", "vanleer", "mc", "first"])
    ap.add_argument("--rk", type=int, default=None, choices=[2, 3])
    ap.add_argument("--state", default="f64", choices=["f64", "f32"],
                    help="f32: single-precision stored state (PAPER.md:250, reading A19), staged path; not the headline")
    ap.add_argument("--batch", type=int, default=1, help="events per context (mf_create_batch); config 4: the seeded events 0..B-1")
    ap.add_argument("--e2e-steps", type=int, default=5)
    ap.add_argument("--ref-crop", type=int, default=64, help="edge of the centred crop the CPU oracle is timed on")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e-pipeline", action="store_true", help="skip the three-context streamed end-to-end leg")
    ap.add_argument("--no-kernel-times", action="store_true",
                    help="no per-kernel-class event pairs inside the timed region: mf_step then replays captured steps (CUDA graph), which is "
                         "what a user's plain mf_step(n) call does; the roofline objects need the pairs and are null")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
