#!/usr/bin/env python
"""bench.py -- throughput of the nodal-DG hot path (libdg, CUDA) on BASELINE.json's workloads.

    python bench.py [--gpus N] [--steps K] [--warmup W]      # config 2 headline + the N = 1..10 x 2 sweep (one JSON line)
    python bench.py --config 3|5 | --config 4 --N deg --model m [--no-sweep]
    python bench.py --integrator ab3                           # the paper's own time stepping (eq. (4)): one r_k per step
    python bench.py --impl reference ...                       # the fp64 oracle on the host cores, same metric
    python bench.py --sweep                                    # config 4 only: every degree, both models -> JSON lines

A "step" is one LSRK(5,4) time step = five fused stage kernels, each of which runs every row of the hot path (volume +
surface + lift + update) over all K elements.  The metric is node-updates per second per RK stage: K*Np*5*steps / time.

Timed region: W untimed warm-up steps, then R (--repeats, default 5) back-to-back runs of EXACTLY K steps, each bracketed
by CUDA events on the launching stream, the whole region by barrier + synchronize; the reported time is the MEDIAN run
(all R are listed), max over ranks.  `rhs_ms` is a single dg_rhs evaluation timed the same way.  The state arrays
(3 x K*Nf*Np floats, 1 GB for config 2) are larger than the 126 MB L2, so no explicit flush is needed.
BASELINE.json's metric is "... vs N ... for every degree N = 1..10": the default single-GPU run therefore also times the
config-4 sweep (one mesh per degree with K Np ~ 2.5e7, both models, the kernel `auto` picks) and reports it as
`roofline.sweep` (compact rows, columns in `roofline.sweep_columns`), each row with its own clock reading.
Multi-GPU (--gpus N under torchrun): the path has no exchange step in scope: N independent
replicas, weak scaling, no data-path collective; the sweep runs at N = 1 only.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1602_07997_b200 import workloads as W  # noqa: E402

METRIC = "node-updates/s per RK stage"
UNIT = "node-updates/s"
FP32_PEAK_TFLOPS = 72.3      # measured FFMA micro-benchmark on this pool's B200; nominal 74.5
HBM_FALLBACK_GBS = 6650.0    # B200_PROFILING.md fallback


def flops_per_element(model: int, N: int, with_update: bool = True) -> float:
    """Algorithmic flops per element per RK stage (FMA = 2)."""
    Np, Nfp = (N + 1) * (N + 2) * (N + 3) // 6, (N + 1) * (N + 2) // 2
    if model == W.ACOUSTIC:
        f = 12 * Np * Np + 32 * Np * Nfp + 52 * Np + 80 * Nfp
        return f - (0 if with_update else 16 * Np)
    f = 36 * Np * Np + 72 * Np * Nfp + 150 * Np + 400 * Nfp
    return f - (0 if with_update else 36 * Np)


def bytes_per_element(model: int, N: int, integrator: str = "lsrk") -> float:
    """Compulsory HBM bytes per element per fused stage: the state arrays -- LSRK: read q, res and
    write q, res = 16 B per value, except in the first stage of a step (A_1 = 0: res is not read, 12 B), i.e. 15.2 B on
    average over the five stages; AB3: read q, r^-1, r^-2, write q, r^0 = 20 B -- plus the per-element constants the
    method needs: 9 g^vol + 16 face (n, g^sur) + 2 | 3 material values = 108 | 112 B, plus 16 B of compressed
    connectivity.  (The records as built are padded to 128 | 192 B: `bytes_as_built`.)"""
    Np = (N + 1) * (N + 2) * (N + 3) // 6
    Nf = W.NFIELDS[model]
    per_value = 15.2 if integrator == "lsrk" else 20.0
    return per_value * Nf * Np + (108 if model == W.ACOUSTIC else 112) + 16


def bytes_as_built(model: int, N: int, integrator: str = "lsrk") -> float:
    Np = (N + 1) * (N + 2) * (N + 3) // 6
    per_value = 15.2 if integrator == "lsrk" else 20.0
    return per_value * W.NFIELDS[model] * Np + (128 if model == W.ACOUSTIC else 192) + 20


def measured_peaks():
    """(HBM GB/s, dense bf16 TFLOP/s sustained, source).  The stage kernels run back to back inside a long
    step, so the sustained tensor figure is the one that applies (B200_PROFILING.md)."""
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), float(d.get("bf16_tflops_sustained", d.get("bf16_tflops", 1400.0))), "measured"
    return HBM_FALLBACK_GBS, 1400.0, "fallback"


def pick_workload(a) -> W.Workload:
    if a.config == 4:
        w = W.config(4, N=a.N or 5, model=W.ELASTIC if a.model == "elastic" else W.ACOUSTIC)
    else:
        w = W.config(a.config)
    if a.cells:
        w = W.config(a.config, N=a.N or 5, model=W.ELASTIC if a.model == "elastic" else W.ACOUSTIC, n=a.cells) \
            if a.config == 4 else W.config(a.config, n=a.cells)
    return w


class ClockSampler:
    """nvidia-smi clocks/throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "20",
                                          "-i", str(index)], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
            t0 = time.time()                 # nvidia-smi can take longer to start than the timed region lasts
            while not self.rows and time.time() - t0 < 10.0 and self.proc.poll() is None:
                time.sleep(0.01)
        except OSError:
            self.proc = None
        self.first = 0

    def mark(self):
        """Start of the timed region: earlier rows are dropped (the last one is kept as a fallback)."""
        self.first = len(self.rows)

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def window(self):
        """Statistics of the rows since the last mark(); the sampler keeps running."""
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = self.rows[self.first:] or self.rows[-1:]
        for r in rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            try:
                pw.append(float(r[2]))
            except (ValueError, IndexError):
                pass
            for nme, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_min_mhz": min(sm) if sm else None,
                "sm_max_mhz": max(mx) if mx else None, "power_w": statistics.median(pw) if pw else None,
                "samples": len(sm), "reasons": sorted(reasons)}

    def stop(self):
        if not self.proc:
            return self.window()
        time.sleep(0.15)
        self.proc.terminate()
        self.t.join(timeout=2)
        return self.window()


# ------------------------------------------------------------------------------------------------
def oracle_sample_run(w: W.Workload, nsteps: int, sample_elems: int, threads: int | None = None):
    """Time the fp64 oracle (as it stands) on a bounded sample of the workload: one LSRK step =
    five evaluations of r_k on `sample_elems` elements of the full-size mesh plus the update on
    those elements.  `threads` limits the BLAS pool (1 = single-threaded).  Returns (seconds per step, threads,
    description, elements)."""
    from oracle import mesh as omesh
    from oracle import physics, refelem, timestep
    try:
        from threadpoolctl import threadpool_info, threadpool_limits
    except Exception:                                   # noqa: BLE001
        threadpool_info = threadpool_limits = None
    ref = refelem.build(w.N)
    vxyz, etov, bc, cell = w.mesh()
    mats = w.material_arrays(cell)
    K = etov.shape[0]
    sample = np.arange(min(sample_elems, K))
    m = omesh.build(ref, vxyz, etov, bc, only_elems=sample)
    # neighbours of the sample may lie outside it: they are read from the global state, never updated
    q = w.initial_fields(m.x).astype(np.float32).astype(np.float64)
    dt = timestep.stable_dt(ref, m, mats[1])
    if w.model == W.ACOUSTIC:
        rhs = lambda qq: physics.rhs_acoustic(ref, m, mats[0], mats[1], qq, sample)          # noqa: E731
    else:
        rhs = lambda qq: physics.rhs_elastic(ref, m, *mats, qq, sample)                      # noqa: E731
    res = np.zeros((len(sample),) + q.shape[1:])
    times = []

    def loop():
        for _ in range(nsteps):
            t0 = time.perf_counter()
            for A, B in zip(timestep.LSRK_A, timestep.LSRK_B):
                res[...] *= A
                res[...] += dt * rhs(q)
                q[sample] += B * res
            times.append(time.perf_counter() - t0)

    if threads is not None and threadpool_limits is not None:
        with threadpool_limits(limits=threads):
            loop()
        used = threads
    else:
        loop()
        used = os.cpu_count() or 1
        if threadpool_info is not None:
            used = max([p.get("num_threads", 1) for p in threadpool_info()] or [1])
    desc = (f"{len(sample)} of {K} elements of {w.name}, {nsteps} LSRK step(s) = {5 * nsteps} r_k evaluations + updates, "
            f"numpy fp64, {used} thread(s)")
    return times, used, desc, len(sample)


def run_reference(a):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    w = pick_workload(a)
    per_stage_flop = flops_per_element(w.model, w.N)
    sample_elems = a.sample or max(256, int(2.0e9 / per_stage_flop / 5))     # ~2 GFLOP per r_k evaluation
    steps = max(1, a.steps)
    times, threads, desc, ns = oracle_sample_run(w, a.warmup + steps, sample_elems)
    tt = times[a.warmup:]
    sec = sum(tt) / len(tt)
    value = ns * w.Np * 5 / sec
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": a.gpus, "steps": steps, "warmup": a.warmup,
        "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": w.name, "K": w.K, "N": w.N, "Np": w.Np, "stages_per_step": 5,
                                        "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "net_gflops": ns * per_stage_flop * 5 / sec * 1e-9,
    }
    print(json.dumps(line))
    return 0


def max_over_ranks(values_ms, device, world):
    """Device-timed durations of one replica each -> the slowest rank's (every rank gets the same numbers)."""
    import torch
    import torch.distributed as dist
    t = torch.tensor(list(values_ms), device=device, dtype=torch.float64)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(world, nodes_per_replica, stages, ms):
    """node-updates/s per RK stage summed over `world` independent replicas (weak scaling), timed by the slowest one."""
    return world * nodes_per_replica * stages / (ms * 1e-3)


# ------------------------------------------------------------------------------------------------
def roofline_of(variant_name, model, N, K, t_stage, integrator="lsrk"):
    """Roofline object for one stage kernel launch of duration t_stage (seconds) over K elements."""
    flops = flops_per_element(model, N) * K
    byts = bytes_per_element(model, N, integrator) * K
    hbm_peak, bf16_peak, which = measured_peaks()
    tensor = variant_name.startswith("tc_")
    # compute roof of the kernel that ran: FP32 FFMA peak for the SIMT kernels; for the tcgen05 kernel one
    # fp32-equivalent MAC costs six bf16 MMAs (BF16x3 split): bf16 peak / 6
    comp_peak = bf16_peak / 6.0 if tensor else FP32_PEAK_TFLOPS
    comp_src = (f"MEASURED_PEAKS.json bf16 sustained ({which}) / 6 (BF16x3 split)" if tensor
                else "FFMA micro-benchmark, measured (DESIGN.md)")
    frac_comp = flops / t_stage / (comp_peak * 1e12)
    frac_hbm = byts / t_stage / (hbm_peak * 1e9)
    fp32_frac = flops / t_stage / (FP32_PEAK_TFLOPS * 1e12)      # the roof north_star names; > 1 is legitimate on the tensor path
    if flops / (comp_peak * 1e12) >= byts / (hbm_peak * 1e9):      # which roof binds the algorithm on this kernel
        roof = {"bound": "tensor" if tensor else "alu", "achieved": flops / t_stage * 1e-12, "peak": comp_peak, "unit": "TFLOP/s",
                "frac": frac_comp, "peak_source": comp_src, "hbm_frac": frac_hbm, "hbm_gbs": byts / t_stage * 1e-9}
    else:
        roof = {"bound": "hbm", "achieved": byts / t_stage * 1e-9, "peak": hbm_peak, "unit": "GB/s", "frac": frac_hbm,
                "peak_source": f"MEASURED_PEAKS.json ({which})", "compute_frac": frac_comp,
                "compute_tflops": flops / t_stage * 1e-12, "compute_peak": comp_peak, "compute_peak_source": comp_src}
    roof["fp32_roof_frac"] = fp32_frac
    roof["fp32_roof_tflops"] = FP32_PEAK_TFLOPS
    roof["bytes_per_element"] = bytes_per_element(model, N, integrator)
    roof["bytes_per_element_as_built"] = bytes_as_built(model, N, integrator)
    roof["flops_per_element"] = flops_per_element(model, N)
    roof["kernel"] = variant_name
    return roof


def time_runs(torch, ctx, d_q, dt, steps, repeats, stream, integrator="lsrk", flush=None):
    """`repeats` back-to-back runs of `steps` time steps, each bracketed by CUDA events on `stream`; returns the list of
    durations in ms and the launches of one run.  `flush`: a device buffer larger than L2, rewritten before every run
    (for workloads whose state would otherwise stay L2-resident from one run to the next)."""
    sptr = stream.cuda_stream
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(repeats)]
    launches = 0
    for e0, e1 in evs:
        if flush is not None:
            flush.add_(1)
        e0.record(stream)
        if integrator == "lsrk":
            ctx.run(d_q.data_ptr(), dt, steps, sptr)
            launches = ctx.last_launch_count
        else:
            ctx.ab3_run(d_q.data_ptr(), dt, steps, sptr)
            launches = ctx.last_launch_count
        e1.record(stream)
    torch.cuda.synchronize()
    return [e0.elapsed_time(e1) for e0, e1 in evs], launches


def time_rhs(torch, ctx, d_q, repeats, stream):
    d_r = torch.empty_like(d_q)
    sptr = stream.cuda_stream
    ctx.rhs(d_q.data_ptr(), d_r.data_ptr(), sptr)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(repeats)]
    for e0, e1 in evs:
        e0.record(stream)
        ctx.rhs(d_q.data_ptr(), d_r.data_ptr(), sptr)
        e1.record(stream)
    torch.cuda.synchronize()
    return statistics.median(e0.elapsed_time(e1) for e0, e1 in evs)


SWEEP_COLUMNS = ["model", "N", "K", "kernel", "ms_per_stage", "Gnode_updates_per_s", "net_tflops", "bound", "frac",
                 "hbm_frac", "fp32_roof_frac", "rhs_ms", "sm_mhz", "throttle"]


def sweep_rows(torch, dg, device, sampler, steps=5, warmup=3, repeats=5, degrees=range(1, 11), log=None, cfg=4):
    """Config 4: one mesh per degree (K Np ~ 2.5e7), both models, the kernel `auto` picks; compact rows (SWEEP_COLUMNS).
    cfg = 6: the paper's own size (N = 1..8, ~2 M nodes per mesh); there the state (96 | 216 MB) is of the
    size of the L2, so the L2 is flushed before every timed run."""
    rows = []
    stream = torch.cuda.current_stream()
    flush = torch.zeros(96 * 1024 * 1024, dtype=torch.float32, device="cuda") if cfg == 6 else None     # 384 MB > L2
    for N in degrees:
        mesh = None
        for model in (W.ACOUSTIC, W.ELASTIC):
            w = W.config(cfg, N=N, model=model)
            if mesh is None:
                mesh = w.mesh()                      # the mesh depends on the degree only
            vxyz, etov, bc, cell = mesh
            mats = w.material_arrays(cell)
            ctx = dg.Context(vxyz, etov, w.N, w.model, mats[0], mats[1], mats[2] if model == W.ELASTIC else None, bc, device=device)
            q0 = w.initial_fields(ctx.node_coords()).astype(np.float32)
            dt = float(np.float32(ctx.stable_dt(0.5)))
            d_q = torch.from_numpy(q0).cuda()
            del q0
            ctx.run(d_q.data_ptr(), dt, warmup, stream.cuda_stream)
            torch.cuda.synchronize()
            if sampler:
                sampler.mark()
            ms_list, _ = time_runs(torch, ctx, d_q, dt, steps, repeats, stream, flush=flush)
            clocks = sampler.window() if sampler else {"sm_mhz": None, "reasons": []}
            rhs_ms = time_rhs(torch, ctx, d_q, repeats, stream)
            assert torch.isfinite(d_q).all().item(), f"state blew up at N = {N}"
            t_stage = statistics.median(ms_list) * 1e-3 / (5 * steps)
            roof = roofline_of(ctx.variant_name, model, N, w.K, t_stage)
            kern = ctx.variant_name.split("<")[0]
            bad = [r for r in clocks["reasons"] if r != "sw_power_cap"]
            rows.append(["ac" if model == W.ACOUSTIC else "el", N, w.K, kern, round(t_stage * 1e3, 4),
                         round(w.K * w.Np / t_stage * 1e-9, 2), round(flops_per_element(model, N) * w.K / t_stage * 1e-12, 2),
                         roof["bound"], round(roof["frac"], 3), round(roof.get("hbm_frac", roof["frac"]), 3),
                         round(roof["fp32_roof_frac"], 3), round(rhs_ms, 4), clocks["sm_mhz"],
                         ",".join(clocks["reasons"]) if clocks["reasons"] else "none"])
            if log:
                log(rows[-1] + (["REJECT: " + ",".join(bad)] if bad else []))
            ctx.close()
            del d_q
            torch.cuda.empty_cache()
    return rows


def run_ours(a):
    import torch
    import torch.distributed as dist
    from paper_1602_07997_b200 import dg           # raises if libdg.so is missing: no fallback

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product path has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = pick_workload(a)
    opts = {}
    if a.E:
        opts["elems_per_thread"] = a.E
    if a.G:
        opts["groups_per_cta"] = a.G
    if a.variant:
        opts["variant"] = a.variant
    if a.surface == "interface":
        opts["surface"] = 1
    ctx = dg.from_workload(w, device=local, **opts)
    xyz = ctx.node_coords()
    q0 = w.initial_fields(xyz).astype(np.float32)
    del xyz
    ab3 = a.integrator == "ab3"
    # AB3's stability region reaches -0.55 on the real axis against about -4.7 for LSRK(5,4): CFL 0.05 instead of 0.5
    dt = float(np.float32(ctx.stable_dt(0.05 if ab3 else 0.5)))
    h_q = torch.from_numpy(q0).pin_memory()
    d_q = h_q.cuda()
    stream = torch.cuda.current_stream()
    sptr = stream.cuda_stream
    stages_per_step = 1 if ab3 else 5

    def one_step():
        if ab3:
            ctx.ab3_step(d_q.data_ptr(), dt, sptr)
        else:
            ctx.step(d_q.data_ptr(), dt, sptr)

    # ---- device-resident timing
    sampler = ClockSampler(local) if rank == 0 else None      # returns once nvidia-smi delivers rows
    for _ in range(a.warmup):
        one_step()
    barrier()
    if sampler:
        sampler.mark()
    ms_list, launches = time_runs(torch, ctx, d_q, dt, a.steps, a.repeats, stream, a.integrator)
    barrier()
    clocks = sampler.window() if sampler else None
    ms = statistics.median(ms_list)
    assert torch.isfinite(d_q).all().item(), "state blew up"
    rhs_ms = time_rhs(torch, ctx, d_q, a.repeats, stream)

    # ---- end to end through the C ABI with host buffers: H2D of the state, one step, D2H of the state
    e2e_steps = max(1, min(a.steps, 5))
    d_q.copy_(h_q, non_blocking=True)
    if ab3:
        ctx.ab3_reset(sptr)
    one_step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    h_out = torch.empty_like(h_q).pin_memory()
    e0.record(stream)
    for _ in range(e2e_steps):
        d_q.copy_(h_q, non_blocking=True)
        one_step()
        h_out.copy_(d_q, non_blocking=True)
    e1.record(stream)
    barrier()
    ms_e2e = e0.elapsed_time(e1)

    ms, ms_e2e, rhs_ms = max_over_ranks([ms, ms_e2e, rhs_ms], "cuda", world)

    nodes = w.K * w.Np
    stages = stages_per_step * a.steps
    value = whole_job_value(world, nodes, stages, ms)
    flops = flops_per_element(w.model, w.N) * w.K
    t_stage = ms * 1e-3 / stages                          # average stage-kernel duration (copy: <1/(5K) of it)
    roof = roofline_of(ctx.variant_name, w.model, w.N, w.K, t_stage, a.integrator)
    tensor = ctx.variant_name.startswith("tc_")
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    # the first run after the (idle) set-up runs at full boost, the later ones under the board's power cap: both are shown
    t_first = ms_list[0] * 1e-3 / stages
    first = roofline_of(ctx.variant_name, w.model, w.N, w.K, t_first, a.integrator)
    roof["first_run"] = {"ms_per_stage": t_first * 1e3, "frac": first["frac"], "note": "first of the timed runs (boost clocks); "
                         "`frac` above is the median run (sustained, power-capped)"}
    roof["traffic"] = None
    if os.path.exists(tpath) and not ab3:
        roof["traffic"] = json.load(open(tpath)).get(w.name + (":tc" if tensor else ":simt"))
    line = {
        "metric": METRIC if not ab3 else "node-updates/s per AB3 time step", "value": value, "unit": UNIT, "n_gpus": world,
        "steps": a.steps, "warmup": a.warmup, "ms_per_step": ms / a.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None,
        "dtype": "f32 (bf16x3 split on tcgen05, fp32 accumulate)" if tensor else "f32",
        "data": "synthetic",
        "config": {"workload": w.name, "model": "acoustic" if w.model == W.ACOUSTIC else "elastic", "K": w.K, "N": w.N,
                   "Np": w.Np, "stages_per_step": stages_per_step, "integrator": a.integrator, "l2": "inputs larger than L2",
                   "replicas": world, "dt": dt, "repeats": a.repeats, "timing": "median of repeats, each exactly `steps` steps"},
        "net_gflops": world * flops * stages / (ms * 1e-3) * 1e-9,
        "ms_per_stage": t_stage * 1e3,
        "ms_per_step_repeats": [round(x / a.steps, 5) for x in ms_list],
        "rhs_ms": rhs_ms,
        "gpu_launches": launches * a.repeats,
        "clocks": clocks,
        "roofline": roof,
        "e2e": {"value": world * nodes * stages_per_step * e2e_steps / (ms_e2e * 1e-3), "unit": UNIT,
                "h2d_bytes_per_step": int(h_q.numel() * 4), "d2h_bytes_per_step": int(h_q.numel() * 4),
                "steps": e2e_steps, "ms_per_step": ms_e2e / e2e_steps},
    }
    ctx.close()
    del d_q, h_out
    torch.cuda.empty_cache()
    if rank == 0:
        if world == 1 and not a.no_sweep and not ab3 and a.config == 2 and not a.variant and a.surface == "element":
            log = (lambda r: print("sweep " + json.dumps(r), file=sys.stderr, flush=True))
            roof["sweep_columns"] = SWEEP_COLUMNS
            roof["sweep"] = sweep_rows(torch, dg, local, sampler, steps=a.sweep_steps, repeats=a.repeats, log=log)
            roof["paper_sized"] = sweep_rows(torch, dg, local, sampler, steps=a.sweep_steps, repeats=a.repeats, degrees=range(1, 9),
                                             log=log, cfg=6)
            roof["paper_sized_note"] = ("the paper's own size, PAPER.md:225: N = 1..8, ~2 M nodes per mesh (same columns); state "
                                        "~ L2 size, L2 flushed before each timed run of 5 steps")
            roof["sweep_note"] = (f"config 4, K Np ~ 2.5e7 per degree, auto variant, median of {a.repeats} runs of {a.sweep_steps} steps; "
                                  "frac = fraction of the binding roof (hbm: measured copy bandwidth; tensor: bf16 sustained / 6; "
                                  "alu: 72.3 TFLOP/s FFMA), fp32_roof_frac = net flops / 72.3 TFLOP/s")
        if sampler:
            sampler.stop()
        if not a.no_cpu and world == 1:
            per_stage_flop = flops_per_element(w.model, w.N)
            sample_elems = a.sample or max(256, int(2.0e9 / per_stage_flop / 5))
            times, threads, desc, ns = oracle_sample_run(w, 6, sample_elems)      # ~10 s of CPU work; the first step is warm-up
            sec = statistics.mean(times[1:])
            line["cpu_baseline"] = {"value": ns * w.Np * 5 / sec, "unit": UNIT, "cores": threads, "kind": "oracle",
                                    "sample": desc, "net_gflops_fp64": ns * per_stage_flop * 5 / sec * 1e-9}
            t1, _, d1, n1 = oracle_sample_run(w, 4, max(128, sample_elems // 4), threads=1)
            line["cpu_baseline"]["single_thread"] = {"value": n1 * w.Np * 5 / statistics.mean(t1[1:]), "unit": UNIT, "cores": 1, "sample": d1}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_sweep(a):
    """Config 4 only: every degree, both models; one JSON line per (model, N)."""
    import torch
    from paper_1602_07997_b200 import dg
    torch.cuda.set_device(0)
    sampler = ClockSampler(0)
    degrees = [a.N] if a.N else (range(1, 9) if a.paper_size else range(1, 11))
    rows = sweep_rows(torch, dg, 0, sampler, steps=a.sweep_steps, repeats=a.repeats, degrees=degrees, cfg=6 if a.paper_size else 4,
                      log=lambda r: print(json.dumps(dict(zip(SWEEP_COLUMNS + ["note"], r))), flush=True))
    sampler.stop()
    return 0 if rows else 1


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--repeats", type=int, default=5, help="timed runs of `steps` steps; the median is reported")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--N", type=int, default=None)
    ap.add_argument("--model", default="acoustic", choices=["acoustic", "elastic"])
    ap.add_argument("--integrator", default="lsrk", choices=["lsrk", "ab3"])
    ap.add_argument("--cells", type=int, default=None, help="override cells per side (reduced sizes)")
    ap.add_argument("--sample", type=int, default=None, help="elements in the oracle's timed sample")
    ap.add_argument("--E", type=int, default=0)
    ap.add_argument("--G", type=int, default=0)
    ap.add_argument("--variant", type=int, default=0, help="0 auto, 1 FP32 SIMT family, 4 pipelined tcgen05 BF16x3 kernel, 5 FP32 SIMT row-per-thread kernel (N <= 3)")
    ap.add_argument("--surface", default="element", choices=["element", "interface"],
                    help="interface: the paper's interface-centric surface kernel feeds the stage kernel (dg_options.surface = 1)")
    ap.add_argument("--no-cpu", action="store_true", help="skip the cpu_baseline leg")
    ap.add_argument("--no-sweep", action="store_true", help="skip the config-4 degree sweep of the default run")
    ap.add_argument("--sweep-steps", type=int, default=5)
    ap.add_argument("--sweep", action="store_true", help="config-4 sweep only, one JSON line per (model, N)")
    ap.add_argument("--paper-size", action="store_true", help="with --sweep: the paper's own size (N = 1..8, ~2 M nodes per mesh)")
    a = ap.parse_args()
    if a.warmup < 3 and a.impl == "ours":
        a.warmup = 3
    a.repeats = max(a.repeats, 1)
    if a.sweep:
        return run_sweep(a)
    if a.impl == "reference":
        return run_reference(a)
    return run_ours(a)


if __name__ == "__main__":
    sys.exit(main())
