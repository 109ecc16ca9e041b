#!/usr/bin/env python
"""bench.py -- throughput of the sledge hot path on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload C3] [--impl sledge|reference]

A "step" is one pass of the whole hot path over the workload: sledge_rk_step (per RK stage: ghost fill +
fused Laplacian/potential/RK-stage kernel; with AMR: subcycling + average-down) followed by
sledge_tag_strings (winding tags + per-32^3 block counts).  Metric: cell-updates per second per RK stage,
`value` = valid cell-stage updates of all levels per step / step time.  Inputs are seeded synthetic
fields (paper_2404_02950_b200.inputs); every state buffer is far larger than L2, so no flush is needed.
Multi-GPU: the path does not shard in this build ("replicas only"): every rank runs an independent replica.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "Gcell-updates/s per RK stage"
UNIT = "Gcell-updates/s"
# Nystrom's classical three-stage fourth-order scheme as rkn.nodes / weights_b / weights_bar_b / tableau (L812-815)
RKN4 = dict(nodes=[0.0, 0.5, 1.0], weights_b=[1 / 6, 4 / 6, 1 / 6], weights_bar_b=[1 / 6, 1 / 3, 0.0],
            tableau=[0.0, 1 / 8, 0.0, 0.0, 0.5, 0.0])


def ncu_traffic(workload, flow):
    """mean dram__bytes_read.sum + dram__bytes_write.sum per K1 launch of this workload / data-flow, from the committed
    `ncu --set full` captures (profiles/r02_traffic.csv; commands in profiles/r02_k1_variants.md and
    profiles/r02_ncu_full.md); a constant read from that file, NOT a measurement of this run; None if that workload
    was not captured."""
    import csv
    try:
        rows = [r for r in csv.DictReader(open(os.path.join(ROOT, "profiles", "r02_traffic.csv")))
                if r["workload"] == workload and r["flow"] == flow and "k_rk_" in r["kernel"]]
    except OSError:
        return None
    if not rows:
        return None
    return {"dram_bytes_per_launch": sum(float(r["dram_bytes_per_launch"]) for r in rows) / len(rows),
            "algorithmic_bytes_per_launch": sum(float(r["algorithmic_bytes_per_launch"]) for r in rows) / len(rows),
            "source": "profiles/r02_traffic.csv (ncu --set full, one capture per sweep kernel; constant, not measured in this run)"}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="C3", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--impl", default="sledge", choices=["sledge", "reference"])
    ap.add_argument("--flow", default="fused", choices=["fused", "fused3", "lean", "classic"])
    ap.add_argument("--ko-order", type=int, default=0, choices=[0, 2, 3],
                    help="Kreiss-Oliger dissipation order (Eq.7); 0 = off, as in every BASELINE.json config")
    ap.add_argument("--ko-strength", type=float, default=0.01)
    ap.add_argument("--interp", type=int, default=0, choices=[0, 4],
                    help="coarse->fine ghost interpolation: 0 = trilinear (BASELINE.json config 5), 4 = quartic (L780)")
    ap.add_argument("--integrator", type=int, default=4, choices=[4, 3, 10, 20],
                    help="integrator.type (L808): 4 = RK4 (every BASELINE.json config), 3 / 10 = SSPRK3, 20 = user RKN "
                         "tableau (here: Nystrom's classical three-stage fourth-order scheme)")
    ap.add_argument("--gw", action="store_true",
                    help="also evolve the 12 gravitational-wave auxiliary components of Eq.16 (sim.gravitational_waves)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-graph", action="store_true", help="skip the C1 CUDA-graph replay leg")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-others", action="store_true",
                    help="skip the short runs of the other BASELINE.json workloads (key other_workloads) and the C5 graph leg")
    ap.add_argument("--other-steps", type=int, default=4)
    ap.add_argument("--e2e-steps", type=int, default=0,
                    help="steps of the end-to-end leg (host buffers); 0 = as many as --steps, at least 4 and at most 20")
    return ap.parse_args()


# ---------------------------------------------------------------------------------------------------
# workload construction (shared recipe; no arithmetic of the method here)
# ---------------------------------------------------------------------------------------------------

def hierarchy(cfg):
    from paper_2404_02950_b200 import inputs
    if cfg.n_levels == 1:
        return None, [(0, (0, 0, 0), (cfg.n0 - 1,) * 3)], [1.0]
    ex = cfg.extra
    rings = inputs.make_rings(cfg.n0, ex["n_rings"], ex["rmin"], ex["rmax"], ex["core_w"], cfg.seeds[0])
    boxes, cover = inputs.amr_boxes_for_rings(rings, n_levels=cfg.n_levels, box=ex["box"], r1=ex["r1"], r2=ex["r2"],
                                              blocking_factor=cfg.blocking_factor)
    return rings, boxes, cover


def cells_per_step(cfg, boxes):
    """valid cell-steps per coarse step: level l takes 2^l steps (Eq.3)."""
    tot = 0
    per_level = [0] * cfg.n_levels
    for l, lo, hi in boxes:
        n = (hi[0] - lo[0] + 1) * (hi[1] - lo[1] + 1) * (hi[2] - lo[2] + 1)
        per_level[l] += n
        tot += n * (1 << l)
    return tot, per_level


def initial_fields(cfg, rings, boxes, device, tdtype):
    """yield (box index, comp, tensor on `device`) for psi1, psi2; Pi = 0 is the zero-filled arena."""
    import torch
    from paper_2404_02950_b200 import inputs
    if cfg.n_levels == 1:
        for c, seed in enumerate(cfg.seeds):
            yield 0, c, inputs.grf(cfg.n0, cfg.grf_f, seed, device=device, dtype=tdtype).contiguous()
    else:
        for ib, (l, lo, hi) in enumerate(boxes):
            re, im = inputs.ring_field(rings, l, lo, hi, device=device)
            yield ib, 0, re.to(tdtype).contiguous()
            yield ib, 1, im.to(tdtype).contiguous()


# ---------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------

class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.samples, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        self.th.join(timeout=2)
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in self.samples:
            f = [x.strip() for x in s.split(",")]
            if len(f) < 6:
                continue
            try:
                sm.append(float(f[0]))
                mx = float(f[1])
            except ValueError:
                continue
            for nm, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


# ---------------------------------------------------------------------------------------------------
# CPU oracle leg (cpu_baseline and --impl reference): the oracle as it stands, on a bounded sample
# ---------------------------------------------------------------------------------------------------

def oracle_sample(cfg):
    """A bounded sample of the workload for the CPU oracle: same stencil, dtype-independent fp64 arithmetic,
    same parameters, a periodic 128^3 (64^3 for C1: 32^3) sub-volume cut into 32^3 boxes so that the oracle's
    OpenMP loops over boxes use the host cores; AMR: the same recipe at base 64^3 with 16^3 boxes."""
    from oracle.oracle import Oracle
    from paper_2404_02950_b200 import inputs
    import numpy as np
    if cfg.n_levels == 1:
        n = min(cfg.n0, 128)
        boxes = inputs.split_level0(n, 32)
        o = Oracle(n, boxes=boxes, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam)
        f = [inputs.grf(n, cfg.grf_f, s).numpy() for s in cfg.seeds]
        for ib, (_, lo, hi) in enumerate(boxes):
            for c in range(2):
                o.set_state(ib, c, np.ascontiguousarray(f[c][lo[2]:hi[2] + 1, lo[1]:hi[1] + 1, lo[0]:hi[0] + 1]))
        desc = f"periodic {n}^3 sub-volume of the workload in 32^3 boxes, same stencil and parameters"
        cells = n ** 3
        levels = 1
    else:
        n = 64
        ex = cfg.extra
        rings = inputs.make_rings(n, 3, 8.0, 16.0, ex["core_w"], cfg.seeds[0])
        boxes, _ = inputs.amr_boxes_for_rings(rings, n_levels=3, box=16, r1=4.0, r2=1.0, blocking_factor=8)
        o = Oracle(n, boxes=boxes, n_levels=3, nghost=cfg.nghost, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam)
        for ib, (l, lo, hi) in enumerate(boxes):
            re, im = inputs.ring_field(rings, l, lo, hi)
            o.set_state(ib, 0, re.numpy())
            o.set_state(ib, 1, im.numpy())
        cells, _ = cells_per_step(cfg, boxes)
        desc = f"3-level ring hierarchy at base {n}^3 with 16^3 boxes ({len(boxes)} boxes), same stencil and parameters"
        levels = 3
    return o, cells, desc, levels


def oracle_step(o, cfg, eta, levels):
    o.rk_step(cfg.dt, eta)
    for l in range(levels):
        o.tag_strings(l)


def cpu_model():
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


def time_oracle(cfg, budget_s=12.0, steps=None, warmup=1):
    from oracle import oracle as orc
    o, cells, desc, levels = oracle_sample(cfg)
    eta = cfg.eta0
    for _ in range(warmup):
        oracle_step(o, cfg, eta, levels)
        eta += cfg.dt
    t0 = time.perf_counter()
    oracle_step(o, cfg, eta, levels)
    eta += cfg.dt
    one = time.perf_counter() - t0
    n = steps if steps is not None else max(1, min(50, int(budget_s / max(one, 1e-6)) - 1))
    t0 = time.perf_counter()
    for _ in range(n):
        oracle_step(o, cfg, eta, levels)
        eta += cfg.dt
    dt = (time.perf_counter() - t0) / n
    cores = orc.omp_threads()
    # the same sample on ONE host thread (single-thread and all-core numbers), two steps
    orc.set_threads(1)
    t0 = time.perf_counter()
    for _ in range(2):
        oracle_step(o, cfg, eta, levels)
        eta += cfg.dt
    dt1 = (time.perf_counter() - t0) / 2
    orc.set_threads(cores)
    return {"value": cells * 4 / dt / 1e9, "unit": UNIT, "cores": cores, "kind": "oracle",
            "note": "the unoptimised correctness oracle (g++ -O2, no -march, one loop nest per definition) on a sample: "
                    "a reported baseline of the checker, not a tuned CPU implementation",
            "sample": f"{desc}; {n} steps of rk_step + tag_strings, {dt * 1e3:.1f} ms/step",
            "single_thread_value": cells * 4 / dt1 / 1e9, "cpu_model": cpu_model()}, dt, n


# ---------------------------------------------------------------------------------------------------
# reference arm: the oracle on the host cores
# ---------------------------------------------------------------------------------------------------

def run_reference(args, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    cpu, dt, n = time_oracle(cfg, steps=args.steps, warmup=max(1, min(args.warmup, 2)))
    line = {"impl": "reference", "metric": METRIC, "value": cpu["value"], "unit": UNIT, "n_gpus": args.gpus,
            "steps": n, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"{cfg.name} (bounded sample for the CPU oracle)", "sample": cpu["sample"]},
            "cpu_baseline": cpu,
            "e2e": {"value": cpu["value"], "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------
# replicas: the path does not shard; N ranks run N independent replicas
# ---------------------------------------------------------------------------------------------------

def max_over_ranks(ms, world, device):
    """Device time of the slowest replica (the contract's max over ranks); one scalar all-reduce, outside the
    timed region.  `device`: where the backend wants the tensor (cuda for nccl, cpu for gloo)."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], device=device, dtype=torch.float64)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(world, cell_steps, ms, stages=4):
    """Gcell-updates/s per RK stage of the whole job: every replica advances `cell_steps` cell-steps (x 4 stages)
    per step, the job takes as long as its slowest replica."""
    return world * cell_steps * stages / (ms * 1e-3) / 1e9


# ---------------------------------------------------------------------------------------------------
# the CUDA arm
# ---------------------------------------------------------------------------------------------------

def measure(args, cfg, dev, world, rank, local, steps, warmup):
    """Build the workload `cfg` on `dev`, run `warmup` + `steps` steps and return (bench line, context, tags, counts,
    boxes, cell_steps).  A step = sledge_rk_step + sledge_tag_strings on every level."""
    import torch
    import torch.distributed as dist
    from paper_2404_02950_b200 import sledge as S
    rings, boxes, cover = hierarchy(cfg)
    cell_steps, per_level = cells_per_step(cfg, boxes)
    s = S.Sledge(cfg.n0, boxes=boxes, n_levels=cfg.n_levels, nghost=max(cfg.nghost, args.ko_order),
                 blocking_factor=cfg.blocking_factor,
                 dtype=cfg.dtype, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, rk_dataflow=args.flow, device=dev,
                 ko_order=args.ko_order, ko_strength=args.ko_strength if args.ko_order else 0.0,
                 integrator=args.integrator, interp=args.interp, gw=args.gw, gw_coupling=1.0 if args.gw else 0.0,
                 rkn=RKN4 if args.integrator == 20 else None)
    ssp = args.integrator in (3, 10)
    rkn_st = len(RKN4["nodes"]) if args.integrator == 20 else 0
    if ssp:
        args.flow = "ssprk3"  # three staged sweeps, 8 + 12 + 12 words per cell-step
    if rkn_st:
        args.flow = "rkn"     # stage i: Psi_i (psi_n itself for i = 0), psi_n, Pi_n, f_0..f_{i-1} in; 4 words out
    if args.gw and args.flow in ("fused", "fused3"):
        args.flow = "lean"    # the source needs psi of every stage state: staged sweeps, plus the auxiliary fields' own
    if args.ko_order and args.flow in ("fused", "fused3"):
        args.flow = "lean"  # with the dissipation term k_psi is not pointwise: every level runs the staged sweeps
    for ib, c, t in initial_fields(cfg, rings, boxes, dev, s.tdtype):
        s.set_state(ib, c, t)
        del t
    torch.cuda.empty_cache()
    tags = [torch.empty(s.level_cells(l)[0], dtype=torch.uint8, device=dev) for l in range(cfg.n_levels)]
    counts = [torch.empty(s.count_shape(l), dtype=torch.int32, device=dev) for l in range(cfg.n_levels)]

    eta = [cfg.eta0]

    def step():
        s.rk_step(cfg.dt, eta[0])
        eta[0] += cfg.dt
        for l in range(cfg.n_levels):
            s.tag_strings(l, tags[l], counts[l])

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(warmup):
        step()
    s.synchronize()
    # ---- timed region: K steps, CUDA events on the launching stream, clocks sampled meanwhile ----
    clk = ClockSampler(local)
    if rank == 0:
        clk.start()
    s.profile_enable(True)
    l0 = s.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(steps):
        step()
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1) / steps
    launches = s.launch_count() - l0
    prof = {k: s.profile_read(kind) for k, kind in
            (("stage", S.KIND_STAGE), ("ghost", S.KIND_GHOST), ("tag", S.KIND_TAG), ("avg", S.KIND_AVG))}
    s.profile_enable(False)
    clocks = clk.stop() if rank == 0 else None
    s.synchronize()
    ms = max_over_ranks(ms, world, dev)

    # ---- roofline of the dominant kernel (K1) -----------------------------------------------------
    esz = 8 if cfg.dtype == "f64" else 4
    # algorithmic words (reals read + written) per cell-step of the data-flow that runs:
    # FUSED 20 on level 0 (finer levels run LEAN), LEAN 52, CLASSIC 64
    # algorithmic words (reals read + written) per cell-step and K1 launches per level-step of the data-flow each
    # level runs, as the library reports them (sledge_level_dataflow)
    flows = [s.level_dataflow(l) for l in range(cfg.n_levels)]
    stage_words_per_step = sum(n * (1 << l) * flows[l][1] for l, n in enumerate(per_level))
    words_per_cell_step = stage_words_per_step / cell_steps
    n_stage, ms_stage = prof["stage"]
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    peak = float(peaks.get("hbm_gbs", 6650.0))
    peak_src = "measured (MEASURED_PEAKS.json hbm_gbs)" if "hbm_gbs" in peaks else "fallback 6650 GB/s (B200_PROFILING.md)"
    # profile counters cover the timed K steps: n_stage launches moved cell_steps * words * esz bytes per step
    stage_bytes_total = stage_words_per_step * esz * steps
    # K1 launches the timed steps must have produced (2 sweeps per level-step FUSED on level 0, one per stage
    # otherwise); the library keeps at most 4096 event pairs per kind, so scale the bytes to the launches it timed
    sweeps = [flows[l][0] * (1 << l) for l in range(cfg.n_levels)]
    expected_stage = steps * sum(sweeps)
    timed_all = n_stage == expected_stage
    if not timed_all and expected_stage > 0:
        stage_bytes_total *= n_stage / expected_stage
    achieved = stage_bytes_total / (ms_stage * 1e-3) / 1e9 if ms_stage > 0 else 0.0
    tr = ncu_traffic(cfg.name, args.flow)
    roofline = {"bound": "hbm", "kernel": "K1 (k_rk_tma FUSED sweeps -- fp64: the W form FUSED_A2 / FUSED_B2, DESIGN.md section 5 -- on every level that can run them; k_rk_pipe staged sweeps otherwise; mean over the "
                                          "stage launches of a step: 2 sweeps per level-step FUSED, 4 otherwise)", "achieved": achieved,
                "peak": peak, "unit": "GB/s", "frac": achieved / peak, "frac_of_nominal_8TBs": achieved / 8000.0,
                "peak_source": peak_src, "traffic": (tr or {}).get("dram_bytes_per_launch"), "traffic_detail": tr,
                "bytes_per_cell_step": words_per_cell_step * esz,
                "avg_launch_ms": ms_stage / max(n_stage, 1), "launches": n_stage, "launches_expected": expected_stage,
                "k1_launches_and_words_per_level": flows,
                "all_launches_timed": timed_all}
    shares = {k: (v[1] / steps) for k, v in prof.items()}

    nstage = 3 if ssp else (rkn_st if rkn_st else 4)
    value = whole_job_value(world, cell_steps, ms, stages=nstage)
    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps,
            "warmup": warmup, "ms_per_step": ms, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": cfg.dtype, "data": "synthetic",
            "config": {"workload": f"{cfg.name}: {cfg.n0}^3 base, {cfg.n_levels} level(s), {cfg.dtype}, "
                                   f"{'13' if cfg.lap_order == 2 else '7'}-point Laplacian, {'SSPRK3' if ssp else ('RKN4 (integrator 20)' if rkn_st else 'RK4')} ({args.flow} data-flow), "
                                   f"dt={cfg.dt}, h0={cfg.h0}, tags + 32^3 counts every step"
                                   + (f", Kreiss-Oliger order {args.ko_order} eps {args.ko_strength}" if args.ko_order else "")
                                   + (", with the 12 gravitational-wave auxiliary components (Eq.16)" if args.gw else "")
                                   + (", quartic conservative coarse->fine interpolation" if args.interp == 4 and cfg.n_levels > 1 else ""),
                       "cells_per_level": per_level, "coverage": cover, "cell_steps_per_step": cell_steps,
                       "boxes_per_level": [len(s.level_boxes(l)) for l in range(cfg.n_levels)],
                       "storage_boxes_per_level": [s.level_storage(l)[0] for l in range(cfg.n_levels)],
                       "l2": "state buffers >> 126 MB L2 (no flush needed)" if cell_steps * esz * 4 > 4e8 else
                             "state fits in L2 (small case; not a roofline workload)",
                       "multi_gpu": "replicas only"},
            "gcell_steps_per_s": value / nstage,
            "kernel_ms_per_step": shares, "roofline": roofline, "gpu_launches": launches, "clocks": clocks}

    return line, s, tags, counts, boxes, cell_steps


def run_sledge(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2404_02950_b200 import build as sbuild
    from paper_2404_02950_b200 import sledge as S

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the sledge path has no CPU fallback)")
    torch.cuda.set_device(local)
    dev = f"cuda:{local}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))
    if not os.path.exists(S.LIB_PATH):
        sbuild.build()

    line, s, tags, counts, boxes, cell_steps = measure(args, cfg, dev, world, rank, local, args.steps, args.warmup)

    # ---- e2e: same step through the C ABI with HOST buffers -----------------------------------------
    if not args.no_e2e:
        line["e2e"] = e2e_leg(args, cfg, s, boxes, cell_steps, world, step_tags=(tags, counts))
    del s
    torch.cuda.empty_cache()
    default_run = args.integrator == 4 and not args.ko_order and args.flow == "fused" and args.interp == 0 and not args.gw
    if rank == 0 and not args.no_graph and args.integrator == 4 and not args.ko_order:
        from paper_2404_02950_b200 import inputs as _inputs
        line["c1_graph_replay"] = graph_leg(_inputs.CONFIGS["C1"], dev, "fused")
        if default_run and not args.no_others:
            line["c5_graph_replay"] = graph_step_leg(_inputs.CONFIGS["C5"], dev, "fused")
    if rank == 0 and default_run and not args.no_others:
        line["other_workloads"] = other_workloads(args, cfg, dev)
    if rank == 0 and not args.no_cpu:
        line["cpu_baseline"], _, _ = time_oracle(cfg)
    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


# ---------------------------------------------------------------------------------------------------
# C1 under CUDA Graph replay (the 32^3 case is launch-bound)
# ---------------------------------------------------------------------------------------------------

def capture_run(s, ic, tags, counts, steps, dt, eta0):
    """Capture `restore the initial state + steps x (sledge_rk_step + sledge_tag_strings)` of a single-level context
    into ONE CUDA graph on the context's stream.  Every library call is an asynchronous launch on that stream (no
    allocation, no host synchronisation), eta enters as kernel arguments, so the whole run replays with one launch.
    The context must have run the same sequence once eagerly (first launches set kernel attributes)."""
    import torch
    g = torch.cuda.CUDAGraph()
    with torch.cuda.graph(g, stream=s.stream):
        for c, t in enumerate(ic):
            s.set_state(0, c, t)
        eta = eta0
        for _ in range(steps):
            s.rk_step(dt, eta)
            eta += dt
            s.tag_strings(0, tags, counts)
    return g


def graph_leg(cfg, dev, flow, replays=20, dt=None):
    """The C1 run (10 steps of 32^3) eagerly and as one CUDA graph replay: ms per step of both."""
    import torch
    from paper_2404_02950_b200 import inputs
    from paper_2404_02950_b200 import sledge as S
    dt = cfg.dt if dt is None else dt
    side = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(side):  # the context adopts torch's current stream: capture needs a non-default one
        s = S.Sledge(cfg.n0, nghost=cfg.nghost, dtype=cfg.dtype, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam,
                     rk_dataflow=flow, device=dev)
        ic = [inputs.grf(cfg.n0, cfg.grf_f, seed, device=dev, dtype=s.tdtype).contiguous() for seed in cfg.seeds]
        ic += [torch.zeros_like(ic[0]), torch.zeros_like(ic[0])]
        tags = torch.empty(s.level_cells(0)[0], dtype=torch.uint8, device=dev)
        counts = torch.empty(s.count_shape(0), dtype=torch.int32, device=dev)

        def eager():
            for c, t in enumerate(ic):
                s.set_state(0, c, t)
            eta = cfg.eta0
            for _ in range(cfg.steps):
                s.rk_step(dt, eta)
                eta += dt
                s.tag_strings(0, tags, counts)

        eager()
        side.synchronize()
        l0 = s.launch_count()
        eager()
        per_run = s.launch_count() - l0
        ref = [s.get_state(0, c).clone() for c in range(4)]
        ref_tags = tags.clone()
        g = capture_run(s, ic, tags, counts, cfg.steps, dt, cfg.eta0)

        def timed(fn):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            for _ in range(3):
                fn()
            side.synchronize()
            e0.record(side)
            for _ in range(replays):
                fn()
            e1.record(side)
            side.synchronize()
            return e0.elapsed_time(e1) / (replays * cfg.steps)

        ms_eager = timed(eager)
        ms_graph = timed(g.replay)
        got = [s.get_state(0, c) for c in range(4)]
        side.synchronize()
        same = all(torch.equal(a.view(torch.int64), b.view(torch.int64)) for a, b in zip(ref, got)) and \
            torch.equal(ref_tags, tags)
        s.close()
    cells = cfg.n0 ** 3
    return {"workload": f"{cfg.name}: {cfg.n0}^3 {cfg.dtype}, {cfg.steps} steps + tags, {flow} data-flow; the graph also "
                        "restores the initial state (4 copy kernels)",
            "launches_per_run": per_run, "ms_per_step_eager": ms_eager, "ms_per_step_graph": ms_graph,
            "value_eager": cells * 4 / (ms_eager * 1e-3) / 1e9, "value_graph": cells * 4 / (ms_graph * 1e-3) / 1e9,
            "unit": UNIT, "replay_equals_eager_bitwise": bool(same)}


def other_workloads(args, main_cfg, dev):
    """Short runs (resident state, same timed-region rules, `--other-steps` steps after 3 warm-up steps) of the other
    BASELINE.json workloads that fit one GPU, so that the bench record carries them: value, ms per step, per-kernel
    time, K1 roofline fraction, clocks.  The headline line and its config stay those of the main workload."""
    import copy
    import torch
    from paper_2404_02950_b200 import inputs
    out = {}
    for name in ("C2", "C4", "C5"):
        if name == main_cfg.name:
            continue
        a = copy.copy(args)
        a.flow = "fused"
        try:
            line, s, tags, counts, _, _ = measure(a, inputs.CONFIGS[name], dev, 1, 0, 0, args.other_steps, 3)
        except Exception as e:  # e.g. out of memory on a smaller part: reported, not fatal for the headline
            out[name] = {"error": str(e)[:200]}
            continue
        out[name] = {"workload": line["config"]["workload"], "value": line["value"], "unit": UNIT, "dtype": line["dtype"],
                     "ms_per_step": line["ms_per_step"], "steps": line["steps"],
                     "kernel_ms_per_step": line["kernel_ms_per_step"], "k1_frac": line["roofline"]["frac"],
                     "k1_achieved_gbs": line["roofline"]["achieved"], "gpu_launches": line["gpu_launches"],
                     "clocks": line["clocks"]}
        s.close()
        del s, tags, counts
        torch.cuda.empty_cache()
    return out


def graph_step_leg(cfg, dev, flow, steps=5):
    """ONE coarse step of `cfg` (sledge_rk_step: subcycled stages, ghost fills, average-downs; then sledge_tag_strings
    on every level) eagerly and as one CUDA graph replay: ms per coarse step of both, and
    whether the replayed step equals the eager one bit for bit.  The graph is captured from a freshly set state, so a
    replay recomputes that same step (the step never writes the buffer it starts from)."""
    import torch
    from paper_2404_02950_b200 import sledge as S
    rings, boxes, _ = hierarchy(cfg)
    side = torch.cuda.Stream(device=dev)
    with torch.cuda.stream(side):
        s = S.Sledge(cfg.n0, boxes=boxes, n_levels=cfg.n_levels, nghost=cfg.nghost, blocking_factor=cfg.blocking_factor,
                     dtype=cfg.dtype, lap_order=cfg.lap_order, h0=cfg.h0, lam=cfg.lam, rk_dataflow=flow, device=dev)
        ic = {(ib, c): t for ib, c, t in initial_fields(cfg, rings, boxes, dev, s.tdtype)}
        zero = {}
        tags = [torch.empty(s.level_cells(l)[0], dtype=torch.uint8, device=dev) for l in range(cfg.n_levels)]
        counts = [torch.empty(s.count_shape(l), dtype=torch.int32, device=dev) for l in range(cfg.n_levels)]

        def restore():
            for ib in range(len(boxes)):
                for c in range(4):
                    t = ic.get((ib, c))
                    if t is None:
                        t = zero.setdefault(tuple(s.box_shape(ib)), torch.zeros(s.box_shape(ib), dtype=s.tdtype, device=dev))
                    s.set_state(ib, c, t)

        def step(eta):
            s.rk_step(cfg.dt, eta)
            for l in range(cfg.n_levels):
                s.tag_strings(l, tags[l], counts[l])

        def timed(fn):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            fn()
            side.synchronize()
            e0.record(side)
            for _ in range(steps):
                fn()
            e1.record(side)
            side.synchronize()
            return e0.elapsed_time(e1) / steps

        restore()
        l0 = s.launch_count()
        step(cfg.eta0)
        per_step = s.launch_count() - l0
        ms_eager = timed(lambda: step(cfg.eta0))
        restore()
        step(cfg.eta0)
        ref = [s.get_state(ib, c).clone() for ib in range(len(boxes)) for c in range(4)]
        ref_tags = [t.clone() for t in tags]
        restore()
        side.synchronize()
        g = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g, stream=side):
            step(cfg.eta0)
        g.replay()
        got = [s.get_state(ib, c) for ib in range(len(boxes)) for c in range(4)]
        side.synchronize()
        same = all(torch.equal(a.view(torch.int64), b.view(torch.int64)) for a, b in zip(ref, got)) and \
            all(torch.equal(a, b) for a, b in zip(ref_tags, tags))
        ms_graph = timed(g.replay)
        s.close()
    cell_steps, _ = cells_per_step(cfg, boxes)
    return {"workload": f"{cfg.name}: one coarse step of the {len(boxes)}-box hierarchy + tags on {cfg.n_levels} levels, {flow} data-flow",
            "launches_per_step": per_step, "ms_per_step_eager": ms_eager, "ms_per_step_graph": ms_graph,
            "value_eager": cell_steps * 4 / (ms_eager * 1e-3) / 1e9, "value_graph": cell_steps * 4 / (ms_graph * 1e-3) / 1e9,
            "unit": UNIT, "replay_equals_eager_bitwise": bool(same)}


def e2e_leg(args, cfg, s, boxes, cell_steps, world, step_tags):
    """Per step: host->device copy of the whole state (4 components of every box, pinned host memory) through
    sledge_set_state_host, rk_step + tag_strings, device->host copy of the new state and the block counts."""
    import torch
    tags, counts = step_tags
    host_in = [[torch.empty(s.box_shape(ib), dtype=s.tdtype).pin_memory() for _ in range(4)] for ib in range(len(boxes))]
    host_out = [[torch.empty(s.box_shape(ib), dtype=s.tdtype).pin_memory() for _ in range(4)] for ib in range(len(boxes))]
    host_counts = [torch.empty(c.shape, dtype=torch.int32).pin_memory() for c in counts]
    for ib in range(len(boxes)):
        for c in range(4):
            s.get_state_host(ib, c, host_in[ib][c])
    s.synchronize()
    bi = sum(t.numel() * t.element_size() for b in host_in for t in b)
    bo = bi + sum(t.numel() * t.element_size() for t in host_counts)
    eta = cfg.eta0

    def one():
        for ib in range(len(boxes)):
            for c in range(4):
                s.set_state_host(ib, c, host_in[ib][c])
        s.rk_step(cfg.dt, eta)
        for l in range(cfg.n_levels):
            s.tag_strings(l, tags[l], counts[l])
            host_counts[l].copy_(counts[l], non_blocking=True)
        for ib in range(len(boxes)):
            for c in range(4):
                s.get_state_host(ib, c, host_out[ib][c])

    one()
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.e2e_steps):
        one()
    s.host_copies_join()  # the context stream waits for the last downloads: e1 includes them
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / args.e2e_steps
    return {"value": whole_job_value(world, cell_steps, ms, stages={3: 3, 10: 3, 20: len(RKN4["nodes"])}.get(args.integrator, 4)),
            "unit": UNIT, "ms_per_step": ms,
            "h2d_bytes_per_step": bi, "d2h_bytes_per_step": bo, "steps": args.e2e_steps,
            "what": "sledge_set_state_host x4/box + sledge_rk_step + sledge_tag_strings + sledge_get_state_host x4/box + counts",
            "note": "every step uploads and downloads the whole state; the library's two copy streams let the downloads of "
                    "step k overlap the uploads of step k+1 (PCIe is full duplex), so the first upload and the last download "
                    "are the only unoverlapped ones and ms_per_step falls towards the one-direction copy time as steps grows"}


def main():
    args = parse()
    if args.e2e_steps <= 0:
        args.e2e_steps = min(max(args.steps, 4), 20)
    from paper_2404_02950_b200 import inputs
    cfg = inputs.CONFIGS[args.workload]
    if args.impl == "reference":
        run_reference(args, cfg)
    else:
        run_sledge(args, cfg)


if __name__ == "__main__":
    main()
