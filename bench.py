#!/usr/bin/env python
"""bench.py -- clipped Voronoi cells/s on B200 (BASELINE.json metric), one JSON line.

A "step" is one pass of the whole hot path (S1 index, S3 seeds, S4+S5 clip + propagate, S6 assemble =
one vd_compute) over one seeded synthetic workload.  `value` is device-timed with the inputs already
resident in HBM (the context holds copies of sites and domain); `e2e` is the same metric through the C
ABI with HOST buffers: vd_create + vd_set_domain + vd_compute + vd_cells_to_host + vd_destroy.

The default run times ALL FIVE BASELINE.json configs in one process and prints ONE line: the top-level keys
(value, ms_per_step, config, roofline, e2e, cpu_baseline) are those of the LARGEST config, C3 (most simplices,
most pairs, longest step); `per_config` holds the same keys for C1, C2, C4, C5, and `c5_under_1s` states
BASELINE.json's target for the 2M-site config.  --config K times only config K.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0|1..5] [--impl reference]

N > 1 (torchrun): the path shards by simplex: rank r clips its contiguous block of M against the
replicated sites, one NCCL all-reduce of per-cell (measure, moment) per step; value = n / max-over-ranks time.
--impl reference: the CPU oracle, as it stands, timed on the host cores on a bounded sample.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "clipped Voronoi cells/sec at 1 B200 (device-timed); achieved % of roofline"
UNIT = "cells/s"
# plain FP64 ALU peak derived from unit counts and clocks: 148 SMs x 64 FP64 FMA
# lanes x 2 flop at the maximum SM clock; no FP64 figure exists in MEASURED_PEAKS.json.
FP64_LANES_PER_SM, SMS = 64, 148
# roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, read by kernel
# name and config from the committed summary of the ncu --set full captures (never from a literal here); null when
# that kernel / config has no capture
TRAFFIC_CSV = os.path.join(ROOT, "profiles", "r02_dram_traffic.csv")
TOP_CONFIG = 3
WORKLOADS = {1: "C1: 2D unit square, 2 triangles, 2,000 uniform sites, seed 0",
             2: "C2: unit cube 20^3 x 6 tets (48,000), 100,000 uniform sites, seed 1",
             3: "C3: unit cube 48^3 x 6 tets (663,552), 1,000,000 clustered sites, seed 2",
             4: "C4: torus 512x256 (262,144 triangles), 200,000 shell sites, seed 3",
             5: "C5: unit cube 32^3 x 6 tets (196,608), 2,000,000 far-slab sites, seed 4"}


class ClockSampler:
    """SM clock and clock-event (throttle) reasons sampled DURING the timed region, through NVML -- the library
    nvidia-smi itself reads --, by the timed loop itself right after every step, outside the event brackets.  (A
    `nvidia-smi -lms 20` child process was measured to slow the phased schedule, which synchronises with the host
    once per round, from 35 to 47 ms per C2 step: every one of its polls holds the driver for milliseconds.)  Falls back to `nvidia-smi -lms 200` when NVML
    cannot be opened.  (About one step in thirty still takes 10-40 ms longer on these shared hosts, with or without
    any sampling: the schedule waits on the host some 25 times per step; `ms_steps` lists every step.)"""

    def __init__(self, index, uuid=None):
        self.index, self.uuid = index, uuid
        self.sm, self.mx, self.reasons = [], [], set()
        self.stop_flag = threading.Event()
        self.thread = None
        self.proc = None
        self.source = None
        self.nv = None
        self.handle = None

    def sample(self):
        """One NVML sample (SM clock, clock-event reasons).  Also called by the timed loop itself between two steps,
        outside the event-bracketed part: an NVML read can hold the driver while the phased schedule waits on it."""
        if self.nv is None:
            return
        nv, h = self.nv, self.handle
        names = {nv.nvmlClocksEventReasonHwSlowdown: "hw_slowdown", nv.nvmlClocksEventReasonHwThermalSlowdown: "hw_thermal_slowdown",
                 nv.nvmlClocksEventReasonSwThermalSlowdown: "sw_thermal_slowdown", nv.nvmlClocksEventReasonSwPowerCap: "sw_power_cap"}
        try:
            self.sm.append(float(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
            r = nv.nvmlDeviceGetCurrentClocksEventReasons(h)
            self.reasons.update(n for bit, n in names.items() if r & bit)
        except Exception:
            pass

    def start(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = None
            if self.uuid:
                for u in (self.uuid, "GPU-" + self.uuid):
                    try:
                        h = nv.nvmlDeviceGetHandleByUUID(u)
                        break
                    except Exception:
                        h = None
            if h is None:
                h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.mx.append(float(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM)))
            self.nv, self.handle = nv, h
            self.source = "nvml, read by the timed loop after every step (outside the event brackets)"
            self.sample()
            return
        except Exception:
            self.thread = None
        q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
             "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
            self.source = "nvidia-smi -lms 200"
        except OSError:
            self.proc = None

    def _read(self):
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in self.proc.stdout:
            r = [x.strip() for x in line.split(",")]
            if len(r) >= 6 and r[0].replace(".", "").isdigit():
                self.sm.append(float(r[0]))
                self.mx.append(float(r[1]))
                self.reasons.update(names[k] for k in range(4) if r[2 + k].startswith("Active"))

    def stop(self):
        self.stop_flag.set()
        if self.thread:
            self.thread.join(timeout=1.0)
        if self.proc:
            self.proc.terminate()
        return {"sm_mhz": float(np.median(self.sm)) if self.sm else None, "sm_max_mhz": max(self.mx) if self.mx else None,
                "reasons": sorted(self.reasons), "samples": len(self.sm), "source": self.source}


def algorithmic_flops(c, kind):
    """algorithmic flop = 8 D + 15 I + sum over clips (2d x corners tested + 60 x new corners) + 30 x fan
    simplices, every term COUNTED by the kernels (D = site distance evaluations, 5 flop each in 2D; I = search
    iterations; a new 2D corner is one 2 x 2 solve = 15 flop).  c = one counter block (a kernel's, or the totals)."""
    flat = kind in (0, 3)
    d = 2 if flat else 3
    return ((5 if flat else 8) * c["dist_evals"] + 15 * c["search_iters"] + 2 * d * c["clip_corners"]
            + (15 if kind in (0, 1, 3) else 60) * c["new_corners"] + 30 * c["fan_simplices"])


def traffic_from_profiles(kernel, cfg):
    """(dram bytes per launch, source) of `kernel` on config `cfg` from profiles/r02_dram_traffic.csv, else (None, None)."""
    try:
        with open(TRAFFIC_CSV) as f:
            rows = [ln.strip().split(",") for ln in f if ln.strip() and not ln.startswith("#")]
    except OSError:
        return None, None
    hdr, rows = rows[0], rows[1:]
    col = {name: k for k, name in enumerate(hdr)}
    for r in rows:
        if r[col["config"]] == f"C{cfg}" and r[col["kernel"]] == kernel.split("<")[0].split(" ")[0]:
            n = max(1, int(r[col["launches"]]))
            return (float(r[col["dram_read_bytes"]]) + float(r[col["dram_write_bytes"]])) / n, r[col["source"]]
    return None, None


def oracle_tier(w):
    return "A" if w.kind == 1 else "B"


def cpu_oracle_sample(w, seconds_target=15.0, seed=12345):
    """The oracle as it stands (tier B for volumes / 2D, tier A for the surface), timed on the host
    cores on a bounded random sample of sites of the same workload."""
    from oracle import oracle
    rng = np.random.default_rng(seed)
    tier = oracle_tier(w)
    k = min(w.n, 32)
    t0 = time.perf_counter()
    r = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=np.sort(rng.choice(w.n, k, replace=False)), tier=tier)
    dt = time.perf_counter() - t0
    per_site = dt / k
    k2 = int(min(w.n, max(k, seconds_target / max(per_site, 1e-9))))
    if k2 > 2 * k:
        k = k2
        t0 = time.perf_counter()
        r = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=np.sort(rng.choice(w.n, k, replace=False)), tier=tier)
        dt = time.perf_counter() - t0
    return {"value": k / dt, "unit": UNIT, "cores": int(r.threads_used), "kind": "oracle",
            "sample": f"{k} seeded-random sites of the workload, tier {tier}, {dt:.1f} s wall"}


def config_dict(w, workload, world, sharded):
    """The `config` object: the same for our arm and for the reference arm."""
    return {"workload": workload, "n_sites": w.n, "n_simplices": w.m, "l2": "flushed between timed steps (256 MiB fill)",
            "parallelism": ("1 GPU" if world == 1 else (f"simplices in {world} contiguous blocks, sites replicated, one all-reduce of cell moments"
                                                       if sharded else "replicas only"))}


def run_reference(args, w, workload):
    """--impl reference: each step = the oracle on a bounded sample of sites of the same workload."""
    from oracle import oracle
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    tier = oracle_tier(w)
    rng = np.random.default_rng(777)
    probe = oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=np.sort(rng.choice(w.n, min(w.n, 16), replace=False)), tier=tier)
    t0 = time.perf_counter()
    oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=np.sort(rng.choice(w.n, min(w.n, 16), replace=False)), tier=tier)
    per_site = (time.perf_counter() - t0) / min(w.n, 16)
    budget = 120.0 / max(1, args.steps + args.warmup)
    k = int(min(w.n, max(8, budget / max(per_site, 1e-9))))
    times = []
    for s in range(args.warmup + args.steps):
        sub = np.sort(rng.choice(w.n, k, replace=False))
        t0 = time.perf_counter()
        oracle.compute(w.sites, w.verts, w.simplices, w.kind, subset=sub, tier=tier)
        if s >= args.warmup:
            times.append(time.perf_counter() - t0)
    total = sum(times)
    val = k * len(times) / total
    sample = f"{k} seeded-random sites per step, tier {tier}"
    sharded = world > 1 and w.simplices is not None
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * total / len(times), "higher_is_better": True,
        "scaling": "strong" if sharded else "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w, workload, world, sharded),
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": int(probe.threads_used), "kind": "oracle", "sample": sample},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def measure(w, workload, cfg, args, env, cpu_seconds):
    """Time args.steps steps of the hot path on workload w (after args.warmup untimed ones); returns the keys of one
    bench line.  env = (torch, dist, binding, ranks, rank, world, dev, stream, flush, sampler, fp64_meas)."""
    torch, dist, binding, ranks, rank, world, dev, stream, flush, sampler, fp64_meas = env

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # inputs resident in HBM before the timed region
    d_sites = torch.from_numpy(w.sites).to(dev)
    d_verts = torch.from_numpy(w.verts).to(dev)
    d_simp = torch.from_numpy(w.simplices).to(dev) if w.simplices is not None else None
    ctx = binding.Context(d_sites)
    ctx.set_stream(stream.cuda_stream)
    # N > 1: the path shards by simplex: rank r clips its block of M against the replicated sites, one
    # all-reduce of per-cell (measure, first moment) combines the partial cells -- inside the timed region.  Simple
    # domains (one piece per cell) have nothing to partition: every rank runs its own replica.
    sharded = world > 1 and w.simplices is not None
    opts = {}
    if sharded:
        blk = ranks.simplex_blocks_balanced(w.sites, w.verts, w.simplices, world)[rank]   # about equal pairs per rank
        opts = dict(simplex_begin=blk[0], simplex_end=blk[1])
        ctx.set_options(**opts)
    ctx.set_domain(d_verts, d_simp, w.kind)
    buf = None
    for _ in range(args.warmup):
        ctx.compute()
        if sharded:
            buf = ranks.combine_partial_cells(ctx, buf)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    clip_ms, launches = 0.0, 0
    phase_ms = {"init": 0.0, "verify": 0.0, "fix": 0.0, "finish": 0.0, "tail": 0.0}
    for k in range(args.steps):
        flush.fill_(k & 0xff)            # L2 flush between timed iterations (not timed)
        ev[k][0].record(stream)
        ctx.compute()
        if sharded:
            ranks.combine_partial_cells(ctx, buf)
        ev[k][1].record(stream)
        sampler.sample()
        clip_ms += ctx.stage_ms()["clip"]
        for name, v in ctx.phase_ms().items():
            phase_ms[name] += v
        launches += ctx.counters()["launches"]
    barrier()
    step_ms = [a.elapsed_time(b) for a, b in ev]
    ms = sum(step_ms)
    cnt = ctx.counters()
    pcnt = ctx.phase_counters()
    stage = ctx.stage_ms()
    sizes = {"nonempty_cells": int(ctx.cells.n_nonempty), "pieces": int(ctx.cells.n_pieces), "corners": int(ctx.cells.n_verts),
             "neighbour_entries": int(ctx.cells.n_nbrs)}
    # sharded: the ranks together made ONE diagram of n cells per step; replicas: one each
    value, ms = ranks.whole_job_rate(float(w.n * args.steps) / (world if sharded else 1), ms, dev)
    # The work counts come from one more, UNTIMED, step on the same inputs with vd_options.count_alg = 2: the
    # timed kernels keep no per-query statistics (their bookkeeping alone is 3-4 % of a step), the counting ones do, and D_alg
    # (next to D_act) is counted there too.  The work is a property of the inputs: the timed step did the same.
    ctx.set_options(count_alg=2, **opts)
    ctx.compute()
    full = ctx.counters()
    d_alg = full["alg_evals"]
    for k in ("queries", "dist_evals", "row_evals", "search_evals", "search_iters", "clips", "clip_corners", "new_corners", "fan_simplices", "pairs", "pieces", "pre_clips"):
        cnt[k] = full[k]
    pcnt = ctx.phase_counters()
    # Alg. 5's site division (vd_options.dissolve; convex tet meshes, one GPU): interior cells as whole cells.  Reported
    # beside the per-piece number, never instead of it (the per-piece output is what parity with SURVEY 8c.1 is defined on)
    dissolve = None
    if w.kind == 2 and not sharded and cfg == 2:
        ctx.set_options(dissolve=1)
        for _ in range(2):
            ctx.compute()
        ts = []
        for k in range(min(args.steps, 5)):
            flush.fill_(k & 0xff)
            ctx.compute()
            ts.append(ctx.stage_ms()["total"])
        ctx.set_options(dissolve=1, count_alg=1)     # the work counts: one more untimed step with the statistics on
        ctx.compute()
        dc = ctx.counters()
        dissolve = {"ms_per_step": float(np.mean(ts)), "value": w.n / (float(np.mean(ts)) * 1e-3), "unit": UNIT, "pairs": dc["pairs"],
                    "queries_per_cell": dc["queries"] / w.n, "paper_queries_per_cell_serial_alg2_cube": 20.54,
                    "timing": "library events around vd_compute (stage total), L2 flushed between steps"}
    # Lloyd iterations on the device (section VII-D, density 1; --lloyd IT): wall time of vd_lloyd, with and without the
    # reuse of the previous iteration's neighbours as first clips (vd_options.reuse_nbrs)
    lloyd = None
    if args.lloyd > 0:
        lloyd = {"iterations": args.lloyd, "paper": "5 M sites x 100 iterations in 31.07 s on an RTX 3080, fp32 (P:L492): another machine, context only"}
        for name, o in (("reuse_nbrs", {}), ("no_reuse", dict(reuse_nbrs=-1))):
            ctx.update_sites(d_sites)
            ctx.set_options(**o)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ctx.lloyd(args.lloyd)
            torch.cuda.synchronize()
            dt = time.perf_counter() - t0
            lloyd[name] = {"seconds": dt, "ms_per_iteration": 1e3 * dt / (args.lloyd + 1), "computes": args.lloyd + 1}
    ctx.destroy()

    # end to end through the C ABI with host buffers: create, set_domain, compute, copy back, destroy
    barrier()
    e2e_steps = max(2, min(args.steps, 5))
    for k in range(e2e_steps + 1):
        if k == 1:      # the first pass is warm-up: it page-locks the staging buffers and fills the memory pool
            torch.cuda.synchronize()
            t0 = time.perf_counter()
        c2 = binding.Context(w.sites)
        c2.set_stream(stream.cuda_stream)
        if sharded:
            c2.set_options(**opts)
        c2.set_domain(w.verts, w.simplices, w.kind)
        c2.compute()
        h = c2.to_host(pinned=True)
        c2.destroy()
    torch.cuda.synchronize()
    e2e_s = (time.perf_counter() - t0) / e2e_steps
    d2h = sum(getattr(h, f).nbytes for f in ("measure", "centroid", "nbr_off", "nbr", "piece_off", "piece_simplex",
                                            "piece_measure", "vert_off", "vert_xyz", "vert_flags"))
    h2d = w.sites.nbytes + w.verts.nbytes + (w.simplices.nbytes if w.simplices is not None else 0)
    e2e_val, _ = ranks.whole_job_rate(float(w.n) / (world if sharded else 1), e2e_s * 1e3, dev)

    flops = algorithmic_flops(cnt, w.kind)
    sm_max = (sampler.mx and max(sampler.mx)) or 1965.0
    peak = SMS * FP64_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
    if sum(phase_ms.values()) > 0:
        # phased schedule: the dominant kernel is the step kernel with the largest device time (CUDA events
        # around every launch, inside the library, on the stream the kernels run on); its flop from ITS counters
        top = max(phase_ms, key=phase_ms.get)
        kernel, kernel_ms, kcnt = "k_ph_" + top, phase_ms[top] / args.steps, pcnt[top]
    else:
        kernel, kernel_ms, kcnt = "k_clip (S4+S5, one-kernel schedule)", clip_ms / args.steps, cnt
    kernel_flops = algorithmic_flops(kcnt, w.kind)
    achieved = kernel_flops / (kernel_ms * 1e-3) / 1e12
    traffic, traffic_src = traffic_from_profiles(kernel, cfg)
    out = {
        "value": value, "unit": UNIT, "ms_per_step": ms / args.steps, "ms_steps": [round(x, 3) for x in step_ms],
        "config": config_dict(w, workload, world, sharded), "result_sizes": sizes,
        "nonempty_cells_per_s": value * sizes["nonempty_cells"] / w.n, "pairs_per_s": value * cnt["pairs"] / w.n,
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h)},
        "gpu_launches": int(launches), "stage_ms": stage, "counters": cnt,
        "counters_source": "launches / syncs / waves: the last timed step; work counts: one extra untimed step with vd_options.count_alg = 2",
        "per_cell": {"queries": cnt["queries"] / w.n, "d_act": cnt["dist_evals"] / w.n, "d_alg": d_alg / w.n,
                     "d_act_over_d_alg": cnt["dist_evals"] / max(1, d_alg), "queries_per_pair": cnt["queries"] / max(1, cnt["pairs"]),
                     "clips": cnt["clips"] / w.n, "pieces": cnt["pieces"] / w.n},
        "phase_ms": {k: v / args.steps for k, v in phase_ms.items()},
        "dissolve_mode": dissolve,
        "lloyd": lloyd,
        "roofline": {"bound": "alu", "kernel": kernel, "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                     "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                     "peak_source": "derived: 148 SMs x 64 FP64 FMA lanes x 2 x max SM clock (DESIGN.md); no FP64 peak in MEASURED_PEAKS.json",
                     "peak_measured": fp64_meas, "frac_of_measured": achieved / fp64_meas,
                     "peak_measured_source": "vd_dfma_peak: 8 dependent DFMA chains per thread, SMs x 8 blocks x 256 threads, best of 3, this run",
                     "algorithmic_flop_per_step": kernel_flops, "kernel_ms_per_step": kernel_ms,
                     "kernel_counters": {k: kcnt[k] for k in ("dist_evals", "search_iters", "clip_corners", "new_corners", "fan_simplices", "clips", "queries")},
                     "flop_formula": "8 D (5 in 2D) + 15 I + 2d clip_corners + 60 new_corners (15 on triangles) + 30 fan_simplices, all counted in the kernels",
                     "share_of_step": kernel_ms * args.steps / ms,
                     "s4_ms_per_step": clip_ms / args.steps, "s4_algorithmic_flop_per_step": flops},
    }
    if rank == 0 and not args.no_cpu_baseline and world == 1 and cpu_seconds > 0:
        out["cpu_baseline"] = cpu_oracle_sample(w, cpu_seconds)
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=0, help="0 (default): all five BASELINE.json configs, top-level = C3 (the largest); "
                    "1..5: only that config")
    ap.add_argument("--box", type=int, default=0, help="instead of a BASELINE config: N white-noise sites in the unit cube, the cube itself "
                    "as a simple domain (VD_BOX_3D; the setting of the paper's Fig. 1 / Table VI)")
    ap.add_argument("--lloyd", type=int, default=0, help="also time vd_lloyd with this many iterations (with --box: the paper's CVT setting)")
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl != "reference" else args.warmup
    from paper_2509_07175_b200 import inputs
    top = args.config if args.config else TOP_CONFIG
    others = [] if (args.config or args.box) else [k for k in (1, 2, 4, 5)]
    w = inputs.box(3, args.box, seed=9) if args.box else inputs.config(top)
    workload = f"whole cells of {args.box} uniform sites in the unit cube (VD_BOX_3D, paper Fig. 1 setting)" if args.box else WORKLOADS[top]
    if args.impl == "reference":
        run_reference(args, w, workload)
        return

    import torch
    import torch.distributed as dist
    from paper_2509_07175_b200 import binding, ranks
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the library has no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl")
    dev = torch.device("cuda", local)
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)   # > 126 MB L2
    fp64_meas, _ = binding.fp64_peak(stream.cuda_stream)   # dependent-FMA-chain kernel (vd_dfma_peak), outside the timed region
    try:
        uuid = str(torch.cuda.get_device_properties(local).uuid)
    except Exception:
        uuid = None
    sampler = ClockSampler(local, uuid)
    sampler.start()
    env = (torch, dist, binding, ranks, rank, world, dev, stream, flush, sampler, fp64_meas)
    res = measure(w, workload, 0 if args.box else top, args, env, 15.0)
    per_config = {}
    for k in others:
        wk = inputs.config(k)
        per_config[f"C{k}"] = measure(wk, WORKLOADS[k], k, args, env, 4.0)
        del wk
    clocks = sampler.stop()
    out = {"metric": METRIC, "value": res.pop("value"), "unit": res.pop("unit"), "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
           "ms_per_step": res.pop("ms_per_step"), "higher_is_better": True,
           "scaling": "strong" if (world > 1 and w.simplices is not None) else "weak", "vs_baseline": None,
           "dtype": "f64", "data": "synthetic", "clocks": clocks}
    out.update(res)
    if per_config:
        out["per_config"] = per_config
        out["c5_under_1s"] = bool(per_config["C5"]["ms_per_step"] < 1000.0)
        out["gpu_launches"] = int(out["gpu_launches"] + sum(v["gpu_launches"] for v in per_config.values()))
    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
