#!/usr/bin/env python
"""bench.py -- throughput of the photon-package hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5|3|4p|4|2|1] [--scaling weak|strong]
                    [--impl ours|reference]

One STEP = one pass of the whole hot path over one batch of synthetic input: for every frequency of the
config, emit / walk / deposit / scatter all packages (soc_simulate_spectrum: one persistent photon kernel per
frequency, rows a1-a10 of DESIGN.md), then the energy-balance temperature update (row a11).  Default workload:
BASELINE.json configs[4] ("config 5": 256^3 lognormal cloud, 10 point sources + background, 128 frequencies,
1e7 packages per frequency, temperature update; one of its 3 iterations per step) -- the largest single-GPU
configuration; see DESIGN.md "Measurement" for why configs[1] (a single ~1 ms launch) is not the default.

--gpus N > 1: one process per GPU over NCCL.  Under torchrun (WORLD_SIZE set) the ranks are the launcher's; run
directly, bench.py re-executes itself under `python -m torch.distributed.run --standalone --nproc-per-node N`.
--scaling weak (default): every rank runs the full package count with seed + rank (independent realisations,
mean by one all-reduce); strong: the package ids of ONE seed are split over the ranks.

Prints ONE JSON line (rank 0).  `value` = cell-steps of all ranks per second of step time (device time, CUDA
events on the launching stream, max over ranks), inputs resident in HBM.  `e2e` = the same through
soc_run_host with pinned HOST buffers (model upload, simulation, download of absorbed energy and
temperatures inside the timed region).  `roofline` / `cpu_baseline` as described in DESIGN.md.

`--impl reference` times the CPU oracle (oracle/, fp64, as it stands) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "photon-package cell-steps/sec per frequency"
UNIT = "cell-steps/s"
ALGO_BYTES_PER_STEP = 12.0          # 4 B density gather + 8 B fp64 scatter-add
WORKLOADS = {
    "1": "configs[0]: regular 32^3 uniform, tau=1, albedo 0.5, g=0, background, 1e5 packages",
    "2": "configs[1]: regular 64^3 lognormal, peak tau 10, albedo 0.6, g=0.6, background, 1e6 packages",
    "3": "configs[2]: regular 128^3 lognormal, 2 point sources + background, 64 frequencies, 4e6 packages/frequency, temperature update",
    "4": "configs[3] (rule as written, theta=4): octree root 64^3, 4 levels, ~3.4M leaves, background, 32 frequencies, 1e6 packages/frequency",
    "4p": "configs[3] (size as written, theta=2): octree root 64^3, 4 levels, ~10M leaves, background, 32 frequencies, 1e6 packages/frequency",
    "5": "configs[4]: regular 256^3 lognormal, 10 point sources + background, 128 frequencies, 1e7 packages/frequency, temperature update (one of the 3 iterations per step)",
}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU every 100 ms while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index = index
        self.stop_flag = threading.Event()
        self.sm, self.reasons, self.sm_max, self.err = [], set(), None, None

    def run(self):
        try:
            import pynvml as nv
            nv.nvmlInit()
            h = nv.nvmlDeviceGetHandleByIndex(self.index)
            self.sm_max = int(nv.nvmlDeviceGetMaxClockInfo(h, nv.NVML_CLOCK_SM))
            names = {
                getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
                getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
                getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
                getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
            }
            get = getattr(nv, "nvmlDeviceGetCurrentClocksEventReasons", None) or nv.nvmlDeviceGetCurrentClocksThrottleReasons
            while not self.stop_flag.is_set():
                self.sm.append(int(nv.nvmlDeviceGetClockInfo(h, nv.NVML_CLOCK_SM)))
                mask = int(get(h))
                for bit, name in names.items():
                    if mask & bit:
                        self.reasons.add(name)
                self.stop_flag.wait(0.1)
        except Exception as e:      # noqa: BLE001 -- the sampler must never kill the bench
            self.err = repr(e)

    def summary(self):
        d = {"sm_mhz": (float(np.median(self.sm)) if self.sm else None), "sm_max_mhz": self.sm_max,
             "reasons": sorted(self.reasons), "samples": len(self.sm)}
        if self.err:
            d["error"] = self.err
        return d


def physical_gpu_index(local_rank):
    vis = os.environ.get("CUDA_VISIBLE_DEVICES")
    if vis:
        try:
            return int(vis.split(",")[local_rank])
        except Exception:
            return local_rank
    return local_rank


# ------------------------------------------------------------------------------------------------ CPU oracle legs
def oracle_sample(P, target_s, threads):
    """Time the oracle, as it stands, on a bounded sample of the workload: equal package-id subsets (straddling
    the background / point-source boundary) at four frequencies spread over the grid.  Returns
    (cell_steps, seconds, description)."""
    import oracle
    og = oracle.Grid(P.nx, P.ny, P.nz, P.n_cells, P.rho, P.child)
    freqs = sorted({int(round(x)) for x in np.linspace(0, P.n_freq - 1, 4)})
    n = P.n_packages

    def run(count):
        steps = 0
        t0 = time.perf_counter()
        for f in freqs:
            begin = max(0, n // 2 - count // 2)
            cnt = min(count, n - begin)
            _, res, _, _ = oracle.simulate(og, P.kabs[f], P.ksca[f], P.g[f], f, P.sources(f), n, P.seed, 1.0,
                                           begin, cnt, threads=threads)
            steps += res.cell_steps
        return steps, time.perf_counter() - t0

    probe = min(n, 4000 * threads)
    s0, t0 = run(probe)
    rate = s0 / max(t0, 1e-6)
    count = int(min(n, max(probe, probe * target_s / max(t0, 1e-6))))
    steps, secs = run(count)
    desc = (f"package ids [n/2-{count // 2}, n/2+{count - count // 2}) of {n} at frequency indices {freqs} "
            f"({len(freqs) * count} packages, {steps} cell-steps; calibration run {rate:.3g} steps/s)")
    return steps, secs, desc


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_1812_06632_b200 import inputs
    P = inputs.make_config(args.config)
    threads = max(1, min(32, os.cpu_count() or 1))
    per_step_target = max(2.0, min(20.0, 120.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(P, per_step_target / 4, threads)
    tot_steps, tot_s, desc = 0, 0.0, ""
    for _ in range(args.steps):
        s, t, desc = oracle_sample(P, per_step_target, threads)
        tot_steps += s
        tot_s += t
    v = tot_steps / tot_s
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / max(1, args.steps), "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOADS[args.config], "sample_per_step": desc},
            "cpu_baseline": {"value": v, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------------------------------------ CUDA path
def run_ours(args):
    import torch
    import torch.distributed as dist
    from paper_1812_06632_b200 import dist as socdist
    from paper_1812_06632_b200 import inputs, soc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback; use --impl reference for the oracle)")
    if world != args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={world}")
    if local_rank >= torch.cuda.device_count():
        raise SystemExit(f"bench.py: rank {rank} has no GPU (LOCAL_RANK {local_rank}, {torch.cuda.device_count()} visible)")
    torch.cuda.set_device(local_rank)
    socdist.init("nccl", rank, world, local_rank)
    soc.load()

    P = inputs.make_config(args.config)
    if args.packages:
        P.n_packages = int(args.packages)
    shard = socdist.plan(args.scaling, rank, world, P.n_packages, P.seed)
    G = soc.Grid.from_problem(P)
    G.set_option("timing", 1)
    for kv in args.opt:
        k, v = kv.split("=")
        G.set_option(k, int(v))
    srcs = [P.sources(f) for f in range(P.n_freq)]
    has_T = P.table_T is not None
    Aint = torch.zeros(P.n_total, dtype=torch.float64, device="cuda")
    T = torch.zeros(P.n_total, dtype=torch.float32, device="cuda")
    l2_bytes = int(torch.cuda.get_device_properties(local_rank).L2_cache_size)
    flush = torch.empty(max(256 << 20, 2 * l2_bytes), dtype=torch.uint8, device="cuda")      # 2 x L2 (B200: 126 MB)
    stream = torch.cuda.current_stream()

    def step(want_results=False):
        Aint.zero_()
        res = G.simulate_spectrum(srcs, P.n_packages, shard.seed, Aint, shard.pkg_begin, shard.pkg_count,
                                  want_results=want_results, stream=stream)
        socdist.combine(Aint, shard)
        if has_T:
            G.update_temperatures(Aint, P.t_scale, P.table_T, P.e_min, P.e_max, T, stream=stream)
        return res

    # ---- warm-up (the first warm-up pass also fetches the device counters: the walk is a deterministic function of
    # (seed, ids), so the counts are those of every later step), and conservation THROUGH THE CELLS: what the cells
    # of this rank hold after the pass = sum_f w_f (emitted_f - escaped_f); the counters alone cannot show a lost
    # scatter-add, and "escaped" is derived from the deposits for most packages (soc.h weight_drift)
    Aint.zero_()
    res = G.simulate_spectrum(srcs, P.n_packages, shard.seed, Aint, shard.pkg_begin, shard.pkg_count, stream=stream)
    w_f = G.freq_weights()
    budget = float(sum(w_f[f] * (res[f].emitted - res[f].escaped) for f in range(P.n_freq)))
    cons_cells = abs(float(Aint.sum()) - budget) / budget
    steps_f = np.array([r.cell_steps for r in res], dtype=np.float64)
    cons = max(abs(r.emitted - r.absorbed - r.escaped) / r.emitted for r in res if r.emitted > 0)
    drift = max(r.weight_drift for r in res)
    scat_total = sum(r.scatterings for r in res)
    for _ in range(max(1, args.warmup - 1)):
        step()
    torch.cuda.synchronize()

    # ---- timed region
    sampler = ClockSampler(physical_gpu_index(local_rank))
    sampler.start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = soc.launch_count()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    kern_ms = np.zeros(P.n_freq)
    t_wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.fill_(k & 0xff)                    # L2 flush between timed steps (outside the event pair)
        ev[k][0].record(stream)
        step()
        ev[k][1].record(stream)
        ev[k][1].synchronize()
        kern_ms += G.timings_ms()
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    t_wall = time.perf_counter() - t_wall0
    launches = soc.launch_count() - launches0
    sampler.stop_flag.set()
    sampler.join(2.0)
    step_ms = float(sum(a.elapsed_time(b) for a, b in ev))
    kern_ms /= max(1, args.steps)

    job = socdist.job_totals(step_ms, float(steps_f.sum()), float(launches), world, device="cuda")
    job_steps = job["cell_steps"]                # cell-steps of all ranks in one step
    job_launches = job["launches"]
    ms_per_step = job["step_ms"] / args.steps
    value = job_steps / (ms_per_step * 1e-3)

    # ---- end to end through the host-buffer entry (soc_run_host)
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory().numpy()        # noqa: E731
    Ph = dataclasses.replace(P, rho=pin(P.rho), child=None if P.child is None else pin(P.child), seed=shard.seed)
    # (soc_run_host runs whole package counts: the e2e figure of a strong-scaling run is per-rank full work, not reported)
    a_out = torch.zeros(P.n_total, dtype=torch.float64).pin_memory().numpy()
    t_out = torch.zeros(P.n_total, dtype=torch.float32).pin_memory().numpy()
    h2d = Ph.rho.nbytes + (0 if P.child is None else Ph.child.nbytes) + 4 * 8 * P.n_freq + \
        (0 if not has_T else 4 * len(P.table_T))
    d2h = a_out.nbytes + (t_out.nbytes if has_T else 0)
    # (median of three calls, every call's time kept in the line: a call creates and destroys a grid -- a dozen cudaMalloc /
    #  cudaFree, pinned staging buffers, a stream -- and one call in ten on the gpurun boxes takes 50-500 ms longer for it)
    n_e2e = max(1, min(args.steps, 3))
    # the first call is the warm-up of the others; it is timed too, with the library's buffer caches emptied before it:
    # what a process pays for its first soc_run_host (every device array allocated afresh)
    soc.release_cached_memory()
    t0 = time.perf_counter()
    soc.run_host(Ph, n_iter=1, absorbed_out=a_out, T_out=t_out if has_T else None)                # warm-up
    e2e_cold_s = time.perf_counter() - t0
    if world > 1:
        dist.barrier()
    e2e_runs = []
    for _ in range(n_e2e):
        t0 = time.perf_counter()
        soc.run_host(Ph, n_iter=1, absorbed_out=a_out, T_out=t_out if has_T else None)
        e2e_runs.append(time.perf_counter() - t0)
    e2e_s = float(np.median(e2e_runs))
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t[0])
    e2e_value = job_steps / e2e_s

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (photon kernel): algorithmic bytes per launch / mean launch time
    peak, peak_src = measured_peaks()
    mean_launch_ms = float(kern_ms.mean())
    algo_bytes = ALGO_BYTES_PER_STEP * float(steps_f.mean())
    achieved = algo_bytes / (mean_launch_ms * 1e-3) / 1e9
    # consecutive frequencies overlap on two streams and soc_get_timings attributes to a launch the advance of the
    # completion front, which alternates between long and short where the launches of one frequency are a sequence of
    # phases (slab-blocked launches): the per-frequency rate is therefore taken over pairs of consecutive frequencies
    pair_ms, pair_steps = kern_ms.copy(), steps_f.copy()
    for i in range(0, len(kern_ms) - 1, 2):
        pair_ms[i] = pair_ms[i + 1] = kern_ms[i] + kern_ms[i + 1]
        pair_steps[i] = pair_steps[i + 1] = steps_f[i] + steps_f[i + 1]
    per_f = pair_steps / (pair_ms * 1e-3)
    roof = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
            "traffic": None, "peak_source": peak_src,
            "kernel": "production photon kernel, chosen per frequency: photon_q_kernel (regular grids beyond L2: slab-blocked, "
                      "one launch per phase, + slab_emit_kernel) / photon_fast_kernel; a 'launch' below = all launches of one frequency",
            "algorithmic_bytes_per_launch": algo_bytes, "mean_launch_ms": mean_launch_ms,
            "kernel_share_of_step": float(kern_ms.sum() / ms_per_step)}
    tr = ncu_traffic(args.config)
    if tr:
        roof["traffic"] = tr["bytes_per_cell_step"] * float(steps_f.mean())
        roof["traffic_source"] = tr["source"]
        roof["traffic_measured_in_run"] = False        # carried from the committed ncu capture named in traffic_source
        roof["traffic_bytes_per_cell_step"] = tr["bytes_per_cell_step"]
    roof["algorithmic_bytes_note"] = ("12 B per cell-step is SURVEY.md 8d.4's contract figure (4 B density + 8 B fp64 add); the path "
                                      "as run adds into an fp32 per-launch accumulator: 4 B + 4 B = 8 B per cell-step")
    roof["achieved_8B"] = achieved * 8.0 / ALGO_BYTES_PER_STEP
    if world == 1 and not args.no_probes:
        roof["components"] = roofline_components(G, P, srcs, shard, Aint, stream, steps_f, kern_ms, peak, roof.get("traffic"))

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": args.scaling,
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "dtype_note": "fp32 package state, weights and per-launch accumulator; fp64 frequency integral and totals",
            "config": {"workload": WORKLOADS[args.config], "cells": int(P.n_total), "n_freq": int(P.n_freq),
                       "packages_per_frequency": int(P.n_packages),
                       "parallelism": "single GPU" if world == 1 else (
                           f"{world} ranks, seed + rank each (independent realisations), one fp64 all-reduce" if args.scaling == "weak"
                           else f"{world} ranks, package ids of one seed split evenly, one fp64 all-reduce"),
                       "l2": f"flushed between timed steps ({flush.numel() >> 20} MB fill; L2 {l2_bytes} B)"},
            "packages_per_s": (world if args.scaling == "weak" else 1) * P.n_packages * P.n_freq / (ms_per_step * 1e-3),
            "cell_steps_per_s_per_frequency": {"median": float(np.median(per_f)), "min": float(per_f.min()),
                                               "max": float(per_f.max()), "note": "over pairs of consecutive frequencies"},
            "cell_steps_per_step": job_steps, "scatterings_per_step_rank0": float(scat_total),
            "cell_steps_per_frequency_rank0": [int(x) for x in steps_f],
            "launch_ms_per_frequency_rank0": [round(float(x), 4) for x in kern_ms],
            "energy_conservation_rel": cons_cells,
            "energy_conservation": {"cells_vs_emitted_minus_escaped": cons_cells, "counters_emitted_absorbed_escaped": cons,
                                    "weight_drift_max": drift,
                                    "note": "cells: |sum_cells absorbed_int - sum_f w_f (emitted - escaped)| / sum; weight_drift: max "
                                            "|w - (1 - deposits)| over escaped packages (fp32 running weight against the deposits made)"},
            "clocks": sampler.summary(),
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "api": "soc_run_host (pinned host buffers)", "s_per_step": e2e_s,
                    "s_per_step_runs": [round(x, 4) for x in e2e_runs],
                    "s_first_call_cold_caches": round(e2e_cold_s, 4),
                    **({"note": "soc_run_host runs whole package counts: under --scaling strong every rank runs the full "
                                "problem end to end, so this is the single-GPU end-to-end figure"} if args.scaling == "strong" and world > 1 else {})},
            "gpu_launches": job_launches,
            "wall_s_timed_region": t_wall,
            "roofline": roof}

    # ---- the iterated run (rows f1 / f3, soc_iterate): constant sources once, then two iterations of dust re-emission with
    # emission-weighted package counts, reference field and ALI -- outside the timed region of the headline metric, timed
    # by wall clock around the call (it synchronises); one untimed call first (lazy per-grid buffers)
    if world == 1 and has_T and not args.no_iterate:
        try:
            n_req = [int(P.n_packages), int(P.n_packages)]
            it_s, hist = None, None
            for _ in range(2):
                torch.cuda.synchronize()
                t0 = time.perf_counter()
                hist = G.iterate(srcs, P.n_packages, P.seed, n_req, P.t_scale, P.table_T, P.e_min, P.e_max, Aint, T,
                                 mode="weighted", cap=10000, reference_field=True, ref_start=1, ali=True, stream=stream)
                it_s = time.perf_counter() - t0
            it_steps = float(sum(h["cell_steps"] for h in hist))
            line["iterate"] = {"value": it_steps / it_s, "unit": UNIT, "s_per_call": round(it_s, 4),
                               "cell_steps_per_call": it_steps, "packages_per_iteration": [int(h["n_packages"]) for h in hist],
                               "api": "soc_iterate: constant sources + 2 dust iterations (weighted counts, cap 10000, reference "
                                      "field, ALI), incl. counts, scans and temperature updates; second of two calls"}
        except Exception as exc:                         # the headline line must not depend on this leg
            line["iterate"] = {"error": str(exc)[:300]}

    if world == 1 and not args.no_cpu_baseline:
        threads = max(1, min(32, os.cpu_count() or 1))
        s, t, desc = oracle_sample(P, 15.0, threads)
        line["cpu_baseline"] = {"value": s / t, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def ncu_traffic(config):
    """DRAM bytes per cell-step of the photon kernel from the NEWEST committed ncu capture: profiles/r*_ncu_dram_traffic.csv
    (columns: config, kernel, cell_steps, dram_read_bytes, dram_write_bytes, weight, source -- one row per captured launch,
    written from the `ncu --set full` capture named in `source`; weight = how many launches of a pass the row stands for,
    so that a config whose frequencies run two different kernels is averaged in the right proportion).  Read at run time so that the figure cannot outlive the capture it came from; None when
    no capture of this config is committed."""
    import csv
    import glob
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_ncu_dram_traffic.csv")))
    for path in reversed(files):
        try:
            with open(path) as fh:
                rows = [r for r in csv.DictReader(fh) if r.get("config") == str(config)]
        except Exception:
            continue
        if rows:
            wt = [float(r.get("weight") or 1.0) for r in rows]
            steps = sum(w * float(r["cell_steps"]) for w, r in zip(wt, rows))
            byts = sum(w * (float(r["dram_read_bytes"]) + float(r["dram_write_bytes"])) for w, r in zip(wt, rows))
            return {"bytes_per_cell_step": byts / steps,
                    "source": f"{os.path.relpath(path, ROOT)} ({'; '.join(sorted({r['source'] for r in rows}))})"}
    return None


def roofline_components(G, P, srcs, shard, Aint, stream, steps_f, kern_ms, hbm_peak, traffic):
    """north_star's "achieved fraction of the gather and atomic roofline": request rates of the photon
    kernels against ceilings measured in the same run.
      requests  = what the lanes issued, counted on the device by the "stats" variant of the same kernels in one extra
                  pass (the walk is a deterministic function of (seed, ids): the timed passes issue exactly these)
      ceilings  = soc_probe_throughput, independent random accesses with no arithmetic, (a) over an L2-RESIDENT footprint
                  (32 MB): the request rate the L1 -> L2 path sustains = the ceiling; (b) over the config's own footprint
                  (8 B per cell): the NO-LOCALITY FLOOR -- every access its own sector, DRAM misses included; the walk
                  beats it through the brick layout and L2 reuse along a path, so a ratio > 1 there is expected
      dram      = ncu DRAM bytes per cell-step of the newest committed capture x cell-steps/s, against the measured HBM peak"""
    from paper_1812_06632_b200 import soc
    import torch
    G.set_option("stats", 1)
    Aint.zero_()
    res = G.simulate_spectrum(srcs, P.n_packages, shard.seed, Aint, shard.pkg_begin, shard.pkg_count, stream=stream)
    G.set_option("stats", 0)
    torch.cuda.synchronize()
    secs = float(kern_ms.sum()) * 1e-3
    gathers, reds = float(sum(r.gather_requests for r in res)), float(sum(r.red_requests for r in res))
    steps = float(steps_f.sum())
    import torch
    l2_bytes = int(torch.cuda.get_device_properties(torch.cuda.current_device()).L2_cache_size)
    vec = P.child is None and 8 * int(P.n_total) > l2_bytes // 126 * 64      # photon_q_kernel (16-byte requests) carries such grids (soc.cu l2_share)
    n_ops = 1 << 30
    rate = lambda kind, fp: n_ops / (soc.probe_throughput(kind, fp, n_ops) * 1e-3)          # noqa: E731
    l2_fp, cfg_fp = min(32 << 20, l2_bytes // 4), 8 * int(P.n_total)
    kg, kr = (6, 4) if vec else (0, 2)
    ceil_g, ceil_r = rate(kg, l2_fp), rate(kr, l2_fp)
    floor_g, floor_r, floor_pair = rate(kg, cfg_fp), rate(kr, cfg_fp), rate(5, cfg_fp)
    comp = {
        "request_width": "16 B (ld.global.nc.v4 / red.global.add.v4.f32, photon_q_kernel)" if vec else "4 B (ld.global.nc / red.global.add.f32)",
        "gather": {"requests_per_cell_step": gathers / steps, "per_s": gathers / secs, "ceiling_per_s": ceil_g,
                   "frac": gathers / secs / ceil_g, "no_locality_floor_per_s": floor_g},
        "red": {"requests_per_cell_step": reds / steps, "per_s": reds / secs, "ceiling_per_s": ceil_r,
                "frac": reds / secs / ceil_r, "no_locality_floor_per_s": floor_r},
        "gather_plus_red_no_locality_floor": {"pairs_per_s": floor_pair, "cell_steps_per_s": steps / secs,
                                              "ratio": steps / secs / floor_pair,
                                              "note": "a FLOOR, not a ceiling: one 4-byte gather + one fp32 add per uniformly random "
                                                      "cell of the config's footprint; ratio > 1 = locality the walk exploits"},
        "ceiling_footprint_bytes": l2_fp, "floor_footprint_bytes": cfg_fp,
    }
    # the ceilings over footprints from L1-sized to beyond L2, uniform addresses, and the hot-spot case
    # -- every thread of the probe into the 343 cells of a hot_r = 3 cube around a source: contended
    # global reductions in fp32 / fp64 against shared-memory partial sums with one fp64 reduction per cell and block
    try:
        n_small = 1 << 28
        r2 = lambda kind, fp, n=n_small: n / (soc.probe_throughput(kind, fp, n) * 1e-3)          # noqa: E731
        comp["ceilings_ops_per_s"] = {
            "footprint_bytes": [128 << 10, 1 << 20, 8 << 20, 64 << 20, 256 << 20],
            "gather_4B": [r2(0, fp) for fp in (128 << 10, 1 << 20, 8 << 20, 64 << 20, 256 << 20)],
            "red_f32": [r2(2, fp) for fp in (128 << 10, 1 << 20, 8 << 20, 64 << 20, 256 << 20)],
            "red_f64": [r2(1, fp) for fp in (128 << 10, 1 << 20, 8 << 20, 64 << 20, 256 << 20)],
            "hot_spot_343_cells": {"red_f32": r2(2, 343 * 4, 1 << 26), "red_f64": r2(1, 343 * 8, 1 << 26),
                                   "shared_f32_then_one_red_f64_per_cell_and_block": r2(7, 343 * 4, 1 << 28)},
            "note": "uniformly random addresses within the footprint, no arithmetic; hot spot = all lanes into 343 cells",
        }
    except Exception as exc:                             # an older library without probe kind 7
        comp["ceilings_ops_per_s"] = {"error": str(exc)[:200]}
    fr = [comp["gather"]["frac"], comp["red"]["frac"]]
    if traffic:
        dram = traffic * len(steps_f) / secs / 1e9
        comp["dram"] = {"GB_per_s": dram, "peak_GB_per_s": hbm_peak, "frac": dram / hbm_peak}
        fr.append(dram / hbm_peak)
    comp["frac_max"] = max(fr)
    comp["binding"] = ["gather", "red", "dram"][int(np.argmax(fr))]
    return comp


def spawn_ranks(args):
    """`python bench.py --gpus N` without a launcher: re-execute under torch.distributed.run, one rank per GPU."""
    import subprocess
    import torch
    if torch.cuda.device_count() < args.gpus:
        raise SystemExit(f"bench.py: --gpus {args.gpus} but only {torch.cuda.device_count()} CUDA device(s) visible")
    cmd = [sys.executable, "-m", "torch.distributed.run", "--standalone", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--local-addr", "127.0.0.1", os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", choices=sorted(WORKLOADS), default="5")
    ap.add_argument("--scaling", choices=["weak", "strong"], default="weak",
                    help="weak: every rank the full package count with seed + rank; strong: ids of one seed split over ranks")
    ap.add_argument("--packages", type=int, default=0, help="override packages per frequency (debugging only)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-iterate", action="store_true", help="skip the soc_iterate leg (dust re-emission iterations)")
    ap.add_argument("--no-probes", action="store_true", help="skip the random gather / scatter-add ceiling probes")
    ap.add_argument("--opt", action="append", default=[], help="library tuning knob key=value (soc_set_option)")
    args = ap.parse_args()
    if args.steps < 1 or args.warmup < 0:
        raise SystemExit("need --steps >= 1 and --warmup >= 0")
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 2)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
