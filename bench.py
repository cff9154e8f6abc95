#!/usr/bin/env python
"""bench.py -- throughput of the tCW track-sum hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config all|cfg1..cfg5] [--impl ours|reference]

One "step" = one pass of the whole hot path (Doppler table, spin-down table, gather-accumulate,
candidate reduction: SURVEY.md section 8(a) rows a1-a6) over the whole template grid of a
workload.  With no --config (= "all") the headline workload is cfg4 = BASELINE.json:configs[3],
the largest single-GPU configuration (three days of 8-s SFTs with gaps, 500-3000 Hz, float32
normalised power, 1.67 GB; 20000 f0 x 64 tau x 9 n x 1 sky = 11.52 M templates), and the same
measurements for cfg2, cfg3 (uint8 and bit-packed) and cfg5 are carried in `per_config`.

Printed: ONE JSON line.  `value` = nominal template-SFT lookups/s (n_templates * n_sft per
step, all ranks) with inputs resident in HBM; `e2e` = the same through tcw_create_async(HOST
spectrogram) + tcw_search_host(HOST outputs) + tcw_destroy, copies inside the timed region;
`roofline` = compulsory bytes B_comp of DESIGN.md section 6 over the gather-accumulate kernel's
device time against the measured HBM peak (the model BASELINE.json asks for); `roofline_binding`
= the bound that actually binds -- warp-instruction issue -- with the kernel's instruction count
(profiles/ncu_summary.json: ncu captures of the shipped build) over its device time against the
issue rate tcw_measure_peaks measures in this process; `cpu_baseline` = oracle/ timed on this
box's host cores on a bounded sample (the oracle is the unoptimised literal definition: a
reported baseline, not a target).

N > 1 (torchrun): strong scaling.  The flattened (sky, tau, n) group index of the headline grid
is cut into N contiguous ranges (shard_groups), rank r searches its range with tcw_search_groups,
the spectrogram is replicated, and there is no data-path collective.

`--impl reference` times the oracle (oracle/, the paper's definition on the host cores); for
this paper there is no reference code to install.
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "template-SFT lookups/s"
UNIT = "lookups/s"
C_LIGHT = 299792458.0
HEADLINE = "cfg4"
FP64_PER_LOOKUP = 34.0      # FP64 instructions per lookup of sum_bank_kernel's fast path (SASS count)
PER_CONFIG = (("cfg2", "f32"), ("cfg3", "u8"), ("cfg3", "bits"), ("cfg5", "bits"))
L2_BYTES = 126e6


def load_ncu_summary():
    """profiles/ncu_summary.json: per workload, what `ncu --set full` measured on ONE launch of the
    gather-accumulate kernel of the shipped build (DRAM traffic, warp instructions, issue-active), the
    commit it was captured at and the profile file with the full command.  Written by
    `python -m paper_2507_07816_b200.profiling summary ...`; bench.py only reads it."""
    path = os.path.join(ROOT, "profiles", "ncu_summary.json")
    if not os.path.exists(path):
        return {}
    with open(path) as f:
        return json.load(f)


# ----------------------------------------------------------------------------- helpers
# The driver keeps the tail of the line: prose and provenance strings stay out of it unless --verbose
# (they are in DESIGN.md section 6), and floats carry five significant digits.
COMPACT_DROP = ("note", "traffic_source", "inst_source", "peak_source", "path", "timing", "samples", "searches_averaged")


def slim_block(b):
    """A per_config entry as the default line carries it: the numbers (time, value, rooflines, e2e, launches), the
    workload by name; the launch geometry, stage split, clocks and full config are in the --verbose line."""
    keep = ("value", "ms_per_step", "kernel_ms", "inband_fraction", "roofline", "roofline_binding", "e2e", "gpu_launches",
            "results", "n", "n_sft", "us_per_template", "exact_chain_lookups", "templates_per_s")
    out = {"workload": b["config"]["workload"].split(" ")[0] + ":" + b["config"]["format"]} if "config" in b else {}
    if "launch" in b:
        out["kernel"] = b["launch"].get("kernel")
    out.update({k: b[k] for k in keep if k in b})
    for r in ("roofline", "roofline_binding"):
        if r in out:
            out[r] = {k: v for k, v in out[r].items() if k not in ("kernel_ms", "algorithmic_bytes_per_launch", "inst_per_launch",
                                                                   "issue_active_pct_ncu", "fp64_pipe_pct_ncu", "bytes_per_inband_lookup")}
    if "cpu_baseline" in b:
        out["cpu_baseline"] = {k: b["cpu_baseline"][k] for k in ("value", "cores", "kind") if k in b["cpu_baseline"]}
    return out


def compact(obj, drop=COMPACT_DROP, top=True):
    if isinstance(obj, dict):
        return {k: compact(v, drop, False) for k, v in obj.items()
                if top or k not in drop or k == "sample"}
    if isinstance(obj, (list, tuple)):
        return [compact(v, drop, False) for v in obj]
    if isinstance(obj, float):
        return float(f"{obj:.5g}") if math.isfinite(obj) else None
    return obj


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def compulsory_bytes(w, sky=None):
    """B_comp of SURVEY.md section 8(d) / DESIGN.md section 6: for every (sky, tau, n) group and
    SFT, the bins between the tracks of the group's first and last f0, clipped to the band, times
    the bytes per bin; plus 4 B per template (out_stat) and 8 B per group (out_best).  This is a
    byte model for the roofline, evaluated with numpy; it is not part of the search."""
    sky = w.sky if sky is None else sky
    bpb = {"f32": 4.0, "u8": 1.0, "bits": 0.125}[w.fmt]
    k_min = int(round(w.f_min * w.T_sft))
    t = w.timestamps
    ok = t >= w.T0
    total = 0.0
    D = 1.0 + (w.velocities @ np.asarray(sky).T) / C_LIGHT           # [n_sft][n_sky]
    for tau in w.tau:
        base = np.where(ok, (t - w.T0) / tau + 1.0, 1.0)
        for n in w.brk:
            g = np.power(base, 1.0 / (1.0 - n))[:, None] * D * w.T_sft   # [n_sft][n_sky]
            k_lo = np.rint(w.f0[0] * g) - k_min
            k_hi = np.rint(w.f0[-1] * g) - k_min
            lo = np.maximum(k_lo, 0)
            hi = np.minimum(k_hi, w.n_bins - 1)
            bins = np.where(ok[:, None], np.maximum(hi - lo + 1, 0), 0)
            total += float(bins.sum()) * bpb
    n_groups = len(sky) * len(w.tau) * len(w.brk)
    return total + 4.0 * n_groups * len(w.f0) + 8.0 * n_groups


class ClockSampler:
    """nvidia-smi clocks and throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._pump, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _pump(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, mx, pw, reasons = [], [], [], set()
        for line in self.lines:
            f = [x.strip() for x in line.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1])); pw.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": float(np.median(sm)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(w, budget_s: float, max_groups: int | None = None, literal: bool = False):
    """The oracle as it stands (oracle/tcw_oracle.c, OpenMP over templates) timed on ONE call.
    Sample = a seeded random sub-grid of WHOLE groups: some tau values x some sky points x every
    braking index x every f0, evaluated whole, so that the oracle's per-(tau, n) spin-down table is
    built for the sampled rows only and the rate does not depend on the sample size (round 2 built
    the table of the whole grid for every sample: VERDICT r2 #7).  A first call on one (sky, tau) row
    sizes the sample to about `budget_s`.  literal=True: the oracle's literal mode (one correctly
    rounded power per (template, SFT), no table: BASELINE.md section 2) on a prefix of that row."""
    import oracle
    oracle.build()
    rng = np.random.default_rng(7)
    tau_order, sky_order = rng.permutation(len(w.tau)), rng.permutation(len(w.sky))
    n_brk, n_f0 = len(w.brk), len(w.f0)

    def sub(n_tau, n_sky):
        return w.subgrid(tau=np.sort(tau_order[:n_tau]), sky=np.sort(sky_order[:n_sky]))

    if literal:
        row, m = sub(1, 1), min(256, n_f0)
        t0 = time.perf_counter()
        oracle.evaluate(row, sel=np.arange(m), literal=True)
        t1 = time.perf_counter() - t0
        m = int(max(m, min(row.n_templates, m * budget_s / t1)))
        t0 = time.perf_counter()
        r = oracle.evaluate(row, sel=np.arange(m), literal=True)
        t_used = time.perf_counter() - t0
        n_templates, what = m, f"the first {m} templates of one (sky,tau) row of {w.name}, literal mode"
    else:
        t0 = time.perf_counter()
        oracle.evaluate(sub(1, 1))                                       # also loads the library
        t1 = time.perf_counter() - t0
        rows = max(1.0, budget_s / t1)
        if max_groups is not None:
            rows = max(1.0, min(rows, max_groups / n_brk))
        n_tau = int(min(len(w.tau), rows))
        n_sky = int(min(len(w.sky), max(1.0, rows / n_tau)))
        sw = sub(n_tau, n_sky)
        t0 = time.perf_counter()
        r = oracle.evaluate(sw)
        t_used = time.perf_counter() - t0
        n_templates = sw.n_templates
        what = f"{n_tau} tau x {n_sky} sky x all {n_brk} n = {n_tau * n_sky * n_brk} of {w.n_groups} whole groups of {w.name}"
    lookups = float(n_templates) * w.n_sft
    inband = float(r.n_inband.sum())
    return dict(value=lookups / t_used, unit=UNIT, cores=oracle.num_threads(), kind="oracle",
                inband_lookups_per_s=inband / t_used,
                sample=f"{what} in one call ({n_templates} templates x {w.n_sft} SFTs = {lookups:.3e} nominal, "
                       f"{inband:.3e} in-band lookups) in {t_used:.1f} s",
                seconds=t_used, templates=n_templates)


def workload_config(w, extra=None):
    """The keys that name the workload; identical in both arms (ours and --impl reference)."""
    cfg = {"workload": f"{w.name} (BASELINE.json:configs[{int(w.name[3:]) - 1}])", "format": w.fmt,
           "n_sft": int(w.n_sft), "n_bins": int(w.n_bins), "n_f0": len(w.f0), "n_tau": len(w.tau),
           "n_brk": len(w.brk), "n_sky": len(w.sky), "n_templates": int(w.n_templates),
           "spectrogram_bytes": int(w.spectrogram.nbytes),
           "l2_policy": ("input larger than L2 (no flush)" if w.spectrogram.nbytes > L2_BYTES else
                         "input smaller than L2: a 256 MB buffer is written between timed steps (L2 flush)")}
    if extra:
        cfg.update(extra)
    return cfg


def headline_name(args) -> tuple[str, str | None]:
    return (HEADLINE, None) if args.config == "all" else (args.config, args.format)


# ----------------------------------------------------------------------------- reference arm
def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    import tcw_inputs
    name, fmt = headline_name(args)
    w = tcw_inputs.make_workload(name, fmt=fmt)
    per_step = max(1.0, min(20.0, 60.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        time_oracle(w, per_step, max_groups=1)
    tot_lookups, tot_s, cores, samples = 0.0, 0.0, 0, []
    for _ in range(args.steps):
        r = time_oracle(w, per_step)
        tot_lookups += r["value"] * r["seconds"]
        tot_s += r["seconds"]
        cores = r["cores"]
        samples.append(r["sample"])
    value = tot_lookups / tot_s
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_s / args.steps,
            "higher_is_better": True, "scaling": "strong" if args.gpus > 1 else "weak", "vs_baseline": None,
            "dtype": "f64", "data": "synthetic", "config": workload_config(w),
            "note": "each step is a bounded sample of the workload evaluated by the oracle on the host cores",
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": samples[-1]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------- our arm
def measure_config(ctx, name, fmt, steps, warmup, e2e_steps, cpu_seconds, opts=None, weighted=False, one_thread=False):
    """Everything bench.py reports for ONE workload on this rank's GPU: device-resident throughput,
    stage times, both rooflines, end to end from host buffers, and the oracle on the host cores."""
    import torch
    tcw, tcw_inputs, dist = ctx["tcw"], ctx["tcw_inputs"], ctx["dist"]
    rank, world, dev = ctx["rank"], ctx["world"], ctx["dev"]
    opts = opts or {}

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    w = tcw_inputs.make_workload(name, fmt=fmt)
    key = f"{w.name}:{w.fmt}"
    grid = tcw.Grid.of(w)
    n_sft, n_f0 = w.n_sft, len(w.f0)
    # N > 1: contiguous whole-group ranges of nearly equal in-band WORK, not equal counts
    g_lo, g_hi = (tcw.shard_groups(grid.n_groups, rank, world, weights=tcw.group_work(grid, w.timestamps, w.T_sft, w.f_min, w.n_bins))
                  if world > 1 else (0, grid.n_groups))
    my_groups = g_hi - g_lo
    nominal = float(grid.n_templates) * n_sft                       # whole job, all ranks
    stream = torch.cuda.current_stream()

    h = tcw.Handle.from_workload(w, device=dev)
    # tcw_create alone (layout copy of a device-resident spectrogram into the padded pitch; untimed in
    # `value`, reported separately as SURVEY.md section 8(d) asks)
    spec_dev = torch.from_numpy(np.ascontiguousarray(w.spectrogram).view(np.int32) if w.spectrogram.dtype == np.uint32
                                else np.ascontiguousarray(w.spectrogram)).to(dev)
    tcw.Handle(spec_dev, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities).close()   # warm-up: the pool grows once
    torch.cuda.synchronize()
    t_c0 = time.perf_counter()
    for _ in range(3):
        tcw.Handle(spec_dev, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities).close()
    torch.cuda.synchronize()
    create_ms = 1e3 * (time.perf_counter() - t_c0) / 3
    del spec_dev
    for k, v in opts.items():
        h.set_option(k, v)
    out_stat = torch.empty((max(my_groups, 1), n_f0), dtype=h.stat_dtype, device=dev)
    out_best = torch.empty((max(my_groups, 1), 2), dtype=torch.int32, device=dev)

    if weighted:
        # NEXT-1: the weighted statistic + critical ratio (tcw_search_weighted) on the same workload,
        # device-resident weights; the step then produces Psi, s and the per-group best Psi
        mean1, var1 = (1.0, 1.0) if w.fmt == "f32" else (math.exp(-1.6), math.exp(-1.6) * (1 - math.exp(-1.6)))
        wts = torch.from_numpy(tcw_inputs.synthetic_weights(w.sky, w.timestamps, w.seed)).to(dev)
        shape4 = (len(w.sky), len(w.tau), len(w.brk), n_f0)
        out_psi = torch.empty(shape4, dtype=torch.float32, device=dev)
        out_stat = torch.empty(shape4, dtype=torch.float32, device=dev)

    def step():
        if my_groups == 0:
            return
        if weighted:
            h.search_weighted(grid, wts, mean1, var1, out_psi, out_stat, out_best)
        elif world > 1:
            h.search_groups(grid, g_lo, g_hi, out_stat, out_best)
        else:
            h.search(grid, out_stat, out_best)

    # L2 policy (timing rules): inputs larger than L2 need no flush; smaller ones get a 256 MB write between steps
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev) if w.spectrogram.nbytes <= L2_BYTES else None
    sampler = ClockSampler(ctx["local"])
    for _ in range(warmup):
        step()
    # short steps: keep warming until the GPU has been busy for 50 ms (clocks and power state settle)
    torch.cuda.synchronize()
    t_w = time.perf_counter()
    while time.perf_counter() - t_w < 0.05:
        step()
        torch.cuda.synchronize()
    h.set_option(tcw.TCW_OPT_TIMING, 1)
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    barrier()
    if rank == 0:
        sampler.start()
    t_host0 = time.perf_counter()
    for e0, e1 in evs:
        if flush is not None:
            flush.fill_(1)
        e0.record(stream)
        step()
        e1.record(stream)
    barrier()
    t_host = time.perf_counter() - t_host0
    clocks = sampler.stop() if rank == 0 else None
    ms_total = float(sum(e0.elapsed_time(e1) for e0, e1 in evs))
    stage_ms, n_timed = h.timing() if my_groups else ((0.0, 0.0, 0.0, 0.0), 0)
    h.set_option(tcw.TCW_OPT_TIMING, 0)
    info = h.info() if my_groups else {}
    if world > 1:
        t = torch.tensor([ms_total], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_total = float(t.item())
    ms_step = ms_total / steps
    value = nominal / (ms_step * 1e-3)

    # in-band lookups: the same search over an all-ones uint8 spectrogram counts them exactly
    inband = 0.0
    if rank == 0:
        ones = torch.ones((n_sft, w.n_bins), dtype=torch.uint8, device=dev)
        with tcw.Handle(ones, "u8", w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities) as h1:
            cnt, _ = h1.search(grid, want_best=False)
            torch.cuda.synchronize()
            inband = float(cnt.sum(dtype=torch.int64).item())
        del ones, cnt

    # ---- end to end through the C ABI with HOST buffers (copies inside the timed region)
    spec_np = np.ascontiguousarray(w.spectrogram)
    if spec_np.dtype == np.uint32:
        spec_np = spec_np.view(np.int32)
    spec_pin = torch.from_numpy(spec_np).pin_memory()
    skip_e2e = e2e_steps <= 0
    e2e_steps = max(1, min(steps, e2e_steps))
    if world == 1:
        stat_pin = torch.empty((len(w.sky), len(w.tau), len(w.brk), n_f0), dtype=h.stat_dtype).pin_memory()
        best_pin = torch.empty((grid.n_groups, 2), dtype=torch.int32).pin_memory()

        def e2e_step():
            # tcw_create_async: the pinned spectrogram travels in pieces while the search already runs;
            # tcw_search_host: outputs of 64 MiB or more come back part by part under the next part's search
            with tcw.Handle(spec_pin, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, async_upload=True) as hh:
                for k, v in opts.items():
                    hh.set_option(k, v)
                hh.search_host(grid, stat_pin.numpy(), best_pin.numpy())
        e2e_path = "tcw_create_async(pinned HOST spectrogram) + tcw_search_host(pinned HOST out_stat, out_best) + tcw_destroy"
    else:
        stat_pin = torch.empty((max(my_groups, 1), n_f0), dtype=h.stat_dtype).pin_memory()
        best_pin = torch.empty((max(my_groups, 1), 2), dtype=torch.int32).pin_memory()

        def e2e_step():
            with tcw.Handle(spec_pin, w.fmt, w.n_bins, w.f_min, w.T_sft, w.timestamps, w.velocities, async_upload=True) as hh:
                if my_groups:
                    hh.search_groups(grid, g_lo, g_hi, out_stat, out_best)
                    stat_pin.copy_(out_stat, non_blocking=True)
                    best_pin.copy_(out_best, non_blocking=True)
                    hh.check()
        e2e_path = ("per rank: tcw_create_async(pinned HOST spectrogram) + tcw_search_groups(own group range) + "
                    "device-to-host copy of its out_stat / out_best slices + tcw_check + tcw_destroy")
    for _ in range(0 if skip_e2e else 2):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(0 if skip_e2e else e2e_steps):
        e2e_step()                      # tcw_search_host / tcw_check synchronise before returning
    torch.cuda.synchronize()
    e2e_s = max(time.perf_counter() - t0, 1e-9)
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    h2d = int(world * (spec_np.nbytes + w.timestamps.nbytes + w.velocities.nbytes)
              + 8 * (len(w.f0) + len(w.tau) + len(w.brk) + 3 * len(w.sky)))
    d2h = int(4 * grid.n_templates + 8 * grid.n_groups)
    e2e_value = nominal * e2e_steps / e2e_s
    h.close()
    del spec_pin, stat_pin, best_pin, out_stat, out_best, flush
    torch.cuda.empty_cache()
    if rank != 0:
        return None

    peak, peak_src = load_peaks()
    b_comp = compulsory_bytes(w)
    sum_ms = stage_ms[1]
    dev_spec_bytes = float(n_sft) * w.n_bins * (4 if w.fmt == "f32" else 1)       # bit-packed input is expanded to one byte per bin
    unique_b = dev_spec_bytes + 4.0 * grid.n_templates + 8.0 * grid.n_groups
    achieved = b_comp / (sum_ms * 1e-3) / 1e9 if sum_ms > 0 else 0.0
    ncu = None if weighted else ctx["ncu"].get("captures", {}).get(key)      # the captures are of the unweighted kernels
    kernel_name = ("sum_skyblock2_kernel" if info.get("kernel") == "skyblock" and info.get("sky_block") == 256
                   else f"sum_{info.get('kernel')}_kernel")
    block = {
        "config": workload_config(w),
        "value": value, "unit": UNIT, "ms_per_step": ms_step,
        "templates_per_s": grid.n_templates / (ms_step * 1e-3),
        "inband_lookups_per_s": inband / (ms_step * 1e-3),
        "inband_fraction": inband / nominal,
        "create_ms": create_ms,
        "launch": {"kernel": info.get("kernel"), "tile_f0": info.get("tile"), "ctas": info.get("ctas"),
                   "smem_bytes": info.get("smem_bytes"), "sky_block": info.get("sky_block"),
                   "sft_chunks": info.get("chunks"), "chunk_rows": info.get("chunk_rows"), "ring_stages": info.get("stages"),
                   "kernels_per_step": info.get("launches"),
                   **({"statistic": "weighted s + critical ratio Psi (tcw_search_weighted), device-resident weights; "
                                    "the e2e leg times the unweighted tcw_search_host"} if weighted else {})},
        "stage_ms": {"tables": stage_ms[0], "sum": stage_ms[1], "best": stage_ms[2], "search": stage_ms[3],
                     "searches_averaged": n_timed, "host_wall_ms_per_step": 1e3 * t_host / steps},
        "kernel_ms": sum_ms,
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                     "traffic": (ncu["dram_bytes_read"] + ncu["dram_bytes_write"]) if ncu else None,
                     "traffic_source": ({"profile": ncu["profile"], "commit": ctx["ncu"].get("commit"), "kernel": ncu["kernel"]}
                                        if ncu else None),
                     "peak_source": peak_src, "kernel": kernel_name, "algorithmic_bytes_per_launch": b_comp, "kernel_ms": sum_ms,
                     "bytes_per_inband_lookup": b_comp / inband if inband else None,
                     # what must leave / enter HBM once: the spectrogram as the device holds it + the outputs.  `frac` above is
                     # BASELINE.json's per-group model, which L2 serves (frac > 1 = the model does not bind: see roofline_binding)
                     "unique_bytes": unique_b, "frac_unique": unique_b / (sum_ms * 1e-3) / 1e9 / peak if sum_ms > 0 else None,
                     "traffic_over_unique": ((ncu["dram_bytes_read"] + ncu["dram_bytes_write"]) / unique_b) if ncu else None},
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": e2e_steps, "ms_per_step": 1e3 * e2e_s / e2e_steps, "path": e2e_path},
        "gpu_launches": (info.get("launches") or 0) * steps,
        "clocks": clocks,
    }
    if skip_e2e:
        del block["e2e"]
    pk = ctx["peaks"]
    if ncu and pk and world == 1 and not opts and not weighted:
        inst = float(ncu["inst_executed"])
        ach = inst / (sum_ms * 1e-3)
        block["roofline_binding"] = {
            "bound": "issue", "achieved": ach, "peak": pk["issue_winst_per_s"], "unit": "warp instructions/s",
            "frac": ach / pk["issue_winst_per_s"],
            "inst_per_launch": inst, "inst_per_32_inband_lookups": 32.0 * inst / inband if inband else None,
            "issue_active_pct_ncu": ncu.get("issue_active_pct"), "fp64_pipe_pct_ncu": ncu.get("fp64_pipe_pct"),
            "inst_source": {"profile": ncu["profile"], "commit": ctx["ncu"].get("commit"), "kernel": ncu["kernel"],
                            "kernel_ms_under_ncu": ncu.get("duration_ms")},
            "peak_source": "tcw_measure_peaks in this process: independent FFMA streams, one warp instruction per scheduler per cycle",
            "note": "warp instructions of one launch (ncu capture of the shipped build) over the live CUDA-event time of the "
                    "kernel, against the measured issue rate; the instruction count per lookup is what a faster kernel lowers"}
        if info.get("kernel") == "staged" and ncu.get("l2_sectors") and pk.get("stage_box_copies_bytes_per_s"):
            # the other co-limit of the staged kernel: bytes its TMA copies draw from L2 (32-byte sectors of the ncu
            # capture) over the live kernel time, against what the same ring draws when it stages alone
            l2b = 32.0 * float(ncu["l2_sectors"])
            block["roofline_binding"]["staging"] = {
                "achieved_l2_bytes_per_s": l2b / (sum_ms * 1e-3), "peak_bytes_per_s": pk["stage_box_copies_bytes_per_s"],
                "frac": l2b / (sum_ms * 1e-3) / pk["stage_box_copies_bytes_per_s"], "l2_bytes_per_launch": l2b,
                "note": "L2 -> shared-memory traffic of the launch (lts__t_sectors of the ncu capture x 32 B) over the live kernel "
                        "time, against the rate the per-warp rings reach with tensor-map copies and no consumer (tcw_measure_peaks)"}
        if info.get("kernel") == "staged" and inband:
            block["roofline_binding"]["lookup_chain"] = {
                "achieved_inband_lookups_per_s": inband / (sum_ms * 1e-3), "peak_lookups_per_s": pk["chain_lookups_per_s"],
                "frac": inband / (sum_ms * 1e-3) / pk["chain_lookups_per_s"],
                "note": "the bare lookup chain of the staged kernel as it ships (two rows per block: DFMA, address, LDS.32, half a FADD2, half a VIMNMX3 per lookup) "
                        "measured alone by tcw_measure_peaks: staging, row metadata and band edges are what separates the two"}
    if world == 1 and cpu_seconds > 0:
        cb = time_oracle(w, cpu_seconds)
        block["cpu_baseline"] = {k: cb[k] for k in ("value", "unit", "cores", "kind", "sample", "inband_lookups_per_s")}
        block["cpu_baseline"]["templates_per_s"] = cb["templates"] / cb["seconds"]
        if one_thread:
            # the same oracle on one thread (all cores and one core), and its literal mode
            # (one correctly rounded power per lookup) on all cores; smaller samples -- the rate
            # no longer depends on the sample size
            import oracle
            all_threads = oracle.num_threads()
            oracle.set_num_threads(1)
            c1 = time_oracle(w, min(4.0, cpu_seconds))
            oracle.set_num_threads(all_threads)
            block["cpu_baseline"]["one_thread"] = {"value": c1["value"], "unit": UNIT, "cores": 1, "sample": c1["sample"]}
            cl = time_oracle(w, min(3.0, cpu_seconds), literal=True)
            block["cpu_baseline"]["literal"] = {"value": cl["value"], "unit": UNIT, "cores": cl["cores"], "sample": cl["sample"]}
    return block


def run_ours(args):
    import torch
    import torch.distributed as dist

    import paper_2507_07816_b200 as tcw
    import tcw_inputs

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the tCW path has no CPU fallback")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    tcw.load_library()
    if args.shard_table:
        return run_shard_table(args, tcw, tcw_inputs, dev)
    if args.shard:
        # one rank's share of an N-GPU strong-scaling run, timed alone on this GPU (no process group): what
        # rank R of `torchrun --nproc-per-node N bench.py --gpus N` executes, for boxes with a single GPU
        r, n = (int(x) for x in args.shard.split("/"))
        if world > 1 or not (0 <= r < n):
            raise SystemExit("bench.py: --shard R/N needs a single process and 0 <= R < N")
        return run_shard(args, tcw, tcw_inputs, dev, r, n)
    ctx = dict(tcw=tcw, tcw_inputs=tcw_inputs, dist=dist, rank=rank, world=world, local=local, dev=dev,
               ncu=load_ncu_summary(), peaks=None)
    if rank == 0:
        ctx["peaks"] = tcw.measure_peaks()          # issue / FP64 / LDS rates of this GPU, now

    opts = {}
    if args.kernel:
        opts[tcw.TCW_OPT_KERNEL] = tcw.KERNELS[args.kernel]
    if args.sky_block:
        opts[tcw.TCW_OPT_SKY_BLOCK] = args.sky_block
    if args.f0_per_lane:
        opts[tcw.TCW_OPT_F0_PER_LANE] = args.f0_per_lane
    if args.chunk_rows:
        opts[tcw.TCW_OPT_CHUNK_ROWS] = args.chunk_rows
    if args.stages:
        opts[tcw.TCW_OPT_STAGES] = args.stages
    if args.exact_index:
        opts[tcw.TCW_OPT_EXACT_INDEX] = 1
    if args.general_f0:
        opts[tcw.TCW_OPT_GENERAL_F0] = 1

    name, fmt = headline_name(args)
    cpu_s = 0.0 if args.no_cpu_baseline else args.cpu_seconds
    head = measure_config(ctx, name, fmt, args.steps, args.warmup, args.e2e_steps, cpu_s, opts, args.weighted, one_thread=True)
    per = {}
    if args.config == "all" and world == 1:
        for cname, cfmt in PER_CONFIG:
            # fewer steps for the side configurations keep the whole run inside a few minutes
            blk = measure_config(ctx, cname, cfmt, min(args.steps, 20), max(3, min(args.warmup, 5)), min(args.e2e_steps, 5),
                                 0.0 if args.no_cpu_baseline else min(3.0, args.cpu_seconds))
            per[f"{cname}:{cfmt}"] = blk
        # the (f) rows of SURVEY.md section 8, a few steps each, so that the driver-run record measures them too:
        # NEXT-1 weighted statistic + Psi (eq. 4), NEXT-2 random bank, NEXT-4 selection
        # (PAPER.md:79), NEXT-3 data preparation
        if not opts and not args.weighted and not args.no_next_rows:
            st, wu = min(args.steps, 10), 3
            per["weighted:cfg2"] = measure_config(ctx, "cfg2", "f32", st, wu, 0, 0.0, weighted=True)
            per["weighted:cfg4"] = measure_config(ctx, "cfg4", "f32", st, wu, 0, 0.0, weighted=True)
            per["bank:cfg2:1M"] = measure_bank("cfg2", "f32", 1_000_000, min(st, 5), wu, ctx["peaks"])
            per["select:393M"] = measure_select(393_216_000, min(st, 5), wu)
            per["prep:10800"] = measure_prep(10800, min(st, 5), wu)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    w_fmt = head["config"]["format"]
    line = {
        "metric": METRIC, "value": head["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": head["ms_per_step"], "higher_is_better": True, "scaling": "strong" if world > 1 else "weak",
        "vs_baseline": None,
        "dtype": {"f32": "f64 index + f32 accumulate", "u8": "f64 index + i32 accumulate",
                  "bits": "f64 index + i32 accumulate"}[w_fmt],
        "data": "synthetic",
        "config": head["config"],
        "parallelism": (f"dp{world}: contiguous ranges of the flattened (sky, tau, n) group index per rank "
                        "(tcw_search_groups), spectrogram replicated, no collective" if world > 1 else "1 GPU"),
        **{k: head[k] for k in ("templates_per_s", "inband_lookups_per_s", "inband_fraction", "create_ms", "launch",
                                "stage_ms", "roofline", "e2e", "gpu_launches", "clocks") if k in head},
    }
    for k in ("roofline_binding", "cpu_baseline"):
        if k in head:
            line[k] = head[k]
    if ctx["peaks"]:
        line["measured_peaks"] = ctx["peaks"]
    if per:
        line["per_config"] = per
        line["gpu_launches"] += sum(b.get("gpu_launches", 0) for b in per.values())
    if per and not args.verbose:
        line["per_config"] = {k: slim_block(b) for k, b in per.items()}
    out = compact(line, drop=() if args.verbose else COMPACT_DROP)
    out["roofline"]["peak_source"] = line["roofline"]["peak_source"]      # the contract wants the headline peak's origin stated
    print(json.dumps(out, separators=(",", ":")), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_shard(args, tcw, tcw_inputs, dev, r, n):
    import torch
    name, fmt = headline_name(args)
    w = tcw_inputs.make_workload(name, fmt=fmt)
    grid = tcw.Grid.of(w)
    lo, hi = tcw.shard_groups(grid.n_groups, r, n, weights=tcw.group_work(grid, w.timestamps, w.T_sft, w.f_min, w.n_bins))
    h = tcw.Handle.from_workload(w, device=dev)
    out_stat = torch.empty((max(hi - lo, 1), len(w.f0)), dtype=h.stat_dtype, device=dev)
    out_best = torch.empty((max(hi - lo, 1), 2), dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream()
    for _ in range(args.warmup):
        h.search_groups(grid, lo, hi, out_stat, out_best)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record(stream)
    for _ in range(args.steps):
        h.search_groups(grid, lo, hi, out_stat, out_best)
    e1.record(stream)
    torch.cuda.synchronize()
    h.check()
    ms = e0.elapsed_time(e1) / args.steps
    info = h.info()
    # the slice must equal the whole search's
    full_stat, full_best = h.search(grid)
    torch.cuda.synchronize()
    same = bool(torch.equal(full_stat.reshape(-1, len(w.f0))[lo:hi], out_stat[: hi - lo]) and
                torch.equal(full_best[lo:hi], out_best[: hi - lo]))
    h.close()
    print(json.dumps({"metric": METRIC + f" (rank {r} of {n}: its group range alone on one GPU)", "unit": UNIT,
                      "config": workload_config(w), "group_range": [lo, hi], "n_groups": grid.n_groups,
                      "ms_per_step": ms, "rank_lookups_per_s": (hi - lo) * len(w.f0) * w.n_sft / (ms * 1e-3),
                      "kernels_per_step": info["launches"], "ctas": info["ctas"],
                      "slice_equals_whole_search": same, "steps": args.steps, "warmup": args.warmup}), flush=True)
    return 0


def run_shard_table(args, tcw, tcw_inputs, dev):
    """--shard-table 2,4,8: ONE-GPU EMULATION of the multi-GPU split, not a scaling measurement.  For every N
    and both cuts (equal group count / equal in-band work) each rank's range is timed alone on this GPU;
    predicted efficiency = (single-GPU time / N) / (slowest rank's time).  What it leaves out: N uploads of
    the spectrogram over PCIe and anything the GPUs share (nothing on the data path)."""
    import torch
    name, fmt = headline_name(args)
    w = tcw_inputs.make_workload(name, fmt=fmt)
    grid = tcw.Grid.of(w)
    work = tcw.group_work(grid, w.timestamps, w.T_sft, w.f_min, w.n_bins)
    h = tcw.Handle.from_workload(w, device=dev)
    out_stat = torch.empty((grid.n_groups, len(w.f0)), dtype=h.stat_dtype, device=dev)
    out_best = torch.empty((grid.n_groups, 2), dtype=torch.int32, device=dev)
    stream = torch.cuda.current_stream()

    def timed(lo, hi):
        if hi == lo:
            return 0.0
        for _ in range(args.warmup):
            h.search_groups(grid, lo, hi, out_stat, out_best)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record(stream)
        for _ in range(args.steps):
            h.search_groups(grid, lo, hi, out_stat, out_best)
        e1.record(stream)
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    single = timed(0, grid.n_groups)
    table = {}
    for n in (int(x) for x in args.shard_table.split(",")):
        row = {}
        for cut, wts in (("equal_count", None), ("equal_work", work)):
            parts = [tcw.shard_groups(grid.n_groups, r, n, weights=wts) for r in range(n)]
            ms = [timed(lo, hi) for lo, hi in parts]
            row[cut] = {"ranges": parts, "ms": [round(x, 3) for x in ms], "max_ms": round(max(ms), 3),
                        "work_max_over_mean": round(float(max(work[lo:hi].sum() for lo, hi in parts) / (work.sum() / n)), 4),
                        "predicted_efficiency": round(single / n / max(ms), 4)}
        table[str(n)] = row
    h.check()
    h.close()
    print(json.dumps({"what": "one-GPU emulation of the group split, not a scaling measurement", "config": workload_config(w),
                      "single_gpu_ms": round(single, 3), "steps": args.steps, "warmup": args.warmup, "n": table}), flush=True)
    return 0


# ----------------------------------------------------------------------------- bank mode (NEXT-2)
def measure_bank(config, fmt, n_bank, steps, warmup, peaks=None):
    """tcw_search_bank on n_bank uniform random templates (PAPER.md:63 (ii)) over the config's data, at the
    config's first sky point.  The path is bound by FP64 arithmetic (one power per lookup), so
    its roofline is an ALU one: FP64_PER_LOOKUP warp-level FP64 instructions per 32 evaluated lookups (counted
    in the SASS of the fast path: DESIGN.md section 7) over the kernel time, against the FP64 issue rate that
    tcw_measure_peaks measures on this GPU."""
    import torch

    import paper_2507_07816_b200 as tcw
    import tcw_inputs

    w = tcw_inputs.make_workload(config, fmt=fmt)
    f_hi = w.f_min + w.n_bins / w.T_sft
    f0, tau, brk, sky = tcw_inputs.random_bank(n_bank, w.f_min, f_hi, w.seed, sky=w.sky[0])
    h = tcw.Handle.from_workload(w, device="cuda:0")
    out = torch.empty(n_bank, dtype=h.stat_dtype, device="cuda:0")
    for _ in range(warmup):
        _, inband, _ = h.search_bank(f0, tau, brk, sky, T0=w.T0, out_stat=out)
    h.set_option(tcw.TCW_OPT_TIMING, 1)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for _ in range(steps):
        _, inband, _ = h.search_bank(f0, tau, brk, sky, T0=w.T0, out_stat=out)
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    stage_ms, n_timed = h.timing()
    n_exact = h.counter(0)
    launches = h.info()["launches"]
    nominal = float(n_bank) * w.n_sft
    evaluated = float(inband.sum(dtype=torch.int64).item())
    kern_ms = stage_ms[1]
    h.close()
    peaks = peaks or tcw.measure_peaks()
    ach = FP64_PER_LOOKUP * evaluated / 32.0 / (kern_ms * 1e-3)
    return {"metric": METRIC + " (random template bank, tcw_search_bank)", "value": nominal / (kern_ms * 1e-3), "unit": UNIT,
            "n_gpus": 1, "steps": steps, "warmup": warmup, "ms_per_step": 1e3 * wall / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64 index + f32/i32 accumulate",
            "data": "synthetic", "config": workload_config(w, {"bank_templates": n_bank, "sky": "shared (PAPER.md:77)"}),
            "templates_per_s": n_bank / (kern_ms * 1e-3), "kernel_ms": kern_ms,
            "host_ms_per_step_incl_parameter_copy": 1e3 * wall / steps,
            "inband_lookups": evaluated, "inband_fraction": evaluated / nominal,
            "exact_chain_lookups": n_exact,
            "us_per_template": 1e3 * kern_ms / n_bank,
            "paper_us_per_template_a100": 15.0,
            "roofline": {"bound": "alu", "achieved": ach, "peak": peaks["fp64_dfma_winst_per_s"], "unit": "FP64 warp instructions/s",
                         "frac": ach / peaks["fp64_dfma_winst_per_s"], "traffic": None, "kernel": "sum_bank_kernel",
                         "fp64_inst_per_lookup": FP64_PER_LOOKUP, "peak_source": "tcw_measure_peaks (DFMA streams) in this process"},
            "gpu_launches": launches * steps}


def run_bank(args):
    """--bank N: one line for tcw_search_bank (not the headline metric)."""
    import torch

    import paper_2507_07816_b200 as tcw
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the tCW path has no CPU fallback")
    torch.cuda.set_device(0)
    tcw.load_library()
    print(json.dumps(measure_bank(args.config, args.format, args.bank, args.steps, args.warmup)), flush=True)
    return 0


# ----------------------------------------------------------------------------- selection mode (NEXT-4)
def measure_select(n, steps, warmup):
    """tcw_topk (K = 1000) and tcw_select_above over n float32 statistics ~ N(0, 1) (the shape of a Psi
    array; cfg5's out_stat has 393 M entries).  HBM-bound streaming passes: the algorithmic bytes are ONE
    read of the array (4 n bytes); top-K reads large arrays twice, threshold selection once plus the rows
    that hold a hit."""
    import torch

    import paper_2507_07816_b200 as tcw
    import tcw_inputs

    w = tcw_inputs.make_workload("cfg1")
    h = tcw.Handle.from_workload(w, device="cuda:0")
    g = torch.Generator(device="cuda").manual_seed(1)
    v = torch.randn(n, generator=g, device="cuda", dtype=torch.float32)
    peak, peak_src = load_peaks()
    res = {}
    for name, fn in (("topk_K1000", lambda: h.topk(v, 1000)), ("select_above_4.5", lambda: h.select_above(v, 4.5, 1 << 20))):
        for _ in range(max(3, warmup)):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / steps
        res[name] = {"ms": ms, "values_per_s": n / (ms * 1e-3),
                     "roofline": {"bound": "hbm", "achieved": 4.0 * n / (ms * 1e-3) / 1e9, "peak": peak, "unit": "GB/s",
                                  "frac": 4.0 * n / (ms * 1e-3) / 1e9 / peak, "traffic": None, "peak_source": peak_src}}
    h.close()
    del v
    torch.cuda.empty_cache()
    return {"metric": "statistics selected per second (tcw_topk / tcw_select_above)", "n": n,
            "steps": steps, "data": "synthetic", "results": res, "gpu_launches": (26 + 3) * steps}


def run_select(args):
    """--select N: one line for the selection calls."""
    import torch

    import paper_2507_07816_b200 as tcw
    torch.cuda.set_device(0)
    tcw.load_library()
    print(json.dumps(measure_select(args.select, args.steps, args.warmup)), flush=True)
    return 0


# ----------------------------------------------------------------------------- data preparation mode (NEXT-3)
def measure_prep(n_sft, steps, warmup):
    """tcw_prepare on n_sft 8-s segments of synthetic strain at 4096 Hz (device-resident), band 500-1000 Hz
    (4000 bins), running median over 101 bins: the step that produces cfg2's / cfg3's input.
    HBM model: one read of the strain (4 B/sample)."""
    import torch

    import paper_2507_07816_b200 as tcw

    fs, T = 4096.0, 8.0
    g = torch.Generator(device="cuda").manual_seed(2)
    x = torch.randn(n_sft * int(fs * T), generator=g, device="cuda", dtype=torch.float32)
    peak, peak_src = load_peaks()
    res = {}
    for fmt in ("f32", "bits"):
        for _ in range(max(2, min(warmup, 3))):
            tcw.prepare(x, fs, T, 500.0, 4000, 101, 1.6, fmt)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        for _ in range(steps):
            tcw.prepare(x, fs, T, 500.0, 4000, 101, 1.6, fmt)      # synchronises its stream
        ms = 1e3 * (time.perf_counter() - t0) / steps
        gbs = 4.0 * x.numel() / (ms * 1e-3) / 1e9
        res[fmt] = {"ms": ms, "sfts_per_s": n_sft / (ms * 1e-3), "samples_per_s": x.numel() / (ms * 1e-3),
                    "roofline": {"bound": "hbm", "achieved": gbs, "peak": peak, "unit": "GB/s", "frac": gbs / peak,
                                 "traffic": None, "peak_source": peak_src}}
    del x
    torch.cuda.empty_cache()
    return {"metric": "SFTs prepared per second (tcw_prepare: window, cuFFT R2C, running median, normalise, threshold)",
            "n_sft": n_sft, "fs": fs, "T_sft": T, "band_bins": 4000, "median_bins": 101, "steps": steps,
            "data": "synthetic", "timing": "host wall clock around the synchronous call (includes plan creation and scratch allocation)",
            "results": res}


def run_prep(args):
    """--prep N_SFT: one line for tcw_prepare."""
    import torch

    import paper_2507_07816_b200 as tcw
    torch.cuda.set_device(0)
    tcw.load_library()
    print(json.dumps(measure_prep(args.prep, args.steps, args.warmup)), flush=True)
    return 0


def main():
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--config", default="all", choices=["all", "cfg1", "cfg2", "cfg3", "cfg4", "cfg5"],
                    help="all (default): cfg4 as the headline plus per_config blocks for cfg2, cfg3 (u8, bits) and cfg5")
    ap.add_argument("--format", default=None, choices=["f32", "u8", "bits"])
    ap.add_argument("--kernel", default=None, choices=["auto", "gather", "staged", "skyblock"])
    ap.add_argument("--sky-block", type=int, default=0, choices=[0, 64, 128, 256])
    ap.add_argument("--f0-per-lane", type=int, default=0)
    ap.add_argument("--chunk-rows", type=int, default=0, help="staged kernel: SFT rows per chunk (0 auto, -1 never)")
    ap.add_argument("--stages", type=int, default=0, help="staged kernel: ring depth limit (0 auto)")
    ap.add_argument("--exact-index", action="store_true", help="staged kernel: defining chain for every bin (no fast index)")
    ap.add_argument("--general-f0", action="store_true", help="staged kernel: do not use the equally-spaced-f0 instantiation")
    ap.add_argument("--shard", default=None, metavar="R/N",
                    help="time rank R's group range of an N-GPU strong-scaling run alone on one GPU (and check it against the whole search)")
    ap.add_argument("--shard-table", default=None, metavar="N1,N2,..",
                    help="one-GPU emulation of the split for each N: every rank's range timed alone, equal-count and equal-work cuts")
    ap.add_argument("--no-next-rows", action="store_true", help="skip the weighted / bank / select / prep per_config entries")
    ap.add_argument("--verbose", action="store_true", help="keep notes and provenance strings in the JSON line")
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-seconds", type=float, default=10.0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--bank", type=int, default=0, help="time tcw_search_bank on this many random templates (NEXT-2)")
    ap.add_argument("--select", type=int, default=0, help="time tcw_topk / tcw_select_above over this many float32 values (NEXT-4)")
    ap.add_argument("--prep", type=int, default=0, help="time tcw_prepare on this many 8-s SFTs of synthetic strain (NEXT-3)")
    ap.add_argument("--weighted", action="store_true",
                    help="time tcw_search_weighted (weighted statistic + critical ratio, NEXT-1) instead of tcw_search")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "ours":
        args.warmup = 3                                  # timing rule: at least 3 warm-up steps
    if (args.bank or args.select or args.prep) and args.config == "all":
        args.config = "cfg2"
    if args.prep and args.impl == "ours":
        return run_prep(args)
    if args.select and args.impl == "ours":
        return run_select(args)
    if args.bank and args.impl == "ours":
        return run_bank(args)
    return run_reference(args) if args.impl == "reference" else run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
