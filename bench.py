#!/usr/bin/env python
"""bench.py -- dedispersion throughput (DM-trial samples/s) and fraction of the binding roofline on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

One "step" is one pass of the whole hot path (stage -> unpack -> shifted accumulate -> convert/store,
DESIGN.md section 2) over one synthetic batch: one dd_execute of BASELINE.json configs[1]
(1024 channels, 2-bit, 1200 DM trials, 2^19 output samples) with the input resident in HBM.
Prints ONE JSON line (rank 0).  N > 1 (torchrun): every rank dedisperses its own beam of the same
shape, no data-path collective (weak scaling); value = total units / slowest rank's time.

`--impl reference` times the CPU oracle (oracle/, as it stands) on the host cores on a bounded
sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "dedispersion throughput (DM-trial samples/s)"
UNIT = "DM-trial samples/s"


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons of one GPU every 100 ms while the timed region runs (NVML)."""

    REASONS = {
        0x8: "hw_slowdown", 0x40: "hw_thermal_slowdown", 0x20: "sw_thermal_slowdown", 0x4: "sw_power_cap",
        0x80: "hw_power_brake_slowdown", 0x2: "applications_clocks_setting", 0x100: "display_clock_setting",
    }

    def __init__(self, index: int):
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:
            self.nv = None

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, name in self.REASONS.items():
                    if mask & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop.wait(0.02)   # the default timed region is ~0.18 s: ~8 samples

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *exc):
        self._stop.set()
        if self._thr is not None:
            self._thr.join(timeout=2)

    def summary(self) -> dict:
        return {"sm_mhz": (statistics.median(self.samples) if self.samples else None),
                "sm_max_mhz": self.max_mhz, "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ helpers
def algorithmic_counts(cfg, max_delay: int, nbeams: int) -> dict:
    """Algorithmic work of one step: channel-adds, input bytes once + output bytes once."""
    esize = {"f32": 4, "u32": 4, "u16": 2}[cfg.out]
    units = nbeams * cfg.ndm * cfg.nsamps
    in_bytes = nbeams * cfg.nchans * ((cfg.nsamps + max_delay) * cfg.nbits // 8)
    return {"units": units, "adds": units * cfg.nchans, "bytes": in_bytes + units * esize,
            "in_bytes": in_bytes, "out_bytes": units * esize}


def info_after(plan) -> int:
    """Kernels the last dd_execute launched (the library's own count)."""
    return int(plan.launch_info()["last_launches"])


KERNEL_NAMES = {1: "dd_direct_v1<{nbits}>", 2: "dd_direct_v2", 3: "dd_direct_bp<{nbits}>",
                4: "dd_direct_bp<pair rows of {nbits}-bit input>", 5: "dd_direct_gs<{nbits}>",
                6: "dd_make_group_rows_staged<{nbits}> + dd_direct_gr<{nbits}>"}


def measured_peaks() -> dict:
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        try:
            return dict(json.load(open(path)), source="measured (MEASURED_PEAKS.json)")
        except Exception:
            pass
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}


def committed_capture(workload: str, variant: int) -> dict:
    """Counters of the committed ncu capture of this (workload, kernel variant): profiles/dram_traffic.csv, one line
    each -- dram bytes per dd_execute, ALU-pipe utilisation of the dominant kernel (%), the summary file."""
    path = os.path.join(ROOT, "profiles", "dram_traffic.csv")
    if os.path.exists(path):
        for line in open(path):
            f = [x.strip() for x in line.split(",")]
            if len(f) >= 5 and not f[0].startswith("#") and f[0] == workload and f[1] == str(variant):
                return {"traffic": float(f[2]), "alu_pipe_pct": float(f[3]) if f[3] else None, "capture": f[4]}
    return {"traffic": None, "alu_pipe_pct": None, "capture": None}


def cpu_sample(cfg, nsamps: int, dm_step: int):
    """The bounded oracle sample: first `nsamps` output samples, every dm_step-th DM trial, all channels."""
    import dd_workloads as W
    import oracle
    sub = W.CONFIGS[cfg.index].reduced(nsamps=nsamps)         # same band, same DM list
    dms = sub.dm_list()[::dm_step]
    tab = oracle.delay_table(sub.nchans, sub.dt, sub.f_top, sub.df, dms)
    packed, stride = W.gen_packed(sub, int(tab.max()))
    desc = (f"{cfg.name}: all {cfg.nchans} channels, first {nsamps} output samples, every {dm_step}th DM trial "
            f"({len(dms)} of {cfg.ndm}), 1 beam")
    return packed[0].numpy(), tab, nsamps, len(dms), desc


def time_oracle(packed, tab, nbits, nsamps, reps: int = 1):
    import oracle
    best = None
    for _ in range(reps):
        t0 = time.perf_counter()
        oracle.dedisperse(packed, nbits, nsamps, tab, nthreads=0)
        dt = time.perf_counter() - t0
        best = dt if best is None else min(best, dt)
    return best


def measure_config(dd, W, torch, cfg, stream, device_index, alu_peak, steps=5, warmup=3) -> dict:
    """One full-size config timed like the headline line (no end-to-end, no oracle): for `other_configs`."""
    plan = dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits).set_dm_list(cfg.dm_list())
    max_delay = plan.max_delay
    tab = plan.delay_table() if cfg.npulses else None
    pulses = W.make_pulses(cfg, lambda idx: tab[idx]) if cfg.npulses else None
    packed, stride = W.gen_packed(cfg, max_delay, pulses, device="cuda", beams=list(range(cfg.nbeams)), chan_chunk=16)
    tdtype = {"f32": torch.float32, "u32": torch.int32, "u16": torch.int16}[cfg.out]
    out = torch.empty((cfg.nbeams, cfg.ndm, cfg.nsamps), dtype=tdtype, device="cuda")
    if cfg.nbeams > 1:
        plan.set_batch(cfg.nbeams, packed.stride(0), out.stride(0) * out.element_size())
    counts = algorithmic_counts(cfg, max_delay, cfg.nbeams)
    for _ in range(warmup):
        plan.execute(cfg.nsamps, packed, stride, out, cfg.out_nbits, stream)
    torch.cuda.synchronize()
    plan.profile_enable(steps)
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(steps + 1)]
    with ClockSampler(device_index) as clk:
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            for k in range(steps):
                plan.execute(cfg.nsamps, packed, stride, out, cfg.out_nbits, stream)
                ev[k + 1].record(stream)
        torch.cuda.synchronize()
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(steps)]
    prepass_ms, main_ms = plan.profile_read()
    plan.profile_enable(0)
    info = plan.launch_info()
    ms = float(np.mean(per_step))
    cap = committed_capture(cfg.name, info["variant"])
    res = {
        "workload": cfg.name, "nchans": cfg.nchans, "nbits": cfg.nbits, "ndm": cfg.ndm, "nsamps": cfg.nsamps,
        "nbeams": cfg.nbeams, "out": cfg.out, "steps": steps, "variant": info["variant"],
        "kernel": KERNEL_NAMES[info["variant"]].format(nbits=cfg.nbits), "kernels_per_step": info["last_launches"],
        "ms_per_step": ms, "step_ms_min_max": [float(min(per_step)), float(max(per_step))],
        "kernel_ms": float(np.mean(main_ms)), "prepass_kernel_ms": float(np.mean(prepass_ms)),
        "value": counts["units"] / (ms * 1e-3), "unit": UNIT,
        "achieved_tadd_s": counts["adds"] / (ms * 1e-3) / 1e12, "frac": counts["adds"] / (ms * 1e-3) / alu_peak,   # of the whole step (every kernel of dd_execute)
        "algorithmic_bytes": counts["bytes"], "traffic": cap["traffic"], "alu_pipe_pct": cap["alu_pipe_pct"],
        "ncu_capture": cap["capture"], "workspace_bytes": plan.workspace_bytes, "clocks": clk.summary(),
    }
    plan.close()
    del packed, out
    torch.cuda.empty_cache()
    return res


# ------------------------------------------------------------------------------------------ reference arm
def measure_trees(dd, torch, cfg, packed_dev, stride, stream, steps=5, warmup=3):
    """`other_methods` of the headline line: the tree algorithm over the whole band and the piecewise linear tree (sub-bands
    of 32 channels, the leading trials of the DM list below the diagonal DM) on the SAME device-resident input as the
    headline measurement, when its rows are long enough; ms per call by CUDA events.  `bench.py --tree` is the full
    side measurement (roofline, oracle timing)."""
    out = []
    for sb in (cfg.nchans, 32):
        if cfg.nchans & (cfg.nchans - 1) or cfg.nchans * ((1 << cfg.nbits) - 1) > 65535:
            break
        tree = dd.Tree(cfg.nchans, sb, cfg.nbits)
        ndm = 0
        if sb < cfg.nchans:
            dms = cfg.dm_list()
            lo, hi = 1, len(dms)
            while lo < hi:
                mid = (lo + hi + 1) // 2
                try:
                    tree.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms[:mid])
                    lo = mid
                except dd.DDError:
                    hi = mid - 1
            tree.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms[:lo])
            ndm = lo
        nrows = ndm if ndm else cfg.nchans
        nsamps = cfg.nsamps
        if stride * 8 < tree.required_samples(nsamps) * cfg.nbits:      # (the rows were sized for the direct transform)
            nsamps = (stride * 8 // cfg.nbits - (tree.required_samples(nsamps) - nsamps)) // 64 * 64
        o = torch.empty((nrows, nsamps), dtype=torch.float32, device="cuda")
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
        with torch.cuda.stream(stream):
            for _ in range(warmup):
                tree.execute(nsamps, packed_dev, stride, o, 32, stream)
            ev[0].record(stream)
            for _ in range(steps):
                tree.execute(nsamps, packed_dev, stride, o, 32, stream)
            ev[1].record(stream)
        torch.cuda.synchronize()
        ms = ev[0].elapsed_time(ev[1]) / steps
        out.append({"method": "tree" if not ndm else "piecewise linear tree", "sb_nchans": sb, "trials": nrows, "nsamps": nsamps,
                    "ms_per_step": ms, "value": nrows * nsamps / (ms * 1e-3), "unit": UNIT, "passes": tree.info()["steps"],
                    "gpu_launches": tree.info()["last_launches"] * steps})
        tree.close()
        del o
    return out


def run_reference(args) -> None:
    import dd_workloads as W
    import oracle
    from paper_1201_5380_b200 import multi
    rank, _, world = multi.env_rank()
    if rank != 0:
        return
    cfg = W.CONFIGS[args.config]
    packed, tab, nsamps, ndm, desc = cpu_sample(cfg, args.cpu_nsamps, args.cpu_dm_step)   # the sample cpu_baseline times
    cores = oracle.threads(0)
    for _ in range(args.warmup):
        oracle.dedisperse(packed, cfg.nbits, nsamps, tab)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle.dedisperse(packed, cfg.nbits, nsamps, tab)
    el = time.perf_counter() - t0
    ms = el / args.steps * 1e3
    value = ndm * nsamps / (ms * 1e-3)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": cfg.name, "sample": desc},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": desc + " per step"},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


# ------------------------------------------------------------------------------------------ time-scrunching (side measurement)
def run_scrunch(args) -> None:
    """`--scrunch MAXF`: the transform with time-scrunching (dd_scrunch_*) on the config's DM list,
    timed like the main arm (CUDA events on the launching stream).  A side measurement, not the headline line."""
    import torch

    import dd_workloads as W
    import paper_1201_5380_b200 as dd

    torch.cuda.set_device(0)
    cfg = W.CONFIGS[args.config]
    stream = torch.cuda.Stream()
    sset = dd.ScrunchSet(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, cfg.dm_list(), args.scrunch)
    lv = sset.levels
    need = sset.required_bytes(cfg.nsamps)
    packed, stride = W.gen_packed(cfg, need * 8 // cfg.nbits - cfg.nsamps, None, device="cuda", beams=[0], chan_chunk=16)
    outs = [torch.empty((l["ndm"], cfg.nsamps // l["factor"]), dtype=torch.float32, device="cuda") for l in lv]
    for _ in range(max(args.warmup, 3)):
        sset.execute(cfg.nsamps, packed[0], stride, outs, 32, stream)
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    with ClockSampler(0) as clk:
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            for _ in range(args.steps):
                sset.execute(cfg.nsamps, packed[0], stride, outs, 32, stream)
            ev[1].record(stream)
        torch.cuda.synchronize()
    ms = ev[0].elapsed_time(ev[1]) / args.steps
    # the same call captured once into a CUDA graph and replayed (one graph launch instead of 2 per level + the cascade)
    graph = torch.cuda.CUDAGraph()
    with torch.cuda.graph(graph, stream=stream):
        sset.execute(cfg.nsamps, packed[0], stride, outs, 32, torch.cuda.current_stream())
    graph.replay()
    torch.cuda.synchronize()
    gev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    gev[0].record()
    for _ in range(args.steps):
        graph.replay()
    gev[1].record()
    torch.cuda.synchronize()
    ms_graph = gev[0].elapsed_time(gev[1]) / args.steps
    units = sum(l["ndm"] * (cfg.nsamps // l["factor"]) for l in lv)
    print(json.dumps({
        "metric": METRIC + " -- with time-scrunching (side measurement)", "value": units / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "ms_per_step_cuda_graph": ms_graph,
        "higher_is_better": True, "dtype": "u32", "data": "synthetic",
        "config": {"workload": cfg.name, "method": "direct with time-scrunching (lower time resolution at high DM)",
                   "max_factor": args.scrunch, "dm_diag": lv[0]["dm_diag_micro"] / 1e6, "levels": lv,
                   "outputs_per_step": units, "full_resolution_outputs": cfg.ndm * cfg.nsamps},
        "full_resolution_equivalent_per_s": cfg.ndm * cfg.nsamps / (ms * 1e-3), "clocks": clk.summary()}))
    sset.close()


# ------------------------------------------------------------------------------------------ tree dedispersion (side measurement)
def run_tree(args) -> None:
    """`--tree SB`: the tree algorithm (dd_tree_*) on the config's band and length.  SB = channels per
    tree: the config's channel count gives the whole-band tree (nchans linear trials); a smaller power of two gives the
    piecewise linear tree for the trials of the config's DM list below its diagonal DM.  Timed like the
    main arm (CUDA events on the launching stream); a side measurement, not the headline line.  The path is bound by memory:
    the roofline counts the packed input read once and the output rows written once."""
    import numpy as np
    import torch

    import dd_workloads as W
    import oracle
    import paper_1201_5380_b200 as dd

    torch.cuda.set_device(0)
    cfg = W.CONFIGS[args.config]
    sb = args.tree
    stream = torch.cuda.Stream()
    padded = sb < 0   # --tree -1: the frequency-padded tree over the stretched band
    tree = dd.Tree.padded(cfg.nchans, cfg.f_top, cfg.df, cfg.nbits) if padded else dd.Tree(cfg.nchans, sb, cfg.nbits)
    dms = None
    if padded:
        sb = tree.nchans
    elif sb < cfg.nchans:   # the leading trials of the DM list whose sub-band trails stay inside their trees (eq. 21)
        all_dms = cfg.dm_list()
        lo, hi = 1, len(all_dms)
        while lo < hi:
            mid = (lo + hi + 1) // 2
            try:
                tree.set_dm_list(cfg.dt, cfg.f_top, cfg.df, all_dms[:mid])
                lo = mid
            except dd.DDError:
                hi = mid - 1
        dms = all_dms[:lo]
        tree.set_dm_list(cfg.dt, cfg.f_top, cfg.df, dms)
    nrows = len(dms) if dms is not None else tree.nchans
    need = tree.required_samples(cfg.nsamps)
    packed, stride = W.gen_packed(cfg, need - cfg.nsamps, None, device="cuda", beams=[0], chan_chunk=16)
    out = torch.empty((nrows, cfg.nsamps), dtype=torch.float32, device="cuda")
    for _ in range(max(args.warmup, 3)):
        tree.execute(cfg.nsamps, packed[0], stride, out, 32, stream)
    torch.cuda.synchronize()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(2)]
    with ClockSampler(0) as clk:
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            for _ in range(args.steps):
                tree.execute(cfg.nsamps, packed[0], stride, out, 32, stream)
            ev[1].record(stream)
        torch.cuda.synchronize()
    ms = ev[0].elapsed_time(ev[1]) / args.steps
    info = tree.info()
    peaks = measured_peaks()
    alg_bytes = cfg.nchans * need * cfg.nbits / 8 + nrows * cfg.nsamps * 4
    cap = committed_capture(cfg.name, f"tree{args.tree}")   # dram bytes of one execute from the committed ncu capture, if any
    achieved = alg_bytes / (ms * 1e-3) / 1e9
    line = {
        "metric": METRIC + " -- tree algorithm (side measurement)", "value": nrows * cfg.nsamps / (ms * 1e-3), "unit": UNIT,
        "n_gpus": 1, "steps": args.steps, "warmup": max(args.warmup, 3), "ms_per_step": ms, "higher_is_better": True,
        "dtype": "u16" if sb * ((1 << cfg.nbits) - 1) <= 65535 else "u32", "data": "synthetic",
        "gpu_launches": info["last_launches"] * args.steps,
        "config": {"workload": cfg.name, "method": "frequency-padded tree" if padded else ("tree" if dms is None else "piecewise linear tree"), "sb_nchans": sb,
                   "trials": nrows, "dm_max": None if dms is None else float(dms[-1]), "passes": info["steps"],
                   "tile_columns": info["tile"], "device_bytes": info["device_bytes"], "l2": "inputs and outputs larger than L2"},
        "roofline": {"bound": "hbm", "achieved": achieved, "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": achieved / peaks["hbm_gbs"],
                     "traffic": cap["traffic"], "ncu_capture": cap["capture"], "peak_source": peaks["source"],
                     "algorithmic_bytes": alg_bytes, "note": "packed input read once + float32 rows written once; the 16-bit rows "
                     "between the passes (written and read once each) are not counted"},
        "clocks": clk.summary()}
    if not args.no_cpu:   # the oracle on a bounded sample: the same band, the first cpu_nsamps outputs
        sub = cfg.reduced(nsamps=args.cpu_nsamps, nbeams=1)
        hp, _ = W.gen_packed(sub, need - cfg.nsamps, None)
        t0 = time.perf_counter()
        if padded:
            oracle.padded_tree(hp[0].numpy(), cfg.nbits, args.cpu_nsamps, cfg.f_top, cfg.df)
        elif dms is None:
            oracle.tree(hp[0].numpy(), cfg.nbits, args.cpu_nsamps)
        else:
            oracle.piecewise_tree(hp[0].numpy(), cfg.nbits, args.cpu_nsamps, cfg.nchans, cfg.dt, cfg.f_top, cfg.df, dms, sb)
        dt = time.perf_counter() - t0
        line["cpu_baseline"] = {"value": nrows * args.cpu_nsamps / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{cfg.name}: all channels, first {args.cpu_nsamps} output samples, {nrows} trials"}
    print(json.dumps(line))
    tree.close()


# ------------------------------------------------------------------------------------------ our arm
def run_ours(args) -> None:
    import torch

    import dd_workloads as W
    import paper_1201_5380_b200 as dd
    from paper_1201_5380_b200 import multi

    rank, local_rank, world = multi.env_rank()
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    multi.init_process_group("nccl")
    cfg = W.CONFIGS[args.config]
    nbeams = cfg.nbeams
    stream = torch.cuda.Stream()

    plan = dd.Plan(cfg.nchans, cfg.dt, cfg.f_top, cfg.df, cfg.nbits, variant=args.variant).set_dm_list(cfg.dm_list())
    max_delay = plan.max_delay
    subband = None
    if args.subband:        # the approximate sub-band method instead of the direct transform
        sb, grp = (int(x) for x in args.subband.split(","))
        plan.set_subband(sb, grp)
        subband = {"sb_nchans": sb, "dm_group": grp, "extent": plan.subband_extent}
        max_delay = max(max_delay, plan.subband_extent)
    # synthetic input generated in HBM; rank r uses beam index r (+ the config's own beams) as generator stream
    beams = [rank * nbeams + b for b in range(nbeams)]
    tab = plan.delay_table() if cfg.npulses else None
    pulses = W.make_pulses(cfg, lambda idx: tab[idx]) if cfg.npulses else None
    packed, stride = W.gen_packed(cfg, max_delay, pulses, device="cuda", beams=beams, chan_chunk=16)
    tdtype = {"f32": torch.float32, "u32": torch.int32, "u16": torch.int16}[cfg.out]
    out = torch.empty((nbeams, cfg.ndm, cfg.nsamps), dtype=tdtype, device="cuda")
    if nbeams > 1:
        plan.set_batch(nbeams, packed.stride(0), out.stride(0) * out.element_size())
    counts = algorithmic_counts(cfg, max_delay, nbeams)
    if subband:             # eq. 27-29: N_SB * T_direct(N_t, N'nu, N_DMnom) + N_DMnom * T_direct(N_t, N_SB, N'DM)
        nsb, ngrp = cfg.nchans // subband["sb_nchans"], -(-cfg.ndm // subband["dm_group"])
        counts["adds"] = nbeams * cfg.nsamps * (ngrp * cfg.nchans + cfg.ndm * nsb)
    info = plan.launch_info()

    def step():
        plan.execute(cfg.nsamps, packed, stride, out, cfg.out_nbits, stream)

    torch.cuda.synchronize()
    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    plan.profile_enable(args.steps)      # 3 CUDA events per dd_execute on the launching stream (no sync)

    # ---- timed region: exactly K steps, CUDA events on the launching stream, barrier + sync on both sides
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps + 1)]
    multi.barrier()
    torch.cuda.synchronize()
    with ClockSampler(local_rank) as clk:
        wall0 = time.perf_counter()
        with torch.cuda.stream(stream):
            ev[0].record(stream)
            for k in range(args.steps):
                step()
                ev[k + 1].record(stream)
        torch.cuda.synchronize()
        wall = time.perf_counter() - wall0
    multi.barrier()
    total_ms = ev[0].elapsed_time(ev[-1])
    per_step = [ev[k].elapsed_time(ev[k + 1]) for k in range(args.steps)]
    prepass_ms, main_ms = plan.profile_read()          # per-kernel times of the same K timed steps
    plan.profile_enable(0)
    assert len(main_ms) == args.steps
    kernels_per_step = info_after(plan)
    ms_step_rank = total_ms / args.steps
    value, ms_step = multi.job_throughput(counts["units"], ms_step_rank)
    kernel_ms = float(np.mean(main_ms))
    if subband:     # three kernels share the work: report the whole step, and step 2's transform kernel beside it
        subband["step2_kernel_ms"] = kernel_ms
        kernel_ms = float(np.mean(np.asarray(main_ms) + np.asarray(prepass_ms)))

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region (all ranks)
    e2e = None
    if not args.no_e2e:
        h_in = packed.cpu().pin_memory()
        h_out = torch.empty((nbeams, cfg.ndm, cfg.nsamps), dtype=tdtype).pin_memory()
        plan.execute_host(cfg.nsamps, h_in, stride, h_out, cfg.out_nbits)        # warm-up (allocates staging)
        reps, rep_ms = 5, []
        multi.barrier()
        t0 = time.perf_counter()
        for _ in range(reps):
            t1 = time.perf_counter()
            plan.execute_host(cfg.nsamps, h_in, stride, h_out, cfg.out_nbits)
            rep_ms.append((time.perf_counter() - t1) * 1e3)
        e2e_ms_rank = (time.perf_counter() - t0) / reps * 1e3      # the mean is what `value` is made of
        e2e_value, e2e_ms = multi.job_throughput(counts["units"], e2e_ms_rank)
        ok = bool(torch.equal(h_out.cuda(), out))
        e2e = {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_ms, "steps": reps,
               "ms_per_step_min_median_max": [min(rep_ms), sorted(rep_ms)[reps // 2], max(rep_ms)],
               "h2d_bytes_per_step": int(h_in.numel() * h_in.element_size()),
               "d2h_bytes_per_step": int(h_out.numel() * h_out.element_size()),
               "kernels_per_step": plan.launch_info()["last_launches"], "matches_device_path": ok,
               "api": "dd_execute_host, pinned host buffers, host<->device copies inside the timed region"}
        del h_in, h_out

    if rank != 0:
        multi.barrier()
        return

    # ---- roofline of the (only) kernel: ALU-bound; HBM shown beside it
    peak_ind = dd.dd_int_add_peak(0, stream)
    peak_3in = dd.dd_int_add_peak(1, stream)
    peak_mix = dd.dd_int_add_peak(2, stream)
    alu_peak = max(peak_ind, peak_3in, peak_mix)
    peaks = measured_peaks()
    achieved_adds = counts["adds"] / (kernel_ms * 1e-3)
    achieved_gbs = counts["bytes"] / (kernel_ms * 1e-3) / 1e9
    cap = committed_capture(cfg.name, info["variant"])
    roofline = {
        "bound": "alu", "achieved": achieved_adds / 1e12, "peak": alu_peak / 1e12, "unit": "Tadd/s",
        "frac": achieved_adds / alu_peak,
        "traffic": cap["traffic"], "alu_pipe_pct": cap["alu_pipe_pct"], "ncu_capture": cap["capture"],
        "kernel": ("sub-band: dd_to_bitplanes + dd_direct_bp<{nbits}> (step 1), dd_to_bitplanes + dd_direct_bp<8> (step 2)"
                   if subband else KERNEL_NAMES[info["variant"]]).format(nbits=cfg.nbits), "kernel_ms": kernel_ms,
        "kernel_ms_p5_p50_p95": [float(np.percentile(main_ms, q)) for q in (5, 50, 95)],
        "kernel_share_of_step": kernel_ms / float(np.mean(per_step)),
        "prepass_kernel_ms": float(np.mean(prepass_ms)),
        "step_ms_p5_p50_p95": [float(np.percentile(per_step, q)) for q in (5, 50, 95)],
        "algorithmic_adds_per_launch": counts["adds"], "algorithmic_bytes_per_launch": counts["bytes"],
        "frac_note": "algorithmic channel-adds / measured scalar integer-add peak; the bit-plane kernels retire 32 "
                     "channel-adds with ~6 ALU instructions, so frac may exceed 1 -- alu_pipe_pct (ncu, committed "
                     "capture) says how busy the limiting pipe is",
        "peak_source": "measured in this run by dd_int_add_peak (32-bit integer additions/s, all SMs): "
                       f"2-input adds {peak_ind / 1e12:.2f}, 3-input IADD3 {peak_3in / 1e12:.2f}, IADD3+IMAD on both "
                       f"pipes {peak_mix / 1e12:.2f} Tadd/s; peak = the largest",
        "hbm": {"achieved": achieved_gbs, "peak": peaks.get("hbm_gbs"), "unit": "GB/s",
                "frac": achieved_gbs / peaks.get("hbm_gbs", float("nan")), "peak_source": peaks["source"]},
    }

    # ---- the other full-size configs of BASELINE.json (cfg4, cfg5, cfg3), 5 timed steps each, same method: inputs
    # generated in HBM, CUDA events on the launching stream, clocks sampled during that config's timed region
    other_configs = None
    other_methods = None
    if args.config == 2 and not subband and not args.no_others and world == 1 and not args.variant:
        plan.close()
        del out
        torch.cuda.empty_cache()
        other_methods = measure_trees(dd, torch, cfg, packed[0], stride, stream, steps=5)   # (on the headline's input rows)
        del packed
        torch.cuda.empty_cache()
        other_configs = [measure_config(dd, W, torch, W.CONFIGS[i], stream, local_rank, alu_peak, steps=5) for i in (4, 5, 3)]

    # ---- the oracle timed beside it on this box's host cores (bounded sample; a baseline, not the target)
    cpu_baseline = None
    if not args.no_cpu and world == 1:
        import oracle
        cpacked, ctab, cns, cndm, desc = cpu_sample(cfg, args.cpu_nsamps, args.cpu_dm_step)
        el = time_oracle(cpacked, ctab, cfg.nbits, cns, reps=4)
        cpu_baseline = {"value": cndm * cns / el, "unit": UNIT, "cores": oracle.threads(0), "kind": "oracle",
                        "sample": desc, "seconds": el}

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": max(args.warmup, 3), "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": cfg.name, "nchans": cfg.nchans, "nbits": cfg.nbits, "ndm": cfg.ndm,
                   "nsamps": cfg.nsamps, "nbeams_per_gpu": nbeams, "out": cfg.out, "max_delay": max_delay,
                   "tile": f"{info['dm_block']} DMs x {info['time_block']} samples, {info['threads']} threads, "
                           f"{info['smem_bytes']} B smem",
                   "l2": f"no flush: each step streams {counts['bytes'] / 1e9:.2f} GB (input {counts['in_bytes'] / 1e6:.0f} MB "
                         f"+ output {counts['out_bytes'] / 1e9:.2f} GB) > 126 MB L2",
                   "parallelism": f"beam-per-gpu x{world}" if world > 1 else "single gpu",
                   **({"method": "sub-band (approximate)", **subband} if subband else {})},
        "clocks": clk.summary(), "e2e": e2e, "gpu_launches": args.steps * kernels_per_step,
        "roofline": roofline, "cpu_baseline": cpu_baseline, "other_configs": other_configs, "other_methods": other_methods,
        "wall_s_timed_region": wall,
    }
    print(json.dumps(line))
    if world > 1:
        multi.barrier()


def main() -> None:
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--subband", default="", help="SB,GRP: time the sub-band method (channels per sub-band, trials per "
                    "nominal DM) instead of the direct transform; implies --no-e2e")
    ap.add_argument("--scrunch", type=int, default=0, help="MAXF: time the transform with time-scrunching up to this "
                    "factor (a power of two) instead -- a side measurement")
    ap.add_argument("--tree", type=int, default=0, help="SB: time the tree algorithm on trees of SB channels (the config's channel "
                    "count: the whole band; smaller: the piecewise linear tree below the diagonal DM; -1: the frequency-padded "
                    "tree) (side measurement)")
    ap.add_argument("--variant", type=int, default=0, help="kernel variant (dd_set_kernel_variant); 0 = the library's choice")
    ap.add_argument("--no-e2e", action="store_true", help="skip the host-buffer end-to-end measurement")
    ap.add_argument("--no-cpu", action="store_true", help="skip the CPU oracle baseline")
    ap.add_argument("--no-others", action="store_true", help="skip the other full-size configs (other_configs)")
    ap.add_argument("--cpu-nsamps", type=int, default=1 << 16, help="output samples of the bounded oracle sample (both the "
                    "cpu_baseline of the main arm and every step of --impl reference time this sample)")
    ap.add_argument("--cpu-dm-step", type=int, default=1, help="the oracle sample takes every n-th DM trial")
    args = ap.parse_args()
    if args.subband:
        args.no_e2e = True
    if args.impl == "reference":
        run_reference(args)
    elif args.scrunch:
        run_scrunch(args)
    elif args.tree:
        run_tree(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
