#!/usr/bin/env python
"""bench.py — throughput of the fused analysis chain (hepk_analysis_chain) on synthetic top-pair-shaped events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--scaling weak|strong] [--impl reference]

One "step" = one pass of the whole hot path (selection, dR cleaning, [calibration variants], per-event
reductions, leading-pair mass, weighted histograms — SURVEY.md 8(a) rows a1..a7) over one batch of events.
Default workload: BASELINE.json configs[2] (10,000,000 events; the configuration north_star's ">= 60 % of
B200 peak HBM bandwidth" target is quoted on).  Prints ONE JSON line (rank 0).

  value          events/s, inputs resident in HBM, CUDA events over K steps, max over ranks
  e2e            the same through hepk_analysis_chain_host: PINNED HOST buffers in, host buffers out, every
                 host<->device copy inside the timed region
  roofline       the fused chain kernel alone: algorithmic bytes per launch / its average device time (CUDA events
                 recorded by the library directly around the kernel), against the measured HBM peak of
                 MEASURED_PEAKS.json; `generic_build` is the same launch through the build that is not specialised
                 for the common output shape
  cpu_baseline   the CPU oracle (oracle/, as it stands) on the same workload and box: one thread, and every core
  other_configs  (1 GPU) configs 1, 3, 4 and the 40-variant run: value, kernel ms, roofline with its bound,
                 cpu_baseline; config 4 also as BASELINE.json defines it: 10 batches of 5 M events streamed from
                 host memory (serial, overlapped, kernel only) against the pinned-copy rate measured in this run
  single_kernels (1 GPU) every hepk_* single kernel: ms, algorithmic GB/s, fraction of the measured peak

`--scaling strong` (N > 1) shards ONE workload over the ranks (sharding.event_shards, offset slices + content_base);
the default `weak` gives every rank its own batch.  `--impl reference` times the oracle instead (no GPU is touched).
"""
from __future__ import annotations

import argparse
import csv
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "fused analysis chain throughput (events/s; achieved HBM GB/s as fraction of B200 peak in `roofline`)"
UNIT = "events/s"
BENCH_OUTPUTS = ("njet", "ht", "maxpt", "argmax", "mjj")      # 20 B x V of per-event outputs
FALLBACK_HBM_GBS = 6650.0                                     # B200_PROFILING.md fallback ("of fallback")
NVML_REASONS = {
    0x1: "gpu_idle", 0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown",
    0x10: "sync_boost", 0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
    0x100: "display_clock_setting",
}


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--config", type=int, default=2, help="BASELINE.json config index (1..4)")
    ap.add_argument("--events", type=int, default=None, help="override the number of events (testing only)")
    ap.add_argument("--impl", default="hepk", choices=["hepk", "reference"])
    ap.add_argument("--scaling", default="weak", choices=["weak", "strong"],
                    help="N > 1: weak = one batch per rank, strong = ONE workload sharded over the ranks")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true", help="skip the other_configs and single_kernels records")
    ap.add_argument("--c4-batches", type=int, default=10, help="batches of the streamed config-4 run (BASELINE.json: 10)")
    ap.add_argument("--single-kernels", action="store_true",
                    help="time each single kernel (SURVEY.md 8(a) rows a1-a6 and the f rows) only; one JSON line")
    ap.add_argument("--sk-eager", action="store_true",
                    help="--single-kernels without the CUDA-graph replay (the launch-list pass of the profiler)")
    ap.add_argument("--variants", type=int, default=None,
                    help="configs 3/4: number of calibration variants (scales 1 +- k*0.0025); the paper's full-systematics scenario is 40")
    ap.add_argument("--tune", default="", help="chain tuning knobs, e.g. warps_per_sm=20 (testing only)")
    ap.add_argument("--ref-sample", type=int, default=1_000_000, help="events per step of the reference arm")
    return ap.parse_args()


def workload_name(cfg, wl):
    return (f"BASELINE.json configs[{cfg}]: {wl.n_events:,} events/GPU, jets Poisson({wl.meta['lam_jet']:g}) cap "
            f"{wl.meta['cap_jet']}{' +1% tail 30-40' if wl.meta['tail'] else ''}, "
            f"{'muons+electrons' if wl.electrons is not None else 'muons'}, "
            f"{1 if wl.calib is None else len(wl.calib['scales'])} variant(s), "
            f"{len(wl.hists)}x{wl.weights.shape[0]} histograms/variant")


def algorithmic_bytes(wl, n_outputs=len(BENCH_OUTPUTS), event_outputs=True):
    """every needed input column read once, required outputs written once (lepton mass is
    not needed; tables and edges are KB-sized)."""
    n = wl.n_events
    v = 1 if wl.calib is None else len(wl.calib["scales"])
    b = 8 * (n + 1) * (3 if wl.electrons is not None else 2)
    b += 16 * wl.jets.n_objects + 12 * wl.muons.n_objects
    if wl.electrons is not None:
        b += 12 * wl.electrons.n_objects
    b += 4 * wl.weights.size
    if event_outputs:
        b += 4 * n_outputs * v * n
    return b


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.005):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.reasons, self.max_mhz = [], 0, None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # NVML missing: report that instead of inventing numbers
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        while not self._stop_evt.is_set():
            try:
                self.samples.append(self.nv.nvmlDeviceGetClockInfo(self.h, self.nv.NVML_CLOCK_SM))
                self.reasons |= int(self.nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
            except Exception:
                try:
                    self.reasons |= int(self.nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                except Exception:
                    pass
            self._stop_evt.wait(self.period)

    def stop(self):
        self._stop_evt.set()
        if self.ok:
            self.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": ["nvml unavailable"]}
        s = sorted(self.samples)
        names = [n for bit, n in NVML_REASONS.items() if self.reasons & bit and n != "gpu_idle"]
        return {"sm_mhz": s[len(s) // 2], "sm_max_mhz": self.max_mhz, "reasons": names, "samples": len(s)}


def measured_peak():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md 6.65 TB/s)"


def traffic_row(config, variants=None):
    """DRAM bytes of one launch from the committed ncu captures: one row per config in profiles/traffic.csv, each
    naming its capture (profiles/traffic.md says how the rows were made)."""
    tp = os.path.join(ROOT, "profiles", "traffic.csv")
    key = f"{config}" if not variants else f"{config}v{variants}"
    try:
        for row in csv.DictReader(open(tp)):
            if row["config"] == key:
                return int(row["dram_bytes_per_launch"]), row["source"]
    except Exception:
        pass
    return None, None


def time_oracle(wl, e0, e1, threads=1):
    from oracle import hepo
    t0 = time.perf_counter()
    res = hepo.analysis_chain(wl, e0, e1, want_mask=False, threads=threads)
    return time.perf_counter() - t0, res


def cpu_baseline(wl, n_single, n_all):
    """The oracle as it stands: one thread on the first n_single events, every core on the first n_all events."""
    from oracle import hepo
    N = wl.n_events
    dt1, ref = time_oracle(wl, 0, n_single, threads=1)
    cores = hepo.max_threads()
    dta, _ = time_oracle(wl, 0, n_all, threads=0)
    out = {"value": n_single / dt1, "unit": UNIT, "cores": 1, "kind": "oracle",
           "sample": f"first {n_single:,} of {N:,} events, one pass, {dt1:.1f} s, single thread of {os.cpu_count()} host cores",
           "all_cores": {"value": n_all / dta, "unit": UNIT, "cores": cores, "kind": "oracle (OpenMP over events, private histograms)",
                         "sample": f"first {n_all:,} of {N:,} events, one pass, {dta:.1f} s, {cores} threads"}}
    return out, (ref if n_single == N else None)


# ------------------------------------------------------------------------------------------ reference arm
def run_reference(args):
    """This tier's reference arm: the CPU oracle, as it stands, single thread, on a bounded sample per step."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import hepgen
    n_s = args.ref_sample if args.events is None else min(args.events, args.ref_sample)
    wl = hepgen.generate(args.config, n_events=n_s)
    for _ in range(max(args.warmup, 1)):
        time_oracle(wl, 0, min(n_s, 50_000))
    tot = 0.0
    for _ in range(args.steps):
        dt, _ = time_oracle(wl, 0, n_s)
        tot += dt
    value = n_s * args.steps / tot
    sample = f"first {n_s:,} events of configs[{args.config}] per step, {args.steps} steps"
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, wl), "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))


# ------------------------------------------------------------------------------------------ our arm
def time_chain(plan, steps, warmup, hk, torch, step=None, barrier=None):
    """(ms per step, chain-kernel ms per step, chain-kernel launches per step, library kernels per step)."""
    step = step or plan.run
    barrier = barrier or torch.cuda.synchronize
    for _ in range(max(warmup, 3)):
        step()
    barrier()
    plan.zero_hists()
    barrier()
    hk.profile_begin()
    l0 = hk.kernel_launches()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        step()
    ev1.record()
    barrier()
    kern_ms, kern_n = hk.profile_end()
    launches = hk.kernel_launches() - l0
    return ev0.elapsed_time(ev1) / steps, kern_ms / steps, kern_n / steps, launches / steps


def chain_roofline(wl, kern_ms_per_step, kern_launches_per_step, hists_only, config, variants=None):
    peak, peak_src = measured_peak()
    alg = algorithmic_bytes(wl, event_outputs=not hists_only)
    achieved = alg / (kern_ms_per_step * 1e-3) / 1e9
    traffic, src = traffic_row(config, variants)
    return {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": traffic,
            "traffic_source": src, "kernel": "hepk::dev::chain_kernel", "kernel_ms_per_step": kern_ms_per_step,
            "kernel_launches_per_step": kern_launches_per_step, "algorithmic_bytes_per_step": alg,
            "bytes_per_event": alg / wl.n_events, "peak_source": peak_src, "frac_of_nominal_8TBs": achieved / 8000.0}


def run_hepk(args):
    import numpy as np
    import torch
    import torch.distributed as dist

    import hepgen
    from paper_1906_06242_b200 import binding as hk, sharding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback); use --impl reference for the oracle")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    hk.lib()
    strong = world > 1 and args.scaling == "strong"

    def with_variants(wl):
        if args.variants and wl.calib is not None:
            wl.calib["scales"] = (1.0 + 0.0025 * (np.arange(args.variants) - args.variants // 2)).astype(np.float32)
        return wl

    if strong:
        # ONE workload, every rank draws the same events and keeps its jet-balanced shard:
        # offset slices + content_base + column slices on the device, nothing rebased
        whole = with_variants(hepgen.generate(args.config, n_events=args.events, batch=0))
        e0, e1 = sharding.event_shards(whole.jets.offsets, world)[rank]
        inp = sharding.shard_inputs(hk.upload(whole), e0, e1, host_offsets=dict(
            jets=whole.jets.offsets, muons=whole.muons.offsets,
            electrons=None if whole.electrons is None else whole.electrons.offsets))
        wl, N_total = whole, whole.n_events
    else:
        # weak scaling: every rank draws its own batch of the same recipe (events are independent)
        wl = with_variants(hepgen.generate(args.config, n_events=args.events, batch=rank))
        inp = hk.upload(wl)
        N_total = wl.n_events * world
    N = wl.n_events
    V = 1 if wl.calib is None else len(wl.calib["scales"])
    hists_only = args.config == 4          # config 4 writes histograms only
    tune = {k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(",") if kv)}
    plan = hk.ChainPlan(inp, want_event_outputs=False if hists_only else BENCH_OUTPUTS, tune=tune or None)
    hist_t = [plan.out["hist_sumw"], plan.out["hist_counts"]]

    def step():
        if world > 1:                      # per-step histograms, merged over ranks: start from zero on every rank
            plan.zero_hists()
        plan.run()
        if world > 1:                      # the one exchange step of the path: histogram merge
            sharding.merge_histograms(hist_t)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    sampler = ClockSampler(local)
    sampler.start()
    ms_step, kern_ms, kern_n, launches = time_chain(plan, args.steps, args.warmup, hk, torch, step, barrier)
    sampler.stop()
    if world > 1:
        t = torch.tensor([ms_step], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        ms_step = float(t.item())
    value = N_total / (ms_step * 1e-3)

    # sanity of the timed work: every event of every step landed in every histogram
    counts = plan.out["hist_counts"].cpu().numpy().reshape(V, -1)
    expect = (N_total if world > 1 else N * args.steps) * len(wl.hists)
    assert (counts.sum(axis=1) == expect).all(), (counts.sum(axis=1), expect)

    if strong:      # the roofline is a per-GPU figure: the shard's bytes over the shard's kernel time
        import copy
        shard_wl = copy.copy(wl)
        shard_wl.n_events = inp.n_events
        nobj = lambda c: None if c is None else int(c.pt.numel())
        class _C:      # sizes only
            def __init__(self, n): self.n_objects = n
        shard_wl.jets, shard_wl.muons = _C(nobj(inp.jets)), _C(nobj(inp.muons))
        shard_wl.electrons = None if inp.electrons is None else _C(nobj(inp.electrons))
        shard_wl.weights = wl.weights[:, :inp.n_events]
        roof = chain_roofline(shard_wl, kern_ms, kern_n, hists_only, args.config, args.variants)
    else:
        roof = chain_roofline(wl, kern_ms, kern_n, hists_only, args.config, args.variants)

    # the same bytes over the WHOLE step's device time (weight-range pre-pass, header memset, chain kernel(s), histogram
    # finalize), the pre-pass's second read of the weights added to the bytes: what a user of the call gets
    prepass = 4.0 * inp.n_events * (wl.weights.shape[0] if wl.weights is not None else 0) * kern_n
    step_bytes = roof["algorithmic_bytes_per_step"] + prepass
    roof["whole_step"] = {"ms": ms_step, "bytes": step_bytes, "achieved": step_bytes / (ms_step * 1e-3) / 1e9,
                          "frac": step_bytes / (ms_step * 1e-3) / 1e9 / roof["peak"],
                          "note": "chain kernel + weight-range pre-pass + memset + finalize; bytes include the pre-pass's read of the weights"}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms_step, "higher_is_better": True, "scaling": "strong" if strong else "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, wl), "events_per_gpu": inp.n_events, "events_total": N_total,
                   "variants": V,
                   "parallelism": ("ONE workload sharded by jet-balanced event ranges" if strong else "one batch per GPU")
                                  + f" over {world} GPU(s), histogram all-reduce" if world > 1 else "1 GPU",
                   "l2": f"inputs {roof['algorithmic_bytes_per_step'] / 1e9:.2f} GB per step >> 126 MB L2, no flush needed",
                   "outputs": list(BENCH_OUTPUTS) if not hists_only else "histograms only"},
        "roofline": roof, "clocks": sampler.summary(),
        # kernels of this library enqueued per step, counted by the library itself (hepk_kernel_launches), x steps
        "gpu_launches": int(round(launches * args.steps)),
        "gpu_launches_per_step": launches,
    }

    if world == 1 and not hists_only and not args.tune:
        # the same launch through the build that is NOT specialised for this output shape
        gplan = hk.ChainPlan(inp, want_event_outputs=BENCH_OUTPUTS, tune=dict(generic_build=1))
        g_ms, g_kern, _, _ = time_chain(gplan, max(10, args.steps // 4), 3, hk, torch)
        groof = chain_roofline(wl, g_kern, 1, False, args.config, args.variants)
        out["roofline"]["generic_build"] = {"kernel_ms_per_step": g_kern, "frac": groof["frac"], "achieved": groof["achieved"],
                                            "ms_per_step": g_ms, "value": N / (g_ms * 1e-3)}
        del gplan

    # ---- end to end through the C ABI with HOST buffers (rank-local; max over ranks)
    if not args.no_e2e and not strong:
        batch = min(N, 2_500_000)
        hplan = hk.HostChainPlan(wl, batch_events=batch, want_event_outputs=False if hists_only else BENCH_OUTPUTS)
        e2e_steps = max(1, min(args.steps, 5))
        hplan.run(overlap=True)
        hplan.zero_hists()
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            hplan.run(overlap=True)       # synchronises before returning: results are in host memory
        barrier()
        dt = time.perf_counter() - t0
        t0 = time.perf_counter()
        hplan.run(overlap=False)
        dt_serial = time.perf_counter() - t0
        if world > 1:
            t = torch.tensor([dt], dtype=torch.float64, device="cuda")
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            dt = float(t.item())
        out["e2e"] = {"value": N * world * e2e_steps / dt, "unit": UNIT, "h2d_bytes_per_step": hplan.h2d_bytes,
                      "d2h_bytes_per_step": hplan.d2h_bytes, "steps": e2e_steps, "batch_events": batch,
                      "overlap": True, "value_no_overlap": N / dt_serial,
                      "h2d_GBps_effective": hplan.h2d_bytes * e2e_steps / dt / 1e9,
                      "timer": "host wall clock around hepk_analysis_chain_host (the call synchronises)"}
        del hplan

    # ---- the oracle on this box's host cores (rank 0, N=1 only)
    if world == 1 and not args.no_cpu_baseline:
        n_s = N if args.config <= 2 else min(N, 1_000_000 if args.config == 3 else 200_000)
        base, ref = cpu_baseline(wl, n_s, N)
        out["cpu_baseline"] = base
        if ref is not None:      # free parity evidence: one fresh GPU step against the oracle's histograms
            plan.zero_hists()
            plan.run()
            torch.cuda.synchronize()
            out["cpu_baseline"]["hist_counts_equal_gpu"] = bool((plan.out["hist_counts"].cpu().numpy() == ref["hist_counts"]).all())

    if world == 1 and not args.no_other_configs and args.config == 2 and args.events is None and not args.tune:
        del plan, inp
        torch.cuda.empty_cache()
        out["other_configs"] = other_configs(args, hk, torch, np, hepgen)
        out["single_kernels"] = single_kernels(args, hk, torch, hepgen, steps=20)["kernels"]

    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def other_configs(args, hk, torch, np, hepgen):
    """Configs 1, 3, 4 and the 40-variant run (1 GPU): device-resident throughput, kernel time, roofline, oracle."""
    res = {}
    steps = max(5, min(args.steps, 20))
    atom_rate = hk.probe_shared_atomics(16, 32768)           # measured on this device in this run
    for key, cfg, variants in (("config1", 1, None), ("config3", 3, None), ("config3_40_variants", 3, 40), ("config4", 4, None)):
        wl = hepgen.generate(cfg)
        if variants:
            wl.calib["scales"] = (1.0 + 0.0025 * (np.arange(variants) - variants // 2)).astype(np.float32)
        V = 1 if wl.calib is None else len(wl.calib["scales"])
        hists_only = cfg == 4
        inp = hk.upload(wl)
        plan = hk.ChainPlan(inp, want_event_outputs=False if hists_only else BENCH_OUTPUTS)
        ms_step, kern_ms, kern_n, launches = time_chain(plan, steps, 3, hk, torch)
        counts = plan.out["hist_counts"].cpu().numpy().reshape(V, -1)
        assert (counts.sum(axis=1) == wl.n_events * steps * len(wl.hists)).all()
        roof = chain_roofline(wl, kern_ms, kern_n, hists_only, cfg, variants)
        rec = {"workload": workload_name(cfg, wl), "value": wl.n_events / (ms_step * 1e-3), "unit": UNIT, "ms_per_step": ms_step,
               "steps": steps, "gpu_launches_per_step": launches, "roofline": roof}
        if cfg == 1:
            rec["note"] = "config 1's inputs (132 MB) fit the 126 MB L2 almost entirely: not an HBM figure"
        if cfg == 4:
            # histogram-bound: 6 observables x (10 weights + 1 count) native shared-memory atomics per event and variant
            lane_atomics = wl.n_events * V * len(wl.hists) * (wl.weights.shape[0] + 1)
            rate = lane_atomics / (kern_ms * 1e-3)
            rec["roofline_atomics"] = {"bound": "alu", "what": "red.shared.add.s32 lane-atomics of the privatised histograms",
                                       "achieved": rate / 1e9, "peak": atom_rate / 1e9, "unit": "G atomics/s",
                                       "frac": rate / atom_rate, "lane_atomics_per_event": lane_atomics / wl.n_events,
                                       "peak_source": "hepk_probe_shared_atomics: 16 warps/SM, random addresses in 32768 words, this run"}
        if not args.no_cpu_baseline:
            n1 = {1: wl.n_events, 3: 500_000, 4: 100_000}[cfg] if not variants else 100_000
            rec["cpu_baseline"], _ = cpu_baseline(wl, n1, wl.n_events if not variants else 1_000_000)
        del plan, inp
        torch.cuda.empty_cache()
        if cfg == 4 and not args.no_e2e:
            rec["streamed"] = streamed_config4(args, hk, torch, hepgen, wl)
        res[key] = rec
    return res


def streamed_config4(args, hk, torch, hepgen, first_batch):
    """BASELINE.json configs[4] as defined: `--c4-batches` batches of 5 M events streamed host -> device through
    hepk_analysis_chain_host (Fig. 1), serial and overlapped, plus the kernels alone, against the
    pinned cudaMemcpyAsync host-to-device rate measured here."""
    nb = max(1, args.c4_batches)
    # distinct seeded batches 0 and 1, alternated (generating ten would only add host time to the run)
    second = hepgen.generate(4, batch=1) if nb > 1 else None
    wl = hepgen.concat([first_batch if b % 2 == 0 else second for b in range(nb)])
    N, B = wl.n_events, first_batch.n_events
    hplan = hk.HostChainPlan(wl, batch_events=B, want_event_outputs=False)
    # pinned host -> device copy rate, one 1 GiB cudaMemcpyAsync
    src = torch.empty(1 << 30, dtype=torch.uint8).pin_memory()
    dst = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    dst.copy_(src, non_blocking=True)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    dst.copy_(src, non_blocking=True)
    e1.record()
    torch.cuda.synchronize()
    h2d_gbps = (1 << 30) / (e0.elapsed_time(e1) * 1e-3) / 1e9
    del src, dst
    hplan.run(overlap=True)                      # warm-up
    hplan.zero_hists()
    res = {}
    for name, ov in (("serial", False), ("overlapped", True)):
        torch.cuda.synchronize()
        hk.profile_begin()
        t0 = time.perf_counter()
        hplan.run(overlap=ov)
        dt = time.perf_counter() - t0
        kern_ms, kern_n = hk.profile_end()
        res[name] = {"value": N / dt, "unit": UNIT, "seconds": dt, "h2d_GBps_effective": hplan.h2d_bytes / dt / 1e9}
    res["kernel_only"] = {"value": N / (kern_ms * 1e-3), "unit": UNIT, "chain_kernel_ms_total": kern_ms, "chain_kernel_launches": kern_n}
    counts = hplan.out["hist_counts"].numpy().reshape(5, -1)
    assert (counts.sum(axis=1) == 2 * N * 6).all()
    res.update({"events": N, "batches": nb, "batch_events": B, "h2d_bytes": hplan.h2d_bytes,
                "pinned_h2d_GBps_measured": h2d_gbps,
                "copy_bound_events_per_s": N / (hplan.h2d_bytes / (h2d_gbps * 1e9)),
                "overlapped_frac_of_copy_bound": res["overlapped"]["value"] / (N / (hplan.h2d_bytes / (h2d_gbps * 1e9))),
                "batches_note": "seeded batches 0 and 1 alternated"})
    del hplan
    return res


def single_kernels(args, hk, torch, hepgen, steps=None):
    """Side measurement (BASELINE.json: "single-kernel throughput"): every hepk_* single kernel on the jets /
    muons of one config, CUDA events over K launches, algorithmic bytes per SURVEY.md 8(d) (the method's bytes:
    every needed input element once, every output element once)."""
    steps = steps or args.steps
    cfg = args.config if args.single_kernels else 2
    wl = hepgen.generate(cfg, n_events=args.events)
    inp = hk.upload(wl)
    j, m = inp.jets, inp.muons
    N, Mj, Mm = wl.n_events, j.pt.numel(), m.pt.numel()
    peak, peak_src = measured_peak()
    jsel = hk.select_mask(j.pt, j.eta, 30.0, 2.4)
    msel = hk.select_mask(m.pt, None, 20.0, float("inf"))
    edges = inp.axes["ht"]
    w = inp.weights[0] if inp.weights is not None else None
    ht = hk.segmented_reduce_sum(j.pt, j.offsets, None, jsel)
    sumw = torch.zeros(edges.numel() + 1, dtype=torch.float32, device="cuda")
    sumw2 = torch.zeros(edges.numel() + 1, dtype=torch.float32, device="cuda")
    counts = torch.zeros(edges.numel() + 1, dtype=torch.int64, device="cuda")
    scratch = j.pt.clone()
    wout = torch.empty(N, dtype=torch.float32, device="cuda")
    sumw2d = torch.zeros((22, 32), dtype=torch.float32, device="cuda")
    counts2d = torch.zeros((22, 32), dtype=torch.int64, device="cuda")
    charge = torch.randint(0, 2, (Mm,), device="cuda", dtype=torch.int32) * 2 - 1
    cal = inp.calib
    if cal is None:
        g = hepgen.generate(3, n_events=1000)
        cal = {k: torch.from_numpy(g.calib[k]).cuda() for k in ("pt_edges", "eta_edges", "table")}
    pu_edges = torch.linspace(0, 60, 31, device="cuda")
    pu_table = torch.rand(30, device="cuda") + 0.5
    pu_x = torch.rand(N, device="cuda") * 70 - 5
    wb = 8 if w is not None else 4
    # inputs smaller than the 126 MB L2 (one 4-byte value per event) exist in three copies used in turn, so that a call
    # never finds its inputs left in L2 by the previous one
    turn = [0]

    def rot(copies):
        turn[0] += 1
        return copies[turn[0] % len(copies)]

    hts = [ht, ht.clone(), ht.clone()]
    ws = [w, w.clone(), w.clone()] if w is not None else [None]
    pus = [pu_x, pu_x.clone(), pu_x.clone()]

    def pick():
        i = rot([0, 1, 2])
        return hts[i], ws[i % len(ws)], pus[i]

    cases = {
        "select_mask": (lambda: hk.select_mask(j.pt, j.eta, 30.0, 2.4, out=jsel), 9 * Mj),
        "segmented_reduce_sum[warp-per-event]": (lambda: hk.segmented_reduce_sum(j.pt, j.offsets, None, jsel, variant=1), 12 * N + 5 * Mj),
        "segmented_reduce_sum[block-per-tile]": (lambda: hk.segmented_reduce_sum(j.pt, j.offsets, None, jsel, variant=2), 12 * N + 5 * Mj),
        "segmented_reduce_max": (lambda: hk.segmented_reduce_max(j.pt, j.offsets, None, jsel), 12 * N + 5 * Mj),
        "segmented_reduce_min": (lambda: hk.segmented_reduce_min(j.pt, j.offsets, None, jsel), 12 * N + 5 * Mj),
        "segmented_reduce_count": (lambda: hk.segmented_reduce_count(None, j.offsets, None, jsel), 12 * N + Mj),
        "segmented_reduce_argmax": (lambda: hk.segmented_reduce_argmax(j.pt, j.offsets, None, jsel), 12 * N + 5 * Mj),
        "deltar_mask": (lambda: hk.deltar_mask(j.eta, j.phi, j.offsets, jsel, m.eta, m.phi, m.offsets, msel, 0.4), 16 * N + 9 * Mj + 9 * Mm + Mj),
        "pair_invmass": (lambda: hk.pair_invmass(j.pt, j.eta, j.phi, j.mass, j.offsets, jsel), 8 * N + 17 * Mj + 12 * N),
        "lookup_binned": (lambda: hk.lookup_binned(j.pt, j.eta, cal["pt_edges"], cal["eta_edges"], cal["table"]), 12 * Mj),
        "fill_histogram": (lambda: (lambda h_, w_, p_: hk.fill_histogram(h_, w_, edges, sumw=sumw, counts=counts))(*pick()), wb * N),
        "fill_histogram_w2": (lambda: (lambda h_, w_, p_: hk.fill_histogram_w2(h_, w_, edges, sumw=sumw, sumw2=sumw2, counts=counts))(*pick()), wb * N),
        "event_weight_lookup": (lambda: (lambda h_, w_, p_: hk.event_weight_lookup(w_, p_, pu_edges, pu_table, out=wout))(*pick()),
                                (12 if w is not None else 8) * N),
        # SURVEY.md 8(f-1), the method's bytes: 8 B of offsets + the one 4-byte element + 4 B out (resp. in) per event
        "get_in_offsets[index 0]": (lambda: hk.get_in_offsets(j.pt, j.offsets, 0, fill=0.0), 16 * N),
        "set_in_offsets[index 0]": (lambda: hk.set_in_offsets(scratch, j.offsets, 0, value=1.0), 12 * N),
        "select_opposite_sign[muons]": (lambda: hk.select_opposite_sign(m.pt, charge, m.offsets), 8 * N + 9 * Mm),
        # float64 arithmetic bound on long events; bytes are the selected jets' four columns + offsets + outputs
        "triplet_mass[selected jets]": (lambda: hk.triplet_mass(j.pt, j.eta, j.phi, j.mass, j.offsets, 172.0, None, jsel), 8 * N + 17 * Mj + 16 * N),
        # SURVEY.md 8(f-2)
        "lookup_interp[50 knots]": (lambda: hk.lookup_interp(j.pt, cal["pt_edges"][:50].contiguous(), cal["table"][:50].contiguous()), 8 * Mj),
        "fill_histogram_2d[20x30]": (lambda: hk.fill_histogram_2d(j.eta, j.pt, None, cal["eta_edges"], cal["pt_edges"][:31].contiguous(),
                                                                  sumw=sumw2d, counts=counts2d), 8 * Mj),
        "fill_histogram_2d_w2[20x30]": (lambda: hk.fill_histogram_2d_w2(j.eta, j.pt, None, cal["eta_edges"], cal["pt_edges"][:31].contiguous(),
                                                                        sumw=sumw2d, counts=counts2d, want=("sumw", "counts")), 8 * Mj),
    }
    out = {}
    reps = max(steps, 12)
    side = torch.cuda.Stream()
    for name, (fn, nbytes) in cases.items():
        for _ in range(3):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms_eager = e0.elapsed_time(e1) / steps
        # The same calls captured once into a CUDA graph and replayed: the launches then follow each other on the
        # device without waiting for the Python caller (15-20 us of host time per call, which a 20-70 us kernel
        # does not hide).  The replay is what `ms` reports; the eager loop is kept beside it.
        ms = ms_eager
        timer = "eager"
        try:
            if getattr(args, "sk_eager", False):
                raise KeyError("--sk-eager")
            g = torch.cuda.CUDAGraph()
            with torch.cuda.stream(side):
                fn()
                with torch.cuda.graph(g, stream=side):
                    for _ in range(reps):
                        fn()
            torch.cuda.synchronize()
            g.replay()
            torch.cuda.synchronize()
            e0.record()
            g.replay()
            e1.record()
            torch.cuda.synchronize()
            ms, timer = e0.elapsed_time(e1) / reps, "graph replay of %d calls" % reps
            del g
        except KeyError:
            timer = "eager (--sk-eager)"
        except RuntimeError as exc:                       # a call that cannot be captured keeps the eager figure
            timer = "eager (capture failed: %s)" % str(exc).splitlines()[0][:80]
            torch.cuda.synchronize()
        out[name] = {"ms": ms, "ms_eager": ms_eager, "timer": timer, "algorithmic_bytes": nbytes, "GBps": nbytes / ms / 1e6,
                     "frac_of_peak": nbytes / ms / 1e6 / peak}
    # one 4-byte element per event costs the memory system a 32-byte sector: the f-1 gathers are bound by sectors, not
    # by the method's bytes (profiles/r02c_single_kernels.md: their DRAM traffic runs at ~0.9 of the copy peak)
    for name, sect in (("get_in_offsets[index 0]", (8 + 32 + 4) * N), ("set_in_offsets[index 0]", (8 + 32 + 32) * N)):
        if name in out:
            out[name]["sector_bytes"] = sect
            out[name]["frac_of_peak_by_sectors"] = sect / out[name]["ms"] / 1e6 / peak
    return {"metric": "single-kernel throughput (algorithmic GB/s; side measurement)", "unit": "GB/s",
            "config": {"workload": workload_name(cfg, wl), "events": N, "jets": Mj, "muons": Mm,
                       "l2": "config 1 (132 MB) is L2-resident on B200; config 2 gives HBM figures",
                       "timer": "CUDA events around one replay of a CUDA graph holding >= 12 back-to-back calls through the binding "
                                "(each call's helper kernels and memsets included); ms_eager = the same calls issued from Python",
                       "l2_note": "inputs smaller than L2 (HT, weights, pile-up variable: 40 MB each) rotate over three copies"},
            "peak": peak, "peak_source": peak_src, "steps": steps, "kernels": out}


def main():
    args = parse_args()
    if args.single_kernels:
        import torch
        import hepgen
        from paper_1906_06242_b200 import binding as hk
        torch.cuda.set_device(0)
        hk.lib()
        print(json.dumps(single_kernels(args, hk, torch, hepgen)))
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_hepk(args)


if __name__ == "__main__":
    main()
