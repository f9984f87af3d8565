#!/usr/bin/env python
"""bench.py — throughput of the fused analysis chain (hepk_analysis_chain) on synthetic top-pair-shaped events.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--impl reference]

One "step" = one pass of the whole hot path (selection, dR cleaning, [calibration variants], per-event
reductions, leading-pair mass, weighted histograms — SURVEY.md 8(a) rows a1..a7) over one batch of events.
Default workload: BASELINE.json configs[2] (10,000,000 events; the configuration north_star's ">= 60 % of
B200 peak HBM bandwidth" target is quoted on).  Prints ONE JSON line (rank 0).

  value         events/s, inputs resident in HBM, CUDA events over K steps, max over ranks
  e2e           the same through hepk_analysis_chain_host: PINNED HOST buffers in, host buffers out, every
                host<->device copy inside the timed region
  roofline      the fused chain kernel alone: algorithmic bytes per launch / its average device time
                (CUDA events recorded by the library directly around the kernel), against the measured HBM
                peak of MEASURED_PEAKS.json
  cpu_baseline  the CPU oracle (oracle/, single thread, as it stands) on the same workload, same box

`--impl reference` times the oracle instead (this tier's reference arm): no GPU is touched.
"""
from __future__ import annotations

import argparse
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
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--single-kernels", action="store_true",
                    help="time each single kernel (SURVEY.md 8(a) rows a1-a6) instead of the fused chain; one JSON line")
    ap.add_argument("--variants", type=int, default=None,
                    help="configs 3/4: number of calibration variants (scales 1 +- k*0.0025); the paper's full-systematics scenario is 40")
    ap.add_argument("--tune", default="", help="chain tuning knobs, e.g. warps_per_sm=20,ctas_per_sm=1 (testing only)")
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


def time_oracle(wl, e0, e1):
    from oracle import hepo
    t0 = time.perf_counter()
    res = hepo.analysis_chain(wl, e0, e1, want_mask=False)
    return time.perf_counter() - t0, res


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

    # weak scaling: every rank draws its own batch of the same recipe (events are independent)
    wl = hepgen.generate(args.config, n_events=args.events, batch=rank)
    if args.variants and wl.calib is not None:
        import numpy as _np
        wl.calib["scales"] = (1.0 + 0.0025 * (_np.arange(args.variants) - args.variants // 2)).astype(_np.float32)
    N = wl.n_events
    V = 1 if wl.calib is None else len(wl.calib["scales"])
    inp = hk.upload(wl)
    hists_only = args.config == 4          # config 4 writes histograms only
    tune = {k: int(v) for k, v in (kv.split("=") for kv in args.tune.split(",") if kv)}
    plan = hk.ChainPlan(inp, want_event_outputs=False if hists_only else BENCH_OUTPUTS, tune=tune or None)
    alg_bytes = algorithmic_bytes(wl, event_outputs=not hists_only)
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

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    plan.zero_hists()
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    hk.profile_begin()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        step()
    ev1.record()
    barrier()
    kern_ms, kern_n = hk.profile_end()
    sampler.stop()
    elapsed_ms = ev0.elapsed_time(ev1)
    if world > 1:
        t = torch.tensor([elapsed_ms], dtype=torch.float64, device="cuda")
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        elapsed_ms = float(t.item())
    value = N * world * args.steps / (elapsed_ms * 1e-3)

    # sanity of the timed work: every event of every step landed in every histogram
    counts = plan.out["hist_counts"].cpu().numpy().reshape(V, -1)
    n_hist = len(wl.hists)
    expect = N * n_hist * (world if world > 1 else args.steps)
    assert (counts.sum(axis=1) == expect).all(), (counts.sum(axis=1), expect)

    peak, peak_src = measured_peak()
    per_launch_ms = kern_ms / max(kern_n, 1)
    achieved = alg_bytes / (per_launch_ms * 1e-3) / 1e9
    traffic = None
    tp = os.path.join(ROOT, "profiles", "traffic.csv")       # copied by hand from the ncu --set full capture
    if os.path.exists(tp):
        try:
            import csv
            for row in csv.DictReader(open(tp)):
                if int(row["config"]) == args.config:
                    traffic = int(row["dram_bytes_per_launch"])
        except Exception:
            traffic = None
    roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "traffic": traffic, "kernel": "hepk::dev::chain_kernel", "kernel_ms_per_launch": per_launch_ms,
                "algorithmic_bytes_per_launch": alg_bytes, "bytes_per_event": alg_bytes / N, "peak_source": peak_src,
                "frac_of_nominal_8TBs": achieved / 8000.0}

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": elapsed_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f32", "data": "synthetic",
        "config": {"workload": workload_name(args.config, wl), "events_per_gpu": N, "variants": V,
                   "parallelism": f"events sharded over {world} GPU(s), histogram all-reduce" if world > 1 else "1 GPU",
                   "l2": f"inputs {alg_bytes / 1e9:.2f} GB per step >> 126 MB L2, no flush needed",
                   "outputs": list(BENCH_OUTPUTS) if not hists_only else "histograms only"},
        "roofline": roofline, "clocks": sampler.summary(),
        "gpu_launches": 3 * args.steps,     # chain_wmax_kernel + chain_kernel + chain_finalize_hist per step (the memset is not a kernel)
    }

    # ---- end to end through the C ABI with HOST buffers (rank-local; max over ranks)
    if not args.no_e2e:
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
        n_s = N if args.config <= 2 else min(N, 3_000_000)
        dt, ref = time_oracle(wl, 0, n_s)
        out["cpu_baseline"] = {"value": n_s / dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                               "sample": f"first {n_s:,} of {N:,} events, one pass, {dt:.1f} s, single thread "
                                         f"of {os.cpu_count()} host cores"}
        if n_s == N:      # free parity evidence: one fresh GPU step against the oracle's histograms
            plan.zero_hists()
            plan.run()
            torch.cuda.synchronize()
            same = bool((plan.out["hist_counts"].cpu().numpy() == ref["hist_counts"]).all())
            out["cpu_baseline"]["hist_counts_equal_gpu"] = same

    if rank == 0:
        print(json.dumps(out))
    if world > 1:
        dist.destroy_process_group()


def run_single_kernels(args):
    """Side measurement (BASELINE.json: "single-kernel throughput"): every hepk_* single kernel on the jets /
    muons of one config, CUDA events over K launches, algorithmic bytes per SURVEY.md 8(d)."""
    import torch

    import hepgen
    from paper_1906_06242_b200 import binding as hk

    torch.cuda.set_device(0)
    hk.lib()
    wl = hepgen.generate(args.config, n_events=args.events)
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
    counts = torch.zeros(edges.numel() + 1, dtype=torch.int64, device="cuda")
    scratch = j.pt.clone()
    sumw2d = torch.zeros((22, 32), dtype=torch.float32, device="cuda")
    counts2d = torch.zeros((22, 32), dtype=torch.int64, device="cuda")
    charge = torch.randint(0, 2, (Mm,), device="cuda", dtype=torch.int32) * 2 - 1
    cal = inp.calib
    if cal is None:
        g = hepgen.generate(3, n_events=1000)
        cal = {k: torch.from_numpy(g.calib[k]).cuda() for k in ("pt_edges", "eta_edges", "table")}
    cases = {
        "select_mask": (lambda: hk.select_mask(j.pt, j.eta, 30.0, 2.4, out=jsel), 9 * Mj),
        "segmented_reduce_sum[warp-per-event]": (lambda: hk.segmented_reduce_sum(j.pt, j.offsets, None, jsel, variant=1), 12 * N + 5 * Mj),
        "segmented_reduce_sum[block-per-tile]": (lambda: hk.segmented_reduce_sum(j.pt, j.offsets, None, jsel, variant=2), 12 * N + 5 * Mj),
        "segmented_reduce_max": (lambda: hk.segmented_reduce_max(j.pt, j.offsets, None, jsel), 12 * N + 5 * Mj),
        "segmented_reduce_count": (lambda: hk.segmented_reduce_count(None, j.offsets, None, jsel), 12 * N + Mj),
        "segmented_reduce_argmax": (lambda: hk.segmented_reduce_argmax(j.pt, j.offsets, None, jsel), 12 * N + 5 * Mj),
        "deltar_mask": (lambda: hk.deltar_mask(j.eta, j.phi, j.offsets, jsel, m.eta, m.phi, m.offsets, msel, 0.4), 16 * N + 9 * Mj + 9 * Mm + Mj),
        "pair_invmass": (lambda: hk.pair_invmass(j.pt, j.eta, j.phi, j.mass, j.offsets, jsel), 8 * N + 17 * Mj + 12 * N),
        "lookup_binned": (lambda: hk.lookup_binned(j.pt, j.eta, cal["pt_edges"], cal["eta_edges"], cal["table"]), 12 * Mj),
        "fill_histogram": (lambda: hk.fill_histogram(ht, w, edges, sumw=sumw, counts=counts), (8 if w is not None else 4) * N),
        # 8 B/event of offsets + one 32-byte sector per touched element + the output
        "get_in_offsets[index 0]": (lambda: hk.get_in_offsets(j.pt, j.offsets, 0, fill=0.0), 8 * N + 32 * N + 4 * N),
        "set_in_offsets[index 0]": (lambda: hk.set_in_offsets(scratch, j.offsets, 0, value=1.0), 8 * N + 2 * 32 * N),
        "select_opposite_sign[muons]": (lambda: hk.select_opposite_sign(m.pt, charge, m.offsets), 8 * N + 9 * Mm),
        # ALU-bound on long events; bytes are the selected jets' four columns + offsets + outputs
        "triplet_mass[selected jets]": (lambda: hk.triplet_mass(j.pt, j.eta, j.phi, j.mass, j.offsets, 172.0, None, jsel), 8 * N + 17 * Mj + 16 * N),
        # SURVEY.md 8(f-2)
        "lookup_interp[50 knots]": (lambda: hk.lookup_interp(j.pt, cal["pt_edges"][:50].contiguous(), cal["table"][:50].contiguous()), 8 * Mj),
        "fill_histogram_2d[20x30]": (lambda: hk.fill_histogram_2d(j.eta, j.pt, None, cal["eta_edges"], cal["pt_edges"][:31].contiguous(),
                                                                  sumw=sumw2d, counts=counts2d), 8 * Mj),
    }
    out = {}
    for name, (fn, nbytes) in cases.items():
        for _ in range(max(args.warmup, 3)):
            fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        out[name] = {"ms": ms, "algorithmic_bytes": nbytes, "GBps": nbytes / ms / 1e6, "frac_of_peak": nbytes / ms / 1e6 / peak}
    print(json.dumps({"metric": "single-kernel throughput (algorithmic GB/s; side measurement)", "unit": "GB/s",
                      "config": {"workload": workload_name(args.config, wl), "events": N, "jets": Mj, "muons": Mm,
                                 "l2": "config 1 (132 MB) is L2-resident on B200; use --config 2 for HBM figures"},
                      "peak": peak, "peak_source": peak_src, "steps": args.steps, "kernels": out}))


def main():
    args = parse_args()
    if args.single_kernels:
        run_single_kernels(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_hepk(args)


if __name__ == "__main__":
    main()
