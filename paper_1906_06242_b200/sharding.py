"""Multi-GPU plumbing of the chain: events are independent, so the path shards by event ranges
with no data-path collective; the only exchange is the histogram merge.  Host logic only."""
from __future__ import annotations

import numpy as np
import torch
import torch.distributed as dist


def event_shards(jet_offsets: np.ndarray, world: int):
    """Contiguous event ranges [e0, e1) per rank, balanced by jet count (jets carry 63 % of the bytes): split
    points by binary search of k * M / world in the jets offsets array."""
    n = len(jet_offsets) - 1
    total = int(jet_offsets[-1] - jet_offsets[0])
    cuts = [0]
    for k in range(1, world):
        target = jet_offsets[0] + (total * k) // world
        e = int(np.searchsorted(jet_offsets, target, side="left"))
        cuts.append(min(max(e, cuts[-1]), n))
    cuts.append(n)
    return [(cuts[r], cuts[r + 1]) for r in range(world)]


def merge_histograms(tensors, group=None):
    """Sum the per-rank histograms in place over the process group (one all-reduce per tensor, <= 122 KB each)."""
    if dist.is_available() and dist.is_initialized() and dist.get_world_size(group) > 1:
        for t in tensors:
            dist.all_reduce(t, op=dist.ReduceOp.SUM, group=group)
    return tensors


def shard_inputs(inp, e0: int, e1: int, host_offsets=None):
    """Device VIEWS of events [e0, e1) of a device-resident workload (binding.ChainInputs): offsets slices, column
    slices starting at the shard's first object with content_base = offsets[e0] (no rebasing, no copies), weight and
    lookup-column slices.  host_offsets: dict name -> numpy offsets, to avoid reading offsets[e0], offsets[e1] back."""
    from .binding import ChainInputs, DeviceCollection

    def coll(c, name):
        if c is None:
            return None
        if host_offsets is not None and name in host_offsets:
            g0, g1 = int(host_offsets[name][e0]), int(host_offsets[name][e1])
        else:
            g0, g1 = (int(v) for v in c.offsets[[e0, e1]].tolist())
        b = c.content_base
        cut = lambda t: None if t is None else t[g0 - b: g1 - b]
        return DeviceCollection(c.offsets[e0: e1 + 1], cut(c.pt), cut(c.eta), cut(c.phi), cut(c.mass), content_base=g0)

    evw = None
    if inp.evw is not None:
        evw = dict(inp.evw, x=inp.evw["x"][e0:e1])
    return ChainInputs(n_events=e1 - e0, jets=coll(inp.jets, "jets"), muons=coll(inp.muons, "muons"),
                       electrons=coll(inp.electrons, "electrons"),
                       weights=None if inp.weights is None else inp.weights[:, e0:e1], cuts=inp.cuts, hists=inp.hists,
                       axes=inp.axes, calib=inp.calib, evw=evw)


class ShardedChain:
    """One device-resident workload run as `n_shards` event shards (jet-balanced contiguous ranges), each through
    hepk_analysis_chain on its own stream, per-event outputs written in place into whole-workload arrays, histograms
    summed afterwards (merge_histograms semantics).  On one GPU this is the single-device image of the multi-GPU
    path: rank r of a job runs shard r on its own device and the histogram sum is the all-reduce."""

    def __init__(self, inp, n_shards, host_jet_offsets=None, want_event_outputs=True, **plan_kwargs):
        from . import binding as hk
        self.inp, self.n_shards = inp, n_shards
        off = host_jet_offsets if host_jet_offsets is not None else inp.jets.offsets.cpu().numpy()
        self.shards = event_shards(off, n_shards)
        V, N, dev = inp.n_variants, inp.n_events, inp.jets.pt.device
        names = () if not want_event_outputs else (hk.ChainPlan.EVENT_OUTPUTS if want_event_outputs is True else tuple(want_event_outputs))
        self.out = {k: torch.empty((V, N), dtype=torch.int32 if k in ("njet", "argmax") else torch.float32, device=dev)
                    for k in names}
        self.plans = []
        for (e0, e1) in self.shards:
            if e1 > e0:
                self.plans.append(hk.ChainPlan(shard_inputs(inp, e0, e1), want_event_outputs=names or False,
                                               out_into=self.out if names else None, out_col=e0, **plan_kwargs))
        self.streams = [torch.cuda.Stream(device=dev) for _ in self.plans]

    def run(self):
        cur = torch.cuda.current_stream()
        for p, st in zip(self.plans, self.streams):
            st.wait_stream(cur)
            p.zero_hists_on(st)
            p.run(stream=st)
        for st in self.streams:
            cur.wait_stream(st)
        res = dict(self.out)
        for k in ("hist_sumw", "hist_sumw2", "hist_counts"):
            parts = [p.out[k] for p in self.plans if k in p.out]
            if parts:
                res[k] = torch.stack(parts).sum(dim=0) if k == "hist_counts" else torch.stack(parts).double().sum(dim=0).float()
        return res
