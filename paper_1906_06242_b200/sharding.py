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
