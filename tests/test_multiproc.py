"""World-size-2 (gloo, CPU) test of the multi-GPU plumbing: event sharding + histogram all-reduce
(SURVEY.md 8(e)).  Each rank runs the oracle chain on its event range; the merged histograms must equal the
oracle's on the whole workload (counts exactly, weighted bins within tolerance)."""
import os
import socket

import numpy as np
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

import hepgen
from _util import assert_exact, assert_tol


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, q):
    from oracle import hepo
    from paper_1906_06242_b200 import sharding
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    wl = hepgen.generate(3, n_events=4001)
    e0, e1 = sharding.event_shards(wl.jets.offsets, world)[rank]
    part = hepo.analysis_chain(wl, e0, e1, want_mask=False)
    counts = torch.from_numpy(part["hist_counts"].astype(np.int64))
    sumw = torch.from_numpy(part["hist_sumw"].astype(np.float64))
    sharding.merge_histograms([counts, sumw])
    n_events = torch.tensor([e1 - e0])
    dist.all_reduce(n_events)
    if rank == 0:
        q.put((counts.numpy(), sumw.numpy(), int(n_events.item()), (e0, e1)))
    dist.destroy_process_group()


def test_sharded_histograms_equal_whole():
    from oracle import hepo
    world = 2
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    counts, sumw, n, (e0, e1) = q.get(timeout=600)      # (a cold `import torch` in two fresh processes can take minutes)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = hepgen.generate(3, n_events=4001)
    ref = hepo.analysis_chain(wl, want_mask=False)
    assert n == wl.n_events and e0 == 0 and 0 < e1 < wl.n_events
    assert_exact(counts, ref["hist_counts"].astype(np.int64), "merged counts")
    assert_tol(sumw, ref["hist_sumw"], "merged sumw")


def test_event_shards_cover_and_balance():
    from paper_1906_06242_b200 import sharding
    wl = hepgen.generate(2, n_events=20_000)
    for world in (1, 2, 3, 8):
        sh = sharding.event_shards(wl.jets.offsets, world)
        assert sh[0][0] == 0 and sh[-1][1] == wl.n_events
        assert all(a[1] == b[0] for a, b in zip(sh, sh[1:]))
        jets = [int(wl.jets.offsets[b] - wl.jets.offsets[a]) for a, b in sh]
        assert max(jets) - min(jets) <= 45          # within one event's jets of the ideal split
    empty = np.zeros(11, np.int64)
    assert sharding.event_shards(empty, 4)[-1][1] == 10
