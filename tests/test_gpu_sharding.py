"""The sharded CUDA path (PAPER.md:L166 multi-GPU, L66-68 independent events): shards of ONE
device-resident workload — offset slices + content_base + column slices, no rebasing — run through hepk_analysis_chain
and merged must equal the oracle on the whole workload."""
import numpy as np
import pytest
import torch

import hepgen
from oracle import hepo
from _util import assert_exact, assert_tol, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hk():
    from paper_1906_06242_b200 import binding
    binding.lib()
    return binding


@pytest.mark.parametrize("cfg,n,shards", [(2, 400_003, 2), (2, 400_003, 8), (3, 100_001, 3), (4, 40_001, 2), (1, 50_000, 5)])
def test_shards_of_one_workload_equal_the_whole(hk, cfg, n, shards):
    from paper_1906_06242_b200 import sharding
    wl = hepgen.generate(cfg, n_events=n)
    ref = hepo.analysis_chain(wl, want_mask=False)
    inp = hk.upload(wl)
    sc = sharding.ShardedChain(inp, shards, host_jet_offsets=wl.jets.offsets)
    assert len(sc.plans) == shards and sc.shards[0][0] == 0 and sc.shards[-1][1] == n
    assert all(p.desc.jets.content_base == int(wl.jets.offsets[e0]) for p, (e0, _) in zip(sc.plans, sc.shards))
    assert any(p.desc.jets.content_base != 0 for p in sc.plans)
    out = sc.run()
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"], "merged counts")
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], "merged sumw")
    for k in ("njet", "argmax", "maxpt", "minpt", "subpt"):
        assert_exact(to_np(out[k]), ref[k], k)
    for k in ("ht", "mjj"):
        assert_tol(to_np(out[k]), ref[k], k)
    # run twice: per-shard histograms start from zero each time
    out2 = sc.run()
    torch.cuda.synchronize()
    assert_exact(to_np(out2["hist_counts"]), ref["hist_counts"])


def test_shard_with_event_weight_lookup_and_sumw2(hk):
    from paper_1906_06242_b200 import sharding
    wl = hepgen.generate(2, n_events=150_001)
    rng = np.random.default_rng(3)
    evw = dict(x=rng.uniform(-3, 65, wl.n_events).astype(np.float32), edges=np.linspace(0, 60, 31).astype(np.float32),
               table=rng.uniform(0.6, 1.4, 30).astype(np.float32))
    ref = hepo.analysis_chain(wl, want_mask=False, evw=evw, want_sumw2=True)
    inp = hk.upload(wl)
    inp.evw = {k: torch.from_numpy(v).cuda() for k, v in evw.items()}
    out = sharding.ShardedChain(inp, 3, host_jet_offsets=wl.jets.offsets, want_event_outputs=("njet", "ht"), want_sumw2=True).run()
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], "sumw")
    assert_tol(to_np(out["hist_sumw2"]), ref["hist_sumw2"], "sumw2")
    assert_exact(to_np(out["njet"]), ref["njet"])


def test_two_ranks_over_nccl_when_two_gpus():
    """With >= 2 GPUs: one process per GPU over NCCL, each rank its shard through libhepk, histograms all-reduced."""
    if torch.cuda.device_count() < 2:
        pytest.skip("needs 2 GPUs (the one-GPU image of this path is test_shards_of_one_workload_equal_the_whole)")
    import torch.multiprocessing as mp
    from test_multiproc import _free_port
    ctx = mp.get_context("spawn")
    q, port = ctx.Queue(), _free_port()
    procs = [ctx.Process(target=_nccl_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    counts, sumw = q.get(timeout=300)
    for p in procs:
        p.join(timeout=120)
        assert p.exitcode == 0
    wl = hepgen.generate(2, n_events=200_001)
    ref = hepo.analysis_chain(wl, want_mask=False)
    assert_exact(counts, ref["hist_counts"])
    assert_tol(sumw, ref["hist_sumw"], "all-reduced sumw")


def _nccl_worker(rank, world, port, q):
    import os
    import torch.distributed as dist
    from paper_1906_06242_b200 import binding as hk, sharding
    os.environ["MASTER_ADDR"], os.environ["MASTER_PORT"] = "127.0.0.1", str(port)
    torch.cuda.set_device(rank)
    dist.init_process_group("nccl", rank=rank, world_size=world, device_id=torch.device("cuda", rank))
    wl = hepgen.generate(2, n_events=200_001)
    e0, e1 = sharding.event_shards(wl.jets.offsets, world)[rank]
    inp = sharding.shard_inputs(hk.upload(wl), e0, e1, host_offsets=dict(jets=wl.jets.offsets, muons=wl.muons.offsets,
                                                                         electrons=wl.electrons.offsets))
    out, _ = hk.analysis_chain(inp, want_event_outputs=False)
    sharding.merge_histograms([out["hist_counts"], out["hist_sumw"]])
    torch.cuda.synchronize()
    if rank == 0:
        q.put((out["hist_counts"].cpu().numpy(), out["hist_sumw"].cpu().numpy()))
    dist.destroy_process_group()
