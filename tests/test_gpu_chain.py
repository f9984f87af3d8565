"""Parity of the fused CUDA chain (hepk_analysis_chain / hepk_analysis_chain_host, through the C ABI)
against the CPU oracle's chain on the same seeded events.  Exact class: jet masks, njet, argmax, maxpt,
minpt, histogram counts.  Tolerance class (1e-5 rel, 1e-6 abs): ht, mjj, subpt(exact in fact), weighted bins."""
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


def compare(out, ref, wl, plan=None, e0=0, e1=None, check_hists=True, what=""):
    sl = slice(e0, e1)
    for k in ("njet", "argmax", "maxpt", "minpt", "subpt"):
        assert_exact(to_np(out[k])[:, sl] if e1 else to_np(out[k]), ref[k], f"{what}{k}")
    for k in ("ht", "mjj"):
        assert_tol(to_np(out[k])[:, sl] if e1 else to_np(out[k]), ref[k], f"{what}{k}")
    if "jet_mask" in out and "jet_mask" in ref:
        assert_exact(to_np(out["jet_mask"]), ref["jet_mask"], f"{what}jet_mask")
    if check_hists:
        assert_exact(to_np(out["hist_counts"]), ref["hist_counts"], f"{what}hist_counts")
        assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], f"{what}hist_sumw")


def run_gpu(hk, wl, **kw):
    inp = hk.upload(wl)
    out, plan = hk.analysis_chain(inp, want_mask=True, **kw)
    torch.cuda.synchronize()
    return out, plan


@pytest.mark.parametrize("config,n", [(0, None), (1, 200_037), (2, 300_011), (3, 100_003), (4, 30_001)])
def test_chain_matches_oracle(hk, config, n):
    wl = hepgen.generate(config, n_events=n)
    ref = hepo.analysis_chain(wl)
    out, plan = run_gpu(hk, wl)
    compare(out, ref, wl)
    # invariants on the device result itself
    for name in wl.hists:
        sw, ct = plan.hist_view(name)
        assert (to_np(ct).sum(axis=1) == wl.n_events).all()


def test_chain_is_repeatable_and_accumulates(hk):
    wl = hepgen.generate(2, n_events=50_000)
    ref = hepo.analysis_chain(wl, want_mask=False)
    inp = hk.upload(wl)
    plan = hk.ChainPlan(inp)
    plan.run(); plan.run()
    torch.cuda.synchronize()
    assert_exact(to_np(plan.out["hist_counts"]), 2 * ref["hist_counts"])       # histograms accumulate
    assert_tol(to_np(plan.out["hist_sumw"]), 2.0 * ref["hist_sumw"].astype(np.float64))
    assert_exact(to_np(plan.out["njet"]), ref["njet"])                          # per-event outputs are overwritten


@pytest.mark.parametrize("tune", [dict(cap_jets=64, cap_leptons=32), dict(cap_jets=300, cap_leptons=16),
                                  dict(cap_jets=4096, cap_leptons=1024, ctas_per_sm=1)])
def test_chain_small_buffers_cut_tiles_and_giant_events(hk, tune):
    """Staging buffers far smaller than a tile: tiles are processed in pieces, and events larger than the
    buffers go through the per-event global-memory path.  Results must not change."""
    for config in (2, 3):
        wl = hepgen.generate(config, n_events=6_000)
        ref = hepo.analysis_chain(wl)
        out, _ = run_gpu(hk, wl, tune=tune)
        compare(out, ref, wl, what=f"cfg{config} {tune} ")


def _custom(n, cj, cm, ce, seed=0, config=2):
    """Workload with prescribed multiplicities."""
    wl = hepgen.generate(config, n_events=n, seed=seed)
    rng = np.random.default_rng(seed + 100)

    def coll(counts, mass):
        off = np.zeros(n + 1, np.int64)
        off[1:] = np.cumsum(counts)
        m = int(off[-1])
        return hepgen.Collection(off, (20 + rng.exponential(30, m)).astype(np.float32),
                                 rng.uniform(-2.5, 2.5, m).astype(np.float32),
                                 rng.uniform(-np.pi, np.pi, m).astype(np.float32),
                                 (rng.exponential(10, m) if mass is None else np.full(m, mass)).astype(np.float32))
    wl.jets, wl.muons = coll(cj, None), coll(cm, 0.1057)
    wl.electrons = coll(ce, 0.000511) if ce is not None else None
    return wl


def test_chain_edge_multiplicities(hk):
    n = 3000
    rng = np.random.default_rng(1)
    z = np.zeros(n, np.int64)
    cases = {
        "no_jets_at_all": (z, rng.poisson(1.5, n), rng.poisson(1, n)),
        "no_leptons_at_all": (rng.poisson(8, n), z, z),
        "everything_empty": (z, z, z),
        "all_at_cap": (np.full(n, 40), np.full(n, 6), np.full(n, 6)),
        "no_electron_collection": (rng.poisson(8, n), rng.poisson(1.5, n), None),
        "single_jet_events": (np.ones(n, np.int64), rng.poisson(1.5, n), rng.poisson(1, n)),
    }
    g = rng.poisson(8, n)
    g[17], g[1500], g[2999] = 3000, 700, 5000          # giant events (first tile, middle, last event)
    gm = rng.poisson(1.5, n)
    gm[1501] = 900                                     # giant lepton event
    cases["giant_events"] = (g, gm, rng.poisson(1, n))
    for name, (cj, cm, ce) in cases.items():
        wl = _custom(n, cj, cm, ce, seed=3)
        ref = hepo.analysis_chain(wl)
        out, _ = run_gpu(hk, wl)
        compare(out, ref, wl, what=name + " ")
    for n1 in (1, 2, 127, 128, 129):
        wl = hepgen.generate(2, n_events=n1, seed=9)
        compare(run_gpu(hk, wl)[0], hepo.analysis_chain(wl), wl, what=f"n={n1} ")


def test_chain_ties_and_threshold_values(hk):
    """Hand-built ties (equal pt) and values sitting exactly on the cuts and on bin edges."""
    n = 4000
    rng = np.random.default_rng(2)
    wl = _custom(n, rng.poisson(6, n) + 2, rng.poisson(1.5, n), rng.poisson(1, n), seed=5)
    j = wl.jets
    pt = j.pt
    for e in range(0, n, 3):                           # equal leading pts -> first index must win, next is subleading
        a, b = j.offsets[e], j.offsets[e + 1]
        k = rng.integers(2, b - a + 1)
        idx = rng.choice(np.arange(a, b), size=k, replace=False)
        pt[idx] = np.float32(200.0)
    pt[rng.random(pt.size) < 0.02] = np.float32(30.0)                      # exactly on the pt cut (fails: strict >)
    j.eta[rng.random(pt.size) < 0.02] = np.float32(2.4)                    # exactly on the eta cut
    j.eta[rng.random(pt.size) < 0.02] = np.float32(-2.4)
    pt[rng.random(pt.size) < 0.02] = np.float32(500.0)                     # on the last edge of the maxpt axis -> overflow
    ref = hepo.analysis_chain(wl)
    out, _ = run_gpu(hk, wl)
    compare(out, ref, wl)
    assert (ref["argmax"][0] >= 0).sum() > 1000


@pytest.mark.parametrize("shifts", [((1, 2, 3, 1), (3, 0, 1, 2), (2, 2, 1, 0)),        # columns disagree: per-event path
                                    ((1, 1, 1, 1), (3, 3, 3, 3), (2, 2, 2, 2))])       # staged path with a shift
def test_chain_misaligned_columns_and_content_base(hk, shifts):
    """Columns that are only 4-byte aligned, and an event range given as an offsets slice plus content_base."""
    wl = hepgen.generate(2, n_events=20_000, seed=4)
    e0, e1 = 4_001, 17_777
    ref = hepo.analysis_chain(wl, e0, e1)
    inp = hk.upload(wl)

    def shifted(t, s):
        buf = torch.empty(t.numel() + 8, dtype=t.dtype, device="cuda")
        v = buf[s: s + t.numel()]
        v.copy_(t)
        return v

    def cut(c, wlc, shifts):
        g0, g1 = int(wlc.offsets[e0]), int(wlc.offsets[e1])
        cols = [shifted(getattr(c, nm)[g0:g1].contiguous(), s) for nm, s in zip(("pt", "eta", "phi", "mass"), shifts)]
        return hk.DeviceCollection(c.offsets[e0:e1 + 1].contiguous(), *cols, content_base=g0)
    inp.jets = cut(inp.jets, wl.jets, shifts[0])
    inp.muons = cut(inp.muons, wl.muons, shifts[1])
    inp.electrons = cut(inp.electrons, wl.electrons, shifts[2])
    inp.weights = inp.weights[:, e0:e1].contiguous()
    inp.n_events = e1 - e0
    out, plan = hk.analysis_chain(inp, want_mask=True)
    torch.cuda.synchronize()
    g0, g1 = int(wl.jets.offsets[e0]), int(wl.jets.offsets[e1])
    ref["jet_mask"] = ref["jet_mask"][:, g0:g1]
    compare(out, ref, wl)


def test_chain_irregular_axes_and_odd_weights(hk):
    """Histogram axes the arithmetic bin guess cannot be used on (binary-search path), and weights the
    fixed-point bins cannot hold (non-finite -> float path) or that span many orders of magnitude."""
    wl = hepgen.generate(4, n_events=20_000, seed=11)
    rng = np.random.default_rng(5)
    for name, hi in (("ht", 1000.0), ("mjj", 1000.0), ("njet", 50.0)):
        nb = wl.axes[name].size - 1
        e = np.sort(rng.uniform(0.0, hi, nb - 1)).astype(np.float32)
        wl.axes[name] = np.unique(np.concatenate([[np.float32(0)], e, [np.float32(hi)]])).astype(np.float32)
    ref = hepo.analysis_chain(wl, want_mask=False)
    out, _ = hk.analysis_chain(hk.upload(wl))
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"], "irregular axes counts")
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], "irregular axes sumw")
    # weights with a wide but same-signed range: every bin within tolerance of the float64 sum
    wl = hepgen.generate(2, n_events=30_000, seed=12)
    wl.weights = (wl.weights * np.float32(3.0e-7)).astype(np.float32)
    ref = hepo.analysis_chain(wl, want_mask=False)
    out, _ = hk.analysis_chain(hk.upload(wl))
    torch.cuda.synchronize()
    got, want = to_np(out["hist_sumw"]).astype(np.float64), ref["hist_sumw"].astype(np.float64)
    assert np.all(np.abs(got - want) <= 1e-5 * np.abs(want) + 1e-12), "tiny weights"
    # one infinite weight: the launch falls back to float bins; only that event's bins become inf
    wl = hepgen.generate(1, n_events=5_000, seed=13)
    wl.weights[0, 1234] = np.float32(np.inf)
    ref = hepo.analysis_chain(wl, want_mask=False)
    out, _ = hk.analysis_chain(hk.upload(wl))
    torch.cuda.synchronize()
    got, want = to_np(out["hist_sumw"]), ref["hist_sumw"]
    assert_exact(np.isinf(got), np.isinf(want), "inf bins")
    fin = np.isfinite(want)
    assert_tol(got[fin], want[fin], "finite bins next to an inf weight")
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"])


def test_chain_calibration_axis_modes(hk):
    """Calibration tables on a log-spaced x uniform grid (arithmetic bin guess), on irregular edges (binary search),
    and with jets sitting exactly on edges and outside the table."""
    rng = np.random.default_rng(21)
    for kind in ("regular", "irregular", "linear_pt"):
        wl = hepgen.generate(3, n_events=30_000, seed=22)
        if kind == "irregular":
            wl.calib["pt_edges"] = np.unique(np.concatenate([[20.0], np.sort(rng.uniform(20, 3000, 49)), [3000.0]])).astype(np.float32)
            wl.calib["eta_edges"] = np.unique(np.concatenate([[-2.5], np.sort(rng.uniform(-2.5, 2.5, 19)), [2.5]])).astype(np.float32)
            wl.calib["table"] = rng.uniform(0.9, 1.1, (wl.calib["pt_edges"].size - 1, wl.calib["eta_edges"].size - 1)).astype(np.float32)
        if kind == "linear_pt":
            wl.calib["pt_edges"] = np.linspace(25.0, 400.0, 51).astype(np.float32)     # jets below and above the table
        pe, ee = wl.calib["pt_edges"], wl.calib["eta_edges"]
        k = rng.integers(0, wl.jets.pt.size, 4000)
        wl.jets.pt[k] = pe[rng.integers(0, pe.size, 4000)]                             # exactly on pt edges
        k = rng.integers(0, wl.jets.pt.size, 4000)
        wl.jets.eta[k] = ee[rng.integers(0, ee.size, 4000)]                            # exactly on eta edges
        ref = hepo.analysis_chain(wl)
        out, _ = run_gpu(hk, wl)
        compare(out, ref, wl, what=f"calib {kind} ")


@pytest.mark.parametrize("config,n", [(1, 150_001), (2, 200_003), (3, 80_001)])
def test_chain_common_shape_build(hk, config, n):
    """The launch shape bench.py times (njet, ht, maxpt, argmax, mjj + HT / leading-pt histograms, one weight column)
    runs a build of the kernel with its feature word fixed at compile time: same results as the generic build."""
    wl = hepgen.generate(config, n_events=n)
    ref = hepo.analysis_chain(wl, want_mask=False)
    names = ("njet", "ht", "maxpt", "argmax", "mjj")
    out, plan = hk.analysis_chain(hk.upload(wl), want_event_outputs=names)
    torch.cuda.synchronize()
    assert set(out) == set(names) | {"hist_sumw", "hist_counts"}
    for k in ("njet", "argmax", "maxpt"):
        assert_exact(to_np(out[k]), ref[k], k)
    for k in ("ht", "mjj"):
        assert_tol(to_np(out[k]), ref[k], k)
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"])
    full, _ = hk.analysis_chain(hk.upload(wl))                    # generic build
    torch.cuda.synchronize()
    for k in names:
        assert_exact(to_np(out[k]), to_np(full[k]), f"common vs generic {k}")


def test_chain_forty_variants(hk):
    """The paper's full-systematics scenario ("increasing the computational complexity ... by about
    40x"): 40 calibration variants in one pass."""
    wl = hepgen.generate(3, n_events=20_011)
    wl.calib["scales"] = (1.0 + 0.0025 * (np.arange(40) - 20)).astype(np.float32)
    ref = hepo.analysis_chain(wl)
    out, _ = run_gpu(hk, wl)
    assert to_np(out["njet"]).shape == (40, wl.n_events)
    compare(out, ref, wl, what="40 variants ")
    assert (np.diff(ref["njet"].astype(np.int64), axis=0) >= 0).all()      # larger scale never loses a jet


def test_chain_optional_outputs(hk):
    wl = hepgen.generate(1, n_events=20_000)
    ref = hepo.analysis_chain(wl, want_mask=False)
    inp = hk.upload(wl)
    out, _ = hk.analysis_chain(inp, want_event_outputs=False)              # histograms only
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"])
    out, _ = hk.analysis_chain(inp, want_hists=False)                      # per-event outputs only
    torch.cuda.synchronize()
    compare(out, ref, wl, check_hists=False)
    inp.weights = None                                                      # weights NULL -> sumw == counts
    out, plan = hk.analysis_chain(inp)
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_sumw"]), ref["hist_counts"].astype(np.float32))


@pytest.mark.parametrize("overlap", [False, True])
def test_chain_host_streaming(hk, overlap):
    """hepk_analysis_chain_host: host buffers in, host buffers out, batches with and without copy/compute overlap."""
    for config, n, batch in ((2, 100_003, 30_000), (4, 20_001, 7_000)):
        wl = hepgen.generate(config, n_events=n)
        ref = hepo.analysis_chain(wl, want_mask=False)
        plan = hk.HostChainPlan(wl, batch_events=batch)
        out = plan.run(overlap=overlap)
        compare({k: v for k, v in out.items()}, ref, wl, what=f"cfg{config} ")
        out = plan.run(overlap=overlap)                                    # histograms accumulate on the host side too
        assert_exact(to_np(out["hist_counts"]), 2 * ref["hist_counts"])


BENCH_OUTPUTS = ("njet", "ht", "maxpt", "argmax", "mjj")       # what bench.py asks for (the common-shape build)


def _oracle_full(wl):
    """The oracle over ALL events of a full-size workload, on every host core (the all-cores leg is pinned to the
    single-thread checker in tests/test_oracle_weights.py: per-event outputs and counts identical, sums in tolerance)."""
    return hepo.analysis_chain(wl, want_mask=False, threads=0)


def test_chain_full_size_config2_generic_build(hk):
    """BASELINE.json config 2 at full size (10 M events), all seven per-event outputs (the GENERIC kernel build):
    per-event outputs on sampled event ranges the single-thread oracle recomputes, histograms over ALL events."""
    wl = hepgen.generate(2)
    inp = hk.upload(wl)
    plan = hk.ChainPlan(inp)
    plan.run()
    torch.cuda.synchronize()
    N = wl.n_events
    for e0 in (0, 1_234_567, 5_000_001, N - 200_000):
        ref = hepo.analysis_chain(wl, e0, e0 + 200_000, want_mask=False)
        out = {k: plan.out[k][:, e0:e0 + 200_000] for k in ("njet", "argmax", "maxpt", "minpt", "subpt", "ht", "mjj")}
        compare(out, ref, wl, check_hists=False, what=f"events {e0}.. ")
    ref = hepo.analysis_chain(wl, want_mask=False)
    assert_exact(to_np(plan.out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(plan.out["hist_sumw"]), ref["hist_sumw"])
    tot = wl.weights.astype(np.float64).sum()
    for name in wl.hists:
        sw, ct = plan.hist_view(name)
        assert to_np(ct).sum() == N
        assert abs(to_np(sw).astype(np.float64).sum() - tot) <= 1e-5 * tot


def _compare_all_events(out, ref, names):
    for k in names:
        if k in ("ht", "mjj"):
            assert_tol(to_np(out[k]), ref[k], k)
        else:
            assert_exact(to_np(out[k]), ref[k], k)


def test_chain_full_size_config2_bench_launch(hk):
    """Config 2, 10 M events, in the launch configuration bench.py times (its five outputs: the common-shape build):
    EVERY per-event output of EVERY event against the oracle, histogram counts exact, weighted bins in tolerance."""
    wl = hepgen.generate(2)
    ref = _oracle_full(wl)
    plan = hk.ChainPlan(hk.upload(wl), want_event_outputs=BENCH_OUTPUTS)
    plan.run()
    torch.cuda.synchronize()
    _compare_all_events(plan.out, ref, BENCH_OUTPUTS)
    assert_exact(to_np(plan.out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(plan.out["hist_sumw"]), ref["hist_sumw"])


def test_chain_full_size_config3(hk):
    """BASELINE.json config 3 at full size: 10 M events x 5 calibration variants, bench.py's launch configuration."""
    wl = hepgen.generate(3)
    ref = _oracle_full(wl)
    plan = hk.ChainPlan(hk.upload(wl), want_event_outputs=BENCH_OUTPUTS)
    plan.run()
    torch.cuda.synchronize()
    _compare_all_events(plan.out, ref, BENCH_OUTPUTS)
    assert_exact(to_np(plan.out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(plan.out["hist_sumw"]), ref["hist_sumw"])
    e0 = 7_000_000                      # and a range through the single-thread checker
    chk = hepo.analysis_chain(wl, e0, e0 + 100_000, want_mask=False)
    for k in ("njet", "argmax", "maxpt"):
        assert_exact(to_np(plan.out[k][:, e0:e0 + 100_000]), chk[k], k)


@pytest.mark.parametrize("group", [0, 5])
def test_chain_full_size_config4_batch(hk, group):
    """One batch of BASELINE.json config 4 at full size: 5 M events, 300 weighted histograms, histograms only
    (bench.py's launch configuration).  Every CTA sees ~34 k events, so the hot bins cross the overflow threshold of
    the privatised bins many times and are moved out while other warps keep filling (group = 5: all variants in one
    launch, the 33,660-bin layout; 0: the automatic variant groups)."""
    wl = hepgen.generate(4)
    ref = _oracle_full(wl)
    plan = hk.ChainPlan(hk.upload(wl), want_event_outputs=False, tune=dict(variants_per_pass=group) if group else None)
    plan.run()
    torch.cuda.synchronize()
    assert_exact(to_np(plan.out["hist_counts"]), ref["hist_counts"])
    assert_tol(to_np(plan.out["hist_sumw"]), ref["hist_sumw"])
    plan.run()                          # accumulates
    torch.cuda.synchronize()
    assert_exact(to_np(plan.out["hist_counts"]), 2 * ref["hist_counts"])


# ---------------------------------------------------------------------------------------------- SURVEY.md 8(f-2)
def _evw_np(wl, seed=5):
    rng = np.random.default_rng(seed)
    return dict(x=rng.uniform(-3, 65, wl.n_events).astype(np.float32), edges=np.linspace(0, 60, 31).astype(np.float32),
                table=rng.uniform(0.6, 1.4, 30).astype(np.float32))


@pytest.mark.gpu
@pytest.mark.parametrize("cfg,n", [(1, 200_003), (2, 100_001), (4, 20_001)])
def test_chain_event_weight_lookup_and_sumw2(hk, cfg, n):
    """hepk_chain_desc.evw_* and hist_sumw2 against the oracle."""
    wl = hepgen.generate(cfg, n_events=n)
    evw = _evw_np(wl)
    ref = hepo.analysis_chain(wl, want_mask=False, evw=evw, want_sumw2=True)
    inp = hk.upload(wl)
    inp.evw = {k: torch.from_numpy(v).cuda() for k, v in evw.items()}
    out, plan = hk.analysis_chain(inp, want_sumw2=True)
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"], "counts")
    assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], "sumw with lookup factor")
    assert_tol(to_np(out["hist_sumw2"]), ref["hist_sumw2"], "sumw2 with lookup factor")
    assert_exact(to_np(out["njet"]), ref["njet"])
    # sumw2 alone, without weights and factor: equals the counts
    inp2 = hk.upload(wl)
    inp2.weights = None
    out2, _ = hk.analysis_chain(inp2, want_event_outputs=False, want_sumw2=True)
    torch.cuda.synchronize()
    V, W = 1 if wl.calib is None else len(wl.calib["scales"]), 1
    assert_exact(to_np(out2["hist_sumw2"]), to_np(out2["hist_counts"]).astype(np.float32), "sumw2 == counts for unit weights")


@pytest.mark.gpu
@pytest.mark.parametrize("kind", ["outlier", "mixed_sign", "one_bin", "one_bin_1M", "tiny_and_huge"])
def test_chain_weight_dynamic_range(hk, kind):
    """Weighted bins with a dynamic range inside one launch: the fixed-point bins are only used when the
    weights span at most a factor 8; every case must stay within the tolerance of the float64 oracle."""
    wl = hepgen.generate(2, n_events=1_000_003 if kind == "one_bin_1M" else 150_001)
    rng = np.random.default_rng(11)
    w = wl.weights.copy()
    if kind == "outlier":
        w[0, 12345] = 2000.0                                   # one large generator weight sets max|w|
    elif kind == "mixed_sign":
        w[0] *= rng.choice(np.float32([-1.0, 1.0]), w.shape[1], p=[0.1, 0.9])
    elif kind in ("one_bin", "one_bin_1M"):
        wl.jets.pt[:] = 25.0                                   # no clean jets: every event lands in the first HT bin
        # (1 M events: ~6.8 k entries per CTA in one fixed-point bin, moved out several times before 2^31)
    elif kind == "tiny_and_huge":
        w[0] *= np.float32(10.0) ** rng.integers(-3, 4, w.shape[1]).astype(np.float32)
    wl.weights = np.ascontiguousarray(w, dtype=np.float32)
    ref = hepo.analysis_chain(wl, want_mask=False, want_sumw2=True)
    out, _ = hk.analysis_chain(hk.upload(wl), want_event_outputs=False, want_sumw2=True)
    torch.cuda.synchronize()
    assert_exact(to_np(out["hist_counts"]), ref["hist_counts"])
    if kind == "mixed_sign":
        # cancelling sums: the bound is relative to sum |w| of the bin (include/hepk.h), checked against sumw2-free abs sums
        absref = hepo.analysis_chain(_with_weights(wl, np.abs(wl.weights)), want_mask=False)["hist_sumw"]
        err = np.abs(to_np(out["hist_sumw"]).astype(np.float64) - ref["hist_sumw"])
        assert (err <= 1e-5 * np.abs(absref) + 1e-6).all(), err.max()
    else:
        assert_tol(to_np(out["hist_sumw"]), ref["hist_sumw"], f"sumw ({kind})")
    assert_tol(to_np(out["hist_sumw2"]), ref["hist_sumw2"], f"sumw2 ({kind})")


def _with_weights(wl, w):
    import copy
    c = copy.copy(wl)
    c.weights = np.ascontiguousarray(w, dtype=np.float32)
    return c


@pytest.mark.gpu
def test_chain_host_event_weight_and_sumw2(hk):
    wl = hepgen.generate(3, n_events=60_001)
    evw = _evw_np(wl)
    ref = hepo.analysis_chain(wl, want_mask=False, evw=evw, want_sumw2=True)
    hp = hk.HostChainPlan(wl, batch_events=17_000, want_sumw2=True, evw=evw)
    out = hp.run(overlap=True)
    assert_exact(out["hist_counts"].numpy(), ref["hist_counts"])
    assert_tol(out["hist_sumw"].numpy(), ref["hist_sumw"], "host path sumw")
    assert_tol(out["hist_sumw2"].numpy(), ref["hist_sumw2"], "host path sumw2")
    for k in ("njet", "argmax", "maxpt"):
        assert_exact(out[k].numpy(), ref[k], k)
    assert_tol(out["ht"].numpy(), ref["ht"], "ht")
