"""Pins of the oracle's SURVEY.md 8(f-2) second half (PAPER.md:L134 lookup-derived event weights, L109 weighted
fill with the sum of squared weights) and of its all-cores timing leg (PAPER.md:L66-68 `prange`).  CPU only."""
import os
import subprocess
import sys

import numpy as np
import pytest

import hepgen
from oracle import build as obuild, hepo
from _util import assert_exact, assert_tol


def _slots(x, edges):
    s = np.searchsorted(edges, x, side="right")      # 0 below, nbins+1 at/after the last edge
    s[np.isnan(x)] = edges.shape[0]                  # NaN -> overflow
    return s


# ---------------------------------------------------------------------------------------------- sumw2
def test_fill_histogram_w2_is_bincount_of_squares():
    rng = np.random.default_rng(1)
    edges = np.linspace(0, 10, 21).astype(np.float32)
    x = rng.uniform(-1, 11, 50_000).astype(np.float32)
    x[::97] = np.nan
    w = rng.normal(1.0, 0.3, x.shape[0]).astype(np.float32)
    sumw, sumw2, counts = hepo.fill_histogram_w2(x, w, edges)
    s = _slots(x, edges)
    want2 = np.bincount(s, w.astype(np.float64) ** 2, minlength=22)
    want1 = np.bincount(s, w.astype(np.float64), minlength=22)
    assert_exact(sumw2, want2.astype(np.float32), "sumw2 == float32(bincount(slot, w^2)) bit for bit")
    assert_exact(sumw, want1.astype(np.float32), "sumw")
    assert_exact(counts, np.bincount(s, minlength=22), "counts")
    # the plain fill is unchanged by the new entry
    sw_plain, ct_plain = hepo.fill_histogram(x, w, edges)
    assert_exact(sumw, sw_plain)
    assert_exact(counts, ct_plain)
    # Cauchy-Schwarz per slot: (sum w)^2 <= n * sum w^2
    assert (want1 ** 2 <= counts * want2 * (1 + 1e-12) + 1e-12).all()


def test_fill_histogram_w2_unit_weights_and_accumulation():
    rng = np.random.default_rng(2)
    edges = np.asarray([0, 1, 2.5, 2.75, 7, 10], np.float32)       # irregular axis
    x = rng.uniform(-2, 12, 10_000).astype(np.float32)
    sumw, sumw2, counts = hepo.fill_histogram_w2(x, None, edges)
    assert_exact(sumw2, counts.astype(np.float32), "weights NULL: sumw2 == counts")
    assert_exact(sumw, counts.astype(np.float32), "weights NULL: sumw == counts")
    # two calls accumulate == one call on the concatenation (values here are exactly representable)
    w = rng.integers(1, 4, x.shape[0]).astype(np.float32)
    a = hepo.fill_histogram_w2(x[:4000], w[:4000], edges)
    b = hepo.fill_histogram_w2(x[4000:], w[4000:], edges, sumw=a[0].copy(), sumw2=a[1].copy(), counts=a[2].copy())
    c = hepo.fill_histogram_w2(x, w, edges)
    for u, v in zip(b, c):
        assert_exact(u, v)
    # a weight of -2 contributes +4 to sumw2 and -2 to sumw
    s1, s2, _ = hepo.fill_histogram_w2(np.asarray([0.5], np.float32), np.asarray([-2], np.float32), edges)
    assert s1[1] == -2.0 and s2[1] == 4.0 and s2.sum() == 4.0


def test_fill_histogram_2d_w2():
    rng = np.random.default_rng(3)
    ex = np.linspace(-2, 2, 9).astype(np.float32)
    ey = np.geomspace(1, 100, 6).astype(np.float32)
    x = rng.uniform(-2.5, 2.5, 20_000).astype(np.float32)
    y = rng.uniform(0.5, 120, 20_000).astype(np.float32)
    w = rng.normal(1, 0.2, 20_000).astype(np.float32)
    sumw, sumw2, counts = hepo.fill_histogram_2d_w2(x, y, w, ex, ey)
    inner2, _, _ = np.histogram2d(x.astype(np.float64), y.astype(np.float64), bins=[ex.astype(np.float64), ey.astype(np.float64)],
                                  weights=w.astype(np.float64) ** 2)
    # numpy closes the last edge; the inputs never sit exactly on it
    assert_tol(sumw2[1:-1, 1:-1], inner2, "inner bins of sumw2 vs np.histogram2d(weights=w^2)")
    sw, ct = hepo.fill_histogram_2d(x, y, w, ex, ey)
    assert_exact(sumw, sw)
    assert_exact(counts, ct)
    # marginal over y == the 1-D fill of x with squared weights
    _, m2, _ = hepo.fill_histogram_w2(x, w, ex)
    assert_tol(sumw2.astype(np.float64).sum(axis=1), m2, "x marginal of sumw2")


# ---------------------------------------------------------------------------------------------- event weight lookup
def test_event_weight_lookup_is_one_float32_multiply():
    rng = np.random.default_rng(4)
    edges = np.linspace(0, 60, 31).astype(np.float32)                 # e.g. number of pileup vertices
    table = rng.uniform(0.5, 1.5, 30).astype(np.float32)
    x = rng.uniform(-5, 70, 100_000).astype(np.float32)
    x[:50] = edges[np.arange(50) % 31]                                # values exactly on edges -> upper bin
    x[50:60] = np.nan
    w = rng.normal(1, 0.1, x.shape[0]).astype(np.float32)
    got = hepo.event_weight_lookup(w, x, edges, table)
    b = np.clip(np.searchsorted(edges, x, side="right") - 1, 0, 29)
    b[np.isnan(x)] = 29                                               # NaN -> last bin (the lookup's clamp rule)
    want = w * table[b]
    assert want.dtype == np.float32
    assert_exact(got, want, "w * table[B(x)] in float32, bit for bit")
    assert_exact(got, w * hepo.lookup_binned(x, None, edges, None, table), "same bin rule as lookup_binned")
    assert_exact(hepo.event_weight_lookup(None, x, edges, table), table[b], "w_in NULL: the table value")
    ones = np.ones(30, np.float32)
    assert_exact(hepo.event_weight_lookup(w, x, edges, ones), w, "unit table: unchanged")


# ---------------------------------------------------------------------------------------------- the chain
def _evw(wl, seed=5):
    rng = np.random.default_rng(seed)
    return dict(x=rng.uniform(-3, 65, wl.n_events).astype(np.float32), edges=np.linspace(0, 60, 31).astype(np.float32),
                table=rng.uniform(0.6, 1.4, 30).astype(np.float32))


@pytest.mark.parametrize("cfg,n", [(1, 20_000), (4, 3_000)])
def test_chain_event_weight_equals_premultiplied_weights(cfg, n):
    """The chain with an event-weight lookup == the chain run on weights multiplied beforehand by
    hepo_event_weight_lookup (the same float32 products, the same float64 sums): bit for bit."""
    wl = hepgen.generate(cfg, n_events=n)
    evw = _evw(wl)
    res = hepo.analysis_chain(wl, want_mask=False, evw=evw, want_sumw2=True)
    wl2 = hepgen.generate(cfg, n_events=n)
    wl2.weights = np.stack([hepo.event_weight_lookup(wl.weights[w], evw["x"], evw["edges"], evw["table"])
                            for w in range(wl.weights.shape[0])])
    ref = hepo.analysis_chain(wl2, want_mask=False, want_sumw2=True)
    assert_exact(res["hist_sumw"], ref["hist_sumw"])
    assert_exact(res["hist_sumw2"], ref["hist_sumw2"])
    assert_exact(res["hist_counts"], ref["hist_counts"])
    for k in ("njet", "ht", "maxpt", "mjj"):
        assert_exact(res[k], ref[k], k)                       # the factor touches weights only
    # and it does something: the unweighted-by-lookup histograms differ
    plain = hepo.analysis_chain(wl, want_mask=False)
    assert not np.array_equal(plain["hist_sumw"], res["hist_sumw"])
    assert_exact(plain["hist_counts"], res["hist_counts"])


def test_chain_sumw2_is_fill_of_the_per_event_outputs():
    """hist_sumw2 of the chain == hepo_fill_histogram_w2 applied to the chain's own per-event observables."""
    wl = hepgen.generate(4, n_events=4_000)
    res = hepo.analysis_chain(wl, want_mask=False, want_sumw2=True)
    V, W = res["layout"]["n_variants"], res["layout"]["n_wvar"]
    spv = res["layout"]["slots_per_variant"]
    s2 = res["hist_sumw2"].reshape(V, W * spv)
    for v in range(V):
        for name in wl.hists:
            p = res["layout"]["prefix"][name]
            nb2 = wl.axes[name].shape[0] + 1
            x = res[name][v].astype(np.float32)
            for w in range(W):
                _, want2, _ = hepo.fill_histogram_w2(x, wl.weights[w], wl.axes[name])
                got = s2[v, W * p + w * nb2: W * p + (w + 1) * nb2]
                assert_exact(got, want2, f"sumw2 v={v} {name} w={w}")
    # without weights sumw2 == counts
    wl.weights = np.ones_like(wl.weights)
    res1 = hepo.analysis_chain(wl, want_mask=False, want_sumw2=True)
    sw, ct = hepo.hist_view(res1, "ht", wl)
    s2v = res1["hist_sumw2"].reshape(V, W * spv)
    p = res1["layout"]["prefix"]["ht"]
    nb2 = wl.axes["ht"].shape[0] + 1
    assert_exact(s2v[:, W * p: W * p + nb2], ct.astype(np.float32))


# ---------------------------------------------------------------------------------------------- all-cores leg
@pytest.mark.parametrize("threads", [2, 3, 0])
def test_omp_chain_equals_single_thread(threads):
    wl = hepgen.generate(3, n_events=10_007)                  # not divisible by the thread counts
    evw = _evw(wl)
    a = hepo.analysis_chain(wl, evw=evw, want_sumw2=True)
    b = hepo.analysis_chain(wl, evw=evw, want_sumw2=True, threads=threads)
    for k in ("njet", "argmax", "ht", "maxpt", "minpt", "mjj", "subpt", "jet_mask", "hist_counts"):
        assert_exact(a[k], b[k], k)
    assert_tol(b["hist_sumw"], a["hist_sumw"], "sumw")
    assert_tol(b["hist_sumw2"], a["hist_sumw2"], "sumw2")
    assert hepo.max_threads() >= 1


# ---------------------------------------------------------------------------------------------- sanitizers
_SAN_SCRIPT = r"""
import sys, ctypes as C
sys.path.insert(0, {root!r})
import numpy as np
from oracle import build as obuild, hepo
obuild.build = lambda force=False: {lib!r}          # the sanitized library instead of libhepo.so
import hepgen
for cfg, n in ((0, 3000), (2, 2000), (4, 600)):
    wl = hepgen.generate(cfg, n_events=n)
    rng = np.random.default_rng(0)
    evw = dict(x=rng.uniform(-3, 65, n).astype(np.float32), edges=np.linspace(0, 60, 31).astype(np.float32),
               table=rng.uniform(0.6, 1.4, 30).astype(np.float32))
    r = hepo.analysis_chain(wl, evw=evw, want_sumw2=True)
    hepo.analysis_chain(wl, threads=2)
    hepo.analysis_chain(wl, 17, n - 5)
    j = wl.jets
    sel = hepo.select_mask(j.pt, j.eta, 30.0, 2.4)
    for op in ("sum", "max", "min", "count", "argmax"):
        hepo.segmented_reduce(op, j.pt, j.offsets, None, sel)
    hepo.deltar_mask(j.eta, j.phi, j.offsets, sel, wl.muons.eta, wl.muons.phi, wl.muons.offsets, None, 0.4)
    hepo.pair_invmass(j.pt, j.eta, j.phi, j.mass, j.offsets, sel)
    hepo.triplet_mass(j.pt, j.eta, j.phi, j.mass, j.offsets, 172.0, None, sel)
    hepo.get_in_offsets(j.pt, j.offsets, 1, None, sel)
    hepo.set_in_offsets(j.pt, j.offsets, 0, value=1.0)
    hepo.select_opposite_sign(wl.muons.pt, np.ones(wl.muons.pt.shape[0], np.int32), wl.muons.offsets)
    hepo.lookup_interp(j.pt, np.linspace(0, 500, 11), np.linspace(1, 2, 11))
    hepo.fill_histogram_w2(j.pt, None, wl.axes["ht"])
    hepo.fill_histogram_2d_w2(j.eta, j.pt, None, np.linspace(-2.5, 2.5, 6), np.linspace(0, 300, 7))
    hepo.event_weight_lookup(None, evw["x"], evw["edges"], evw["table"])
    hepo.validate_offsets(j.offsets, j.pt.shape[0])
print("SANITIZED-RUN-OK")
"""


def test_oracle_under_address_and_ub_sanitizers(tmp_path):
    """the oracle built with -fsanitize=address,undefined runs every entry on small inputs clean."""
    lib = obuild.build_sanitized(str(tmp_path))
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    env = dict(os.environ, LD_PRELOAD=obuild.asan_runtime(), ASAN_OPTIONS="detect_leaks=0:abort_on_error=0",
               UBSAN_OPTIONS="print_stacktrace=1:halt_on_error=1", OMP_NUM_THREADS="2")
    p = subprocess.run([sys.executable, "-c", _SAN_SCRIPT.format(root=root, lib=lib)], env=env, capture_output=True,
                       text=True, timeout=600)
    assert p.returncode == 0, p.stderr[-4000:]
    assert "SANITIZED-RUN-OK" in p.stdout
    assert "ERROR: AddressSanitizer" not in p.stderr and "runtime error:" not in p.stderr, p.stderr[-4000:]
