"""Parity of the single CUDA kernels (through the C ABI) against the CPU oracle, element by element on the
same seeded inputs.  Exact class: masks, counts, argmax/top-2 indices, max/min, unweighted bins.
Tolerance class (1e-5 relative, 1e-6 absolute floor): sums, masses, weighted bins."""
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


def dev(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def misaligned(a, shift=1):
    """Device tensor whose data pointer is offset by `shift` elements from a 256-byte aligned allocation."""
    buf = torch.empty(a.shape[0] + shift + 64, dtype=torch.from_numpy(a[:0]).dtype, device="cuda")
    view = buf[shift:shift + a.shape[0]]
    view.copy_(torch.from_numpy(a))
    return view


@pytest.fixture(scope="module")
def wl1():
    return hepgen.generate(1, n_events=200_037)      # many tiles and a ragged last tile


@pytest.fixture(scope="module")
def wl2():
    return hepgen.generate(2, n_events=150_011)      # heavy tail 30-40 jets, electrons


# --------------------------------------------------------------------------- select_mask
@pytest.mark.parametrize("with_eta", [True, False])
@pytest.mark.parametrize("shift", [0, 1, 3])
def test_select_mask(hk, wl1, with_eta, shift):
    pt, eta = wl1.jets.pt, wl1.jets.eta
    want = hepo.select_mask(pt, eta if with_eta else None, 30.0, 2.4)
    mk = (lambda a: misaligned(a, shift)) if shift else dev
    got = hk.select_mask(mk(pt), mk(eta) if with_eta else None, 30.0, 2.4)
    assert_exact(to_np(got), want)


def test_select_mask_edges(hk):
    eta24 = np.float32(2.4)
    pt = np.array([30.0, np.nextafter(np.float32(30), np.float32(31)), 100, 100, 100, np.nan, 100], np.float32)
    eta = np.array([0, 0, eta24, -eta24, np.nextafter(eta24, np.float32(0)), 0, np.nan], np.float32)
    assert_exact(to_np(hk.select_mask(dev(pt), dev(eta), 30.0, 2.4)), hepo.select_mask(pt, eta, 30.0, 2.4))
    assert hk.select_mask(torch.empty(0, device="cuda"), None, 30.0, 2.4).numel() == 0
    for n in (1, 15, 16, 17, 31, 33, 4097):
        p = (20 + np.random.default_rng(n).exponential(30, n)).astype(np.float32)
        e = np.random.default_rng(n + 1).uniform(-2.5, 2.5, n).astype(np.float32)
        assert_exact(to_np(hk.select_mask(dev(p), dev(e), 30.0, 2.4)), hepo.select_mask(p, e, 30.0, 2.4))


# --------------------------------------------------------------------------- segmented reductions
OPS = ("sum", "max", "min", "count", "argmax")


def _reduce_all(hk, data, off, rows, mask, variant, content_base=0, d_data=None, d_mask=None):
    d_data = dev(data) if d_data is None else d_data
    d_off = dev(off)
    d_rows = None if rows is None else dev(rows)
    if d_mask is None and mask is not None:
        d_mask = dev(mask)
    out = {}
    for op in OPS:
        fn = getattr(hk, f"segmented_reduce_{op}")
        out[op] = to_np(fn(d_data, d_off, d_rows, d_mask, content_base=content_base, variant=variant))
    return out


def _check_reductions(got, data, off, rows, mask, content_base=0):
    for op in OPS:
        want = hepo.segmented_reduce(op, data, off, rows, mask, content_base=content_base)
        if op == "sum":
            assert_tol(got[op], want, op)
        else:
            assert_exact(got[op], want, op)


@pytest.mark.parametrize("variant", [0, 1, 2])
@pytest.mark.parametrize("masks", ["none", "content", "both"])
def test_segmented_reduce_configs(hk, wl1, wl2, variant, masks):
    for wl in (wl1, wl2):
        j = wl.jets
        rng = np.random.default_rng(5)
        mask = (rng.random(j.n_objects) < 0.7).astype(np.uint8) if masks != "none" else None
        rows = (rng.random(wl.n_events) < 0.9).astype(np.uint8) if masks == "both" else None
        got = _reduce_all(hk, j.pt, j.offsets, rows, mask, variant)
        _check_reductions(got, j.pt, j.offsets, rows, mask)


def test_segmented_variants_bitwise_equal(hk, wl2):
    j = wl2.jets
    mask = (np.random.default_rng(8).random(j.n_objects) < 0.6).astype(np.uint8)
    a = _reduce_all(hk, j.pt, j.offsets, None, mask, 1)
    b = _reduce_all(hk, j.pt, j.offsets, None, mask, 2)
    for op in ("count", "max", "min", "argmax"):
        assert_exact(a[op], b[op], op)


@pytest.mark.parametrize("variant", [1, 2])
def test_segmented_reduce_edge_cases(hk, variant):
    rng = np.random.default_rng(21)
    cases = {}
    cases["all_empty"] = np.zeros(300, np.int64)
    cases["single_event"] = np.array([7], np.int64)
    cases["max_size"] = np.full(1000, 40, np.int64)                       # every event at the cap
    c = rng.poisson(3, 5000)
    c[::50] = 0
    c[77] = 9000                                                          # one event larger than any staging buffer
    c[4000] = 2600                                                        # one event that just exceeds the tile buffer
    cases["giant_events"] = c.astype(np.int64)
    c = rng.poisson(30, 700)                                              # tiles that overflow and are cut in pieces
    cases["dense_tiles"] = c.astype(np.int64)
    for name, counts in cases.items():
        off = np.zeros(counts.size + 1, np.int64)
        off[1:] = np.cumsum(counts)
        m = int(off[-1])
        data = rng.normal(50, 30, m).astype(np.float32)
        mask = (rng.random(m) < 0.5).astype(np.uint8)
        rows = (rng.random(counts.size) < 0.8).astype(np.uint8)
        got = _reduce_all(hk, data, off, rows, mask, variant)
        for op in OPS:
            want = hepo.segmented_reduce(op, data, off, rows, mask)
            if op == "sum":
                # signed data: judge the sum against sum|x|
                scale = hepo.segmented_reduce("sum", np.abs(data), off, rows, mask)
                assert np.all(np.abs(got[op].astype(np.float64) - want) <= np.maximum(1e-5 * scale, 1e-6)), name
            else:
                assert_exact(got[op], want, f"{name}:{op}")


@pytest.mark.parametrize("variant", [1, 2])
def test_segmented_ties_nan_and_inf(hk, variant):
    off = np.array([0, 4, 8, 10, 12, 12], np.int64)
    data = np.array([7, 7, 7, 7, 1, 9, 9, 2, np.nan, 3, -np.inf, -np.inf], np.float32)
    mask = np.array([0, 0, 1, 1, 1, 0, 1, 1, 1, 1, 1, 1], np.uint8)
    for mk in (None, mask):
        got = _reduce_all(hk, data, off, None, mk, variant)
        for op in ("max", "min", "count", "argmax"):
            assert_exact(got[op], hepo.segmented_reduce(op, data, off, None, mk), op)
        want = hepo.segmented_reduce("sum", data, off, None, mk)
        assert np.array_equal(np.isnan(got["sum"]), np.isnan(want))


@pytest.mark.parametrize("variant", [1, 2])
@pytest.mark.parametrize("shift", [1, 2, 3])
def test_segmented_content_base_and_misalignment(hk, wl1, variant, shift):
    j = wl1.jets
    e0 = 12345
    base = int(j.offsets[e0])
    mask = (np.random.default_rng(2).random(j.n_objects) < 0.7).astype(np.uint8)
    data_s, mask_s, off_s = j.pt[base:], mask[base:], j.offsets[e0:]
    got = _reduce_all(hk, data_s, off_s, None, mask_s, variant, content_base=base,
                      d_data=misaligned(data_s, shift), d_mask=misaligned(mask_s, shift + 4))
    _check_reductions(got, data_s, off_s, None, mask_s, content_base=base)


# --------------------------------------------------------------------------- deltar_mask
def test_deltar_mask_configs(hk, wl1, wl2):
    for wl, second in ((wl1, "muons"), (wl2, "muons"), (wl2, "electrons")):
        j, l = wl.jets, getattr(wl, second)
        rng = np.random.default_rng(3)
        for use_sel in (False, True):
            s1 = (rng.random(j.n_objects) < 0.7).astype(np.uint8) if use_sel else None
            s2 = (rng.random(l.n_objects) < 0.8).astype(np.uint8) if use_sel else None
            want = hepo.deltar_mask(j.eta, j.phi, j.offsets, s1, l.eta, l.phi, l.offsets, s2, 0.4)
            got = hk.deltar_mask(dev(j.eta), dev(j.phi), dev(j.offsets), None if s1 is None else dev(s1),
                                 dev(l.eta), dev(l.phi), dev(l.offsets), None if s2 is None else dev(s2), 0.4)
            assert_exact(to_np(got), want)
            assert want.sum() > 100


def test_deltar_mask_edge_cases(hk):
    rng = np.random.default_rng(4)
    n = 3000
    c1 = rng.poisson(6, n)
    c2 = rng.poisson(2, n)
    c1[5], c2[5] = 5000, 3          # giant collection-1 event
    c1[900], c2[900] = 4, 2000      # giant collection-2 event
    c1[100:140] = 40                # dense run: tile cut in pieces
    c2[100:140] = 12
    c1[200:260] = 0
    c2[300:380] = 0
    off1 = np.zeros(n + 1, np.int64); off1[1:] = np.cumsum(c1)
    off2 = np.zeros(n + 1, np.int64); off2[1:] = np.cumsum(c2)
    m1, m2 = int(off1[-1]), int(off2[-1])
    eta1 = rng.uniform(-2.5, 2.5, m1).astype(np.float32); phi1 = rng.uniform(-np.pi, np.pi, m1).astype(np.float32)
    eta2 = rng.uniform(-2.5, 2.5, m2).astype(np.float32); phi2 = rng.uniform(-np.pi, np.pi, m2).astype(np.float32)
    s1 = (rng.random(m1) < 0.7).astype(np.uint8); s2 = (rng.random(m2) < 0.7).astype(np.uint8)
    want = hepo.deltar_mask(eta1, phi1, off1, s1, eta2, phi2, off2, s2, 0.4)
    got = hk.deltar_mask(dev(eta1), dev(phi1), dev(off1), dev(s1), dev(eta2), dev(phi2), dev(off2), dev(s2), 0.4)
    assert_exact(to_np(got), want)
    # misaligned columns + content_base on both collections
    e0 = 1000
    b1, b2 = int(off1[e0]), int(off2[e0])
    want = hepo.deltar_mask(eta1[b1:], phi1[b1:], off1[e0:], s1[b1:], eta2[b2:], phi2[b2:], off2[e0:], s2[b2:], 0.4, b1, b2)
    got = hk.deltar_mask(misaligned(eta1[b1:], 1), misaligned(phi1[b1:], 2), dev(off1[e0:]), misaligned(s1[b1:], 3),
                         misaligned(eta2[b2:], 3), misaligned(phi2[b2:], 1), dev(off2[e0:]), misaligned(s2[b2:], 5), 0.4,
                         base1=b1, base2=b2)
    assert_exact(to_np(got), want)


def test_deltar_threshold_and_wrap_exactness(hk):
    # pairs placed within a few ulp of the threshold and across the +-pi seam: float32, no FMA, same as the oracle
    rng = np.random.default_rng(6)
    n = 200_000
    off = np.arange(n + 1, dtype=np.int64)
    eta2 = rng.uniform(-2.4, 2.4, n).astype(np.float32)
    phi2 = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    ang = rng.uniform(0, 2 * np.pi, n)
    r = 0.4 * (1 + rng.uniform(-3e-7, 3e-7, n))
    eta1 = (eta2 + r * np.cos(ang)).astype(np.float32)
    phi1 = (phi2 + r * np.sin(ang))
    phi1 = ((phi1 + np.pi) % (2 * np.pi) - np.pi).astype(np.float32)
    want = hepo.deltar_mask(eta1, phi1, off, None, eta2, phi2, off, None, 0.4)
    got = hk.deltar_mask(dev(eta1), dev(phi1), dev(off), None, dev(eta2), dev(phi2), dev(off), None, 0.4)
    assert 0.2 < want.mean() < 0.8
    assert_exact(to_np(got), want)


# --------------------------------------------------------------------------- pair_invmass
def test_pair_invmass_configs(hk, wl1, wl2):
    for wl in (wl1, wl2):
        j = wl.jets
        for mask in (None, hepo.select_mask(j.pt, j.eta, 30.0, 2.4)):
            wm, w1, w2 = hepo.pair_invmass(j.pt, j.eta, j.phi, j.mass, j.offsets, mask)
            gm, g1, g2 = hk.pair_invmass(dev(j.pt), dev(j.eta), dev(j.phi), dev(j.mass), dev(j.offsets),
                                         None if mask is None else dev(mask))
            assert_exact(to_np(g1), w1, "i1")
            assert_exact(to_np(g2), w2, "i2")
            assert_tol(to_np(gm), wm, "mass")


def test_pair_invmass_hard_cases(hk):
    """Near-collinear pairs, pairs straddling the +-pi seam, tiny masses, equal-pt ties: the places where a
    float32 E^2-p^2 evaluation loses everything."""
    rng = np.random.default_rng(13)
    n = 100_000
    off = 2 * np.arange(n + 1, dtype=np.int64)
    pt = (20 + rng.exponential(60, 2 * n)).astype(np.float32)
    pt[0:2000:2] = pt[1:2000:2]                                      # ties
    eta = rng.uniform(-2.5, 2.5, 2 * n).astype(np.float32)
    phi = rng.uniform(-np.pi, np.pi, 2 * n).astype(np.float32)
    mass = rng.exponential(10, 2 * n).astype(np.float32)
    k = n // 4
    eta[1:2 * k:2] = (eta[0:2 * k:2] + rng.normal(0, 1e-3, k)).astype(np.float32)       # collinear
    phi[1:2 * k:2] = (phi[0:2 * k:2] + rng.normal(0, 1e-3, k)).astype(np.float32)
    np.clip(phi, -np.float32(np.pi), np.float32(np.pi), out=phi)
    mass[0:2 * k] = rng.exponential(0.05, 2 * k).astype(np.float32)                     # tiny masses
    s = slice(2 * k, 4 * k)
    phi[s][0::2] = (np.pi - rng.exponential(0.02, k)).astype(np.float32)                # seam straddlers
    phi[s][1::2] = (-np.pi + rng.exponential(0.02, k)).astype(np.float32)
    eta[s][1::2] = (eta[s][0::2] + rng.normal(0, 0.02, k)).astype(np.float32)
    mass[s] = rng.exponential(0.5, 2 * k).astype(np.float32)
    mass[4 * k:5 * k] = 0.0                                                              # massless
    wm, w1, w2 = hepo.pair_invmass(pt, eta, phi, mass, off)
    gm, g1, g2 = hk.pair_invmass(dev(pt), dev(eta), dev(phi), dev(mass), dev(off))
    assert_exact(to_np(g1), w1)
    assert_exact(to_np(g2), w2)
    assert_tol(to_np(gm), wm, "mass")


def test_pair_invmass_edge_cases(hk):
    rng = np.random.default_rng(14)
    c = rng.poisson(4, 2000)
    c[:40] = 0
    c[40:80] = 1
    c[500] = 7000                      # event larger than the staging buffer
    c[600:650] = 40
    off = np.zeros(c.size + 1, np.int64); off[1:] = np.cumsum(c)
    m = int(off[-1])
    pt = (20 + rng.exponential(30, m)).astype(np.float32)
    pt[rng.random(m) < 0.01] = np.nan
    eta = rng.uniform(-2.5, 2.5, m).astype(np.float32); phi = rng.uniform(-np.pi, np.pi, m).astype(np.float32)
    mass = rng.exponential(10, m).astype(np.float32)
    mask = (rng.random(m) < 0.6).astype(np.uint8)
    e0 = 300
    b = int(off[e0])
    for args, kw, dv in (
        ((pt, eta, phi, mass, off, mask), {}, (dev(pt), dev(eta), dev(phi), dev(mass), dev(off), dev(mask))),
        ((pt[b:], eta[b:], phi[b:], mass[b:], off[e0:], mask[b:]), dict(content_base=b),
         (misaligned(pt[b:], 1), misaligned(eta[b:], 2), misaligned(phi[b:], 3), misaligned(mass[b:], 1), dev(off[e0:]),
          misaligned(mask[b:], 7))),
    ):
        wm, w1, w2 = hepo.pair_invmass(*args, **kw)
        gm, g1, g2 = hk.pair_invmass(*dv, **kw)
        assert_exact(to_np(g1), w1)
        assert_exact(to_np(g2), w2)
        assert_tol(to_np(gm), wm, "mass")


# --------------------------------------------------------------------------- lookup_binned
def test_lookup_binned(hk, wl2):
    cal = hepgen.calibration_table(np.random.default_rng(3))
    j = wl2.jets
    x = j.pt.copy()
    y = j.eta.copy()
    x[:60] = np.concatenate([cal["pt_edges"], [5.0, 1e6, np.nan, 20.0, 3000.0, 19.999, 2999.9, 0, -1]]).astype(np.float32)[:60]
    y[:21] = cal["eta_edges"]
    y[21:24] = [np.nan, -3.0, 3.0]
    want = hepo.lookup_binned(x, y, cal["pt_edges"], cal["eta_edges"], cal["table"])
    got = hk.lookup_binned(dev(x), dev(y), dev(cal["pt_edges"]), dev(cal["eta_edges"]), dev(cal["table"]))
    assert_exact(to_np(got), want)
    # 1-D form, misaligned, odd length
    xs = x[: 100_003]
    t1 = np.arange(50, dtype=np.float32)
    want = hepo.lookup_binned(xs, None, cal["pt_edges"], None, t1)
    got = hk.lookup_binned(misaligned(xs, 3), None, dev(cal["pt_edges"]), None, dev(t1))
    assert_exact(to_np(got), want)
    # irregular edges (binary-search path) and a uniform pt axis (linear guess)
    rng = np.random.default_rng(4)
    pe = np.unique(np.concatenate([[20.0], np.sort(rng.uniform(20, 3000, 37)), [3000.0]])).astype(np.float32)
    tab = rng.uniform(0.9, 1.1, (pe.size - 1, 20)).astype(np.float32)
    x[100:100 + pe.size] = pe
    assert_exact(to_np(hk.lookup_binned(dev(x), dev(y), dev(pe), dev(cal["eta_edges"]), dev(tab))),
                 hepo.lookup_binned(x, y, pe, cal["eta_edges"], tab))
    pl = np.linspace(25.0, 500.0, 51).astype(np.float32)
    x[200:251] = pl
    assert_exact(to_np(hk.lookup_binned(dev(x), dev(y), dev(pl), dev(cal["eta_edges"]), dev(cal["table"]))),
                 hepo.lookup_binned(x, y, pl, cal["eta_edges"], cal["table"]))


# --------------------------------------------------------------------------- fill_histogram
def test_fill_histogram(hk, wl2):
    res = hepo.analysis_chain(wl2, want_mask=False)
    edges = hepgen.hist_axes(["ht"])["ht"]
    x = res["ht"][0].copy()
    x[:5] = [np.nan, np.inf, -np.inf, 1000.0, -1.0]
    x[5:106] = edges
    w = wl2.weights[0]
    ws, wc = hepo.fill_histogram(x, w, edges)
    gs, gc = hk.fill_histogram(dev(x), dev(w), dev(edges))
    assert_exact(to_np(gc), wc, "counts")
    assert_tol(to_np(gs), ws, "sumw")
    # unweighted: sumw == counts exactly; accumulation across two calls
    gs, gc = hk.fill_histogram(dev(x[:70_001]), None, dev(edges))
    gs, gc = hk.fill_histogram(misaligned(x[70_001:], 1), None, dev(edges), gs, gc)
    assert_exact(to_np(gc), wc)
    assert_exact(to_np(gs), wc.astype(np.float32))


def test_fill_histogram_concentrated_and_nonuniform(hk):
    rng = np.random.default_rng(15)
    n = 2_000_003
    # njet-like: everything in a handful of bins (worst case for float32 accumulation)
    x = rng.poisson(4, n).astype(np.float32)
    w = rng.normal(1, 0.1, n).astype(np.float32)
    edges = np.linspace(0, 50, 101).astype(np.float32)
    ws, wc = hepo.fill_histogram(x, w, edges)
    gs, gc = hk.fill_histogram(dev(x), dev(w), dev(edges))
    assert_exact(to_np(gc), wc)
    assert_tol(to_np(gs), ws, "sumw")
    # non-uniform and inexact edges (the arithmetic guess must be repaired by the edge check)
    edges = np.sort(np.concatenate([[0.0], rng.uniform(0, 10, 61), np.arange(1, 40) * 0.05 + 10, [20.0]])).astype(np.float32)
    x = np.concatenate([rng.uniform(-1, 21, 300_000).astype(np.float32), edges, np.nextafter(edges, np.float32(-1)),
                        np.nextafter(edges, np.float32(99))])
    ws, wc = hepo.fill_histogram(x, None, edges)
    gs, gc = hk.fill_histogram(dev(x), None, dev(edges))
    assert_exact(to_np(gc), wc)
    edges = (np.arange(0, 201) * np.float32(0.05)).astype(np.float32)         # width 0.05: inexact edges
    x = np.concatenate([rng.uniform(-0.5, 10.5, 500_000).astype(np.float32), edges])
    ws, wc = hepo.fill_histogram(x, None, edges)
    gs, gc = hk.fill_histogram(dev(x), None, dev(edges))
    assert_exact(to_np(gc), wc)


def test_fill_histogram_output_subsets_axes_and_sizes(hk):
    """The lane-private kernel's cell layouts (counts only, sums only, both), its three axis modes (uniform, log-spaced,
    irregular), pointers that are not 16-byte aligned, and a histogram too large for lane-private copies (per-CTA
    bins), all against the oracle; +-inf, NaN and exact edges included."""
    rng = np.random.default_rng(77)
    n = 300_007
    w = rng.normal(1, 0.1, n).astype(np.float32)
    axes = {
        "uniform": np.linspace(0, 500, 61).astype(np.float32),
        "log": np.geomspace(20, 3000, 51).astype(np.float32),
        "irregular": np.sort(np.concatenate([[0.0], rng.uniform(0, 500, 40), [500.0]])).astype(np.float32),
        "large": np.linspace(0, 500, 2001).astype(np.float32),
    }
    for name, edges in axes.items():
        x = (rng.exponential(120, n) - 5).astype(np.float32)
        x[:4] = [np.nan, np.inf, -np.inf, 0.0]
        x[4:4 + edges.size] = edges
        ws, wc = hepo.fill_histogram(x, w, edges)
        us, uc = hepo.fill_histogram(x, None, edges)
        for shift in (0, 1):
            xd, wd = (misaligned(x, 1), misaligned(w, 3)) if shift else (dev(x), dev(w))
            gs, gc = hk.fill_histogram(xd, wd, dev(edges))
            assert_exact(to_np(gc), wc, name + " counts")
            assert_tol(to_np(gs), ws, name + " sumw")
            gs, gc = hk.fill_histogram(xd, wd, dev(edges), want_counts=False)
            assert gc is None
            assert_tol(to_np(gs), ws, name + " sumw alone")
            gs, gc = hk.fill_histogram(xd, wd, dev(edges), want_sumw=False)
            assert gs is None
            assert_exact(to_np(gc), wc, name + " counts alone")
            gs, gc = hk.fill_histogram(xd, None, dev(edges))
            assert_exact(to_np(gc), uc, name + " unweighted counts")
            assert_exact(to_np(gs), uc.astype(np.float32), name + " unweighted sumw")


# --------------------------------------------------------------------------- dense collections (fewer lanes per tile)
@pytest.mark.parametrize("mean1,mean2", [(30, 6), (90, 20), (400, 3), (7, 70)])
def test_jagged_kernels_on_dense_collections(hk, mean1, mean2):
    """Collections dense enough that 32 lanes per tile would overflow the fixed staging buffers: the streaming
    kernels (hepk_tiles.cu) then take 16, 8, ... lanes per tile, decided on the device from offsets[n_events].
    Odd total sizes and shifted pointers also exercise the array-end and array-start slices."""
    rng = np.random.default_rng(1000 + mean1)
    n = 4003
    c1 = rng.poisson(mean1, n).astype(np.int64)
    c2 = rng.poisson(mean2, n).astype(np.int64)
    c1[17] = 0; c2[23] = 0; c1[n - 1] += 3
    off1 = np.zeros(n + 1, np.int64); off1[1:] = np.cumsum(c1)
    off2 = np.zeros(n + 1, np.int64); off2[1:] = np.cumsum(c2)
    m1, m2 = int(off1[-1]), int(off2[-1])
    pt = (20 + rng.exponential(30, m1)).astype(np.float32)
    eta1 = rng.uniform(-2.5, 2.5, m1).astype(np.float32); phi1 = rng.uniform(-np.pi, np.pi, m1).astype(np.float32)
    mass = rng.exponential(10, m1).astype(np.float32)
    eta2 = rng.uniform(-2.5, 2.5, m2).astype(np.float32); phi2 = rng.uniform(-np.pi, np.pi, m2).astype(np.float32)
    s1 = (rng.random(m1) < 0.7).astype(np.uint8); s2 = (rng.random(m2) < 0.8).astype(np.uint8)
    rows = (rng.random(n) < 0.9).astype(np.uint8)
    for shift in (0, 3):
        mk = (lambda a: misaligned(a, shift)) if shift else dev
        got = _reduce_all(hk, pt, off1, rows, s1, 2, d_data=mk(pt), d_mask=mk(s1))
        _check_reductions(got, pt, off1, rows, s1)
        got = _reduce_all(hk, pt, off1, None, None, 2, d_data=mk(pt))
        _check_reductions(got, pt, off1, None, None)
        want = hepo.deltar_mask(eta1, phi1, off1, s1, eta2, phi2, off2, s2, 0.4)
        g = hk.deltar_mask(mk(eta1), mk(phi1), dev(off1), mk(s1), mk(eta2), mk(phi2), dev(off2), mk(s2), 0.4)
        assert_exact(to_np(g), want)
        wm, w1, w2 = hepo.pair_invmass(pt, eta1, phi1, mass, off1, s1)
        gm, g1, g2 = hk.pair_invmass(mk(pt), mk(eta1), mk(phi1), mk(mass), dev(off1), mk(s1))
        assert_exact(to_np(g1), w1, "i1"); assert_exact(to_np(g2), w2, "i2")
        assert_tol(to_np(gm), wm, "mass")


def test_jagged_kernels_with_columns_of_different_alignment(hk, wl2):
    """Columns of one collection that do not share their alignment modulo 16 bytes cannot be staged with one slice
    geometry: the launch takes the global-memory path (one lane per event).  Same results."""
    j, l = wl2.jets, wl2.muons
    n = 20_001
    jo, lo_ = j.offsets[:n + 1], l.offsets[:n + 1]
    mj, ml = int(jo[-1]), int(lo_[-1])
    pt, eta, phi, mass = j.pt[:mj], j.eta[:mj], j.phi[:mj], j.mass[:mj]
    sel = hepo.select_mask(pt, eta, 30.0, 2.4)
    want = hepo.deltar_mask(eta, phi, jo, sel, l.eta[:ml], l.phi[:ml], lo_, None, 0.4)
    got = hk.deltar_mask(misaligned(eta, 1), misaligned(phi, 2), dev(jo), dev(sel), misaligned(l.eta[:ml], 3), dev(l.phi[:ml]),
                         dev(lo_), None, 0.4)
    assert_exact(to_np(got), want)
    wm, w1, w2 = hepo.pair_invmass(pt, eta, phi, mass, jo, sel)
    gm, g1, g2 = hk.pair_invmass(misaligned(pt, 1), dev(eta), misaligned(phi, 3), misaligned(mass, 2), dev(jo), dev(sel))
    assert_exact(to_np(g1), w1, "i1"); assert_exact(to_np(g2), w2, "i2")
    assert_tol(to_np(gm), wm, "mass")
