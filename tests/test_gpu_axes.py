"""Parity of the bin search on every kind of axis (through the C ABI, against the CPU oracle, bit-exact).

The lookup and histogram kernels find a bin by an arithmetic guess on axes that are uniform in v or in log2 v, fixed by
one step against the edges (padded copies of the edges absorb the range tests: hepk_common.cuh pad_axis_find), and by
a binary search on any other axis; which of the three an axis takes is decided per launch.  The results are exact
class (the bin of a value is B(v), edges[b] <= v < edges[b+1]; readings R5 / R9 for NaN and
out-of-range values), so every kind of axis, pairs of kinds, and the values where a guess can go wrong (every edge and
its two float32 neighbours, +-0, denormals, +-inf, NaN, negative values on a log axis, the largest float) must agree
with the oracle's search bit for bit.
"""
import itertools
import zlib

import numpy as np
import pytest
import torch

from oracle import hepo
from _util import assert_exact, assert_tol, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hk():
    from paper_1906_06242_b200 import binding
    binding.lib()
    return binding


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def axis(kind, rng):
    """float32 edges, strictly ascending"""
    if kind == "uniform":
        e = np.linspace(-2.5, 2.5, 21)
    elif kind == "uniform_jitter":           # accepted as uniform (every edge within 0.45 bins), but the guess is off by one often
        e = np.linspace(20.0, 500.0, 41)
        e[1:-1] += rng.uniform(-0.4, 0.4, 39) * 12.0
    elif kind == "log":
        e = np.geomspace(20.0, 3000.0, 31)
    elif kind == "log_jitter":
        e = 2.0 ** (np.linspace(np.log2(0.5), np.log2(800.0), 26) + np.r_[0, rng.uniform(-0.4, 0.4, 24), 0] * (np.log2(1600.0) / 25))
    elif kind == "irregular":
        e = np.unique(np.r_[-3.0, np.sort(rng.uniform(-3, 70, 17)) ** 3 / 400.0, 900.0])
    elif kind == "one_bin":
        e = np.array([1.0, 2.0])
    elif kind == "two_bins":
        e = np.array([-1.0, 0.0, 4.0])
    elif kind == "tiny_log":                 # lower edge close to the smallest normal float: denormal values lie below it
        e = np.geomspace(2e-38, 1e-30, 9)
    else:
        raise ValueError(kind)
    e = np.unique(e.astype(np.float32))
    assert e.size >= 2
    return e


KINDS = ["uniform", "uniform_jitter", "log", "log_jitter", "irregular", "one_bin", "two_bins", "tiny_log"]


def values(e, rng, n):
    """n float32 values: the axis range and beyond at random, then every edge with its float32 neighbours and the
    special values"""
    lo, hi = float(e[0]), float(e[-1])
    span = hi - lo
    v = rng.uniform(lo - 0.2 * span, hi + 0.2 * span, n).astype(np.float32)
    if lo > 0:
        v[: n // 2] = np.exp(rng.uniform(np.log(lo) - 1.0, np.log(hi) + 1.0, n // 2)).astype(np.float32)
    inf = np.float32(np.inf)
    sp = np.r_[e, np.nextafter(e, -inf), np.nextafter(e, inf),
               np.array([0.0, -0.0, 1e-45, -1e-45, 1e-39, 1.1754944e-38, np.inf, -np.inf, np.nan, -1.0, -1e30, 3.4028235e38,
                         -3.4028235e38], dtype=np.float32)].astype(np.float32)
    v[-sp.size:] = sp
    rng.shuffle(v)
    return v


@pytest.mark.parametrize("kx,ky", list(itertools.product(KINDS, ["uniform", "log_jitter", "irregular", "one_bin"]))
                         + [("log", "log"), ("uniform_jitter", "uniform_jitter"), ("tiny_log", "tiny_log")])
def test_two_axis_kernels_on_axis_kinds(hk, kx, ky):
    rng = np.random.default_rng(zlib.crc32(f"{kx}/{ky}".encode()))
    ex, ey = axis(kx, rng), axis(ky, rng)
    n = 40_003
    x, y = values(ex, rng, n), values(ey, rng, n)
    rng.shuffle(y)
    # lookup_binned: the table holds the flat bin index, so a wrong bin on either axis shows
    table = np.arange((ex.size - 1) * (ey.size - 1), dtype=np.float32).reshape(ex.size - 1, ey.size - 1)
    assert_exact(to_np(hk.lookup_binned(cu(x), cu(y), cu(ex), cu(ey), cu(table))), hepo.lookup_binned(x, y, ex, ey, table),
                 "lookup_binned")
    # fill_histogram_2d: counts only (integer path), then weighted
    w = rng.normal(1.0, 0.1, n).astype(np.float32)
    _, ct = hk.fill_histogram_2d(cu(x), cu(y), None, cu(ex), cu(ey), want_sumw=False)
    sw_ref, ct_ref = hepo.fill_histogram_2d(x, y, w, ex, ey)
    assert_exact(to_np(ct), ct_ref, "fill_histogram_2d counts")
    sw, ct = hk.fill_histogram_2d(cu(x), cu(y), cu(w), cu(ex), cu(ey))
    assert_exact(to_np(ct), ct_ref, "fill_histogram_2d counts (weighted call)")
    assert_tol(to_np(sw), sw_ref, "fill_histogram_2d sumw")
    # the general histogram kernel
    rs, r2, rc = hepo.fill_histogram_2d_w2(x, y, w, ex, ey)
    gs, g2, gc = hk.fill_histogram_2d_w2(cu(x), cu(y), cu(w), cu(ex), cu(ey))
    assert_exact(to_np(gc), rc, "fill_histogram_2d_w2 counts")
    assert_tol(to_np(gs), rs, "fill_histogram_2d_w2 sumw")
    assert_tol(to_np(g2), r2, "fill_histogram_2d_w2 sumw2")


@pytest.mark.parametrize("kind", KINDS)
@pytest.mark.parametrize("shift", [0, 1])
def test_one_axis_kernels_on_axis_kinds(hk, kind, shift):
    rng = np.random.default_rng(zlib.crc32(kind.encode()) + shift)
    e = axis(kind, rng)
    n = 50_001
    xa = values(e, rng, n + shift)
    x = xa[shift:]
    xd = cu(xa)[shift:]                      # shift = 1: not 16-byte aligned (scalar path)
    nb = e.size - 1
    t1 = np.arange(nb, dtype=np.float32) + 0.5
    assert_exact(to_np(hk.lookup_binned(xd, None, cu(e), None, cu(t1))), hepo.lookup_binned(x, None, e, None, t1), "lookup_binned 1-D")
    w = rng.normal(1.0, 0.1, n).astype(np.float32)
    assert_exact(to_np(hk.event_weight_lookup(cu(w), xd, cu(e), cu(t1))), hepo.event_weight_lookup(w, x, e, t1), "event_weight_lookup")
    # interpolation over the edges as knots: knots are reproduced exactly, values outside take the end values
    ys = rng.uniform(0.9, 1.1, e.size).astype(np.float32)
    got, want = to_np(hk.lookup_interp(xd, cu(e), cu(ys))), hepo.lookup_interp(x, e, ys)
    assert_tol(got, want, "lookup_interp")
    on_knot = np.isin(x, e)
    assert_exact(got[on_knot], want[on_knot], "lookup_interp on the knots")
    out = ~(x > e[0]) | ~(x < e[-1])         # (NaN included)
    assert_exact(got[out], want[out], "lookup_interp outside the knots")
    # 1-D histograms: the lane-private kernel and the general one (all three outputs)
    sw_ref, ct_ref = hepo.fill_histogram(x, w, e)
    sw, ct = hk.fill_histogram(xd, cu(w), cu(e))
    assert_exact(to_np(ct), ct_ref, "fill_histogram counts")
    assert_tol(to_np(sw), sw_ref, "fill_histogram sumw")
    rs, r2, rc = hepo.fill_histogram_w2(x, w, e)
    gs, g2, gc = hk.fill_histogram_w2(xd, cu(w), cu(e))
    assert_exact(to_np(gc), rc, "fill_histogram_w2 counts")
    assert_tol(to_np(gs), rs, "fill_histogram_w2 sumw")
    assert_tol(to_np(g2), r2, "fill_histogram_w2 sumw2")


def test_large_one_axis_histogram_takes_the_general_kernel(hk):
    """5,000 bins do not fit lane-private copies: the general kernel (shared-memory atomics, padded axis) on one axis"""
    rng = np.random.default_rng(77)
    for e in (np.linspace(0.0, 1000.0, 5001).astype(np.float32), np.geomspace(1.0, 1e6, 5001).astype(np.float32)):
        x = values(e, rng, 300_007)
        w = rng.normal(1.0, 0.1, x.size).astype(np.float32)
        rs, r2, rc = hepo.fill_histogram_w2(x, w, e)
        gs, g2, gc = hk.fill_histogram_w2(cu(x), cu(w), cu(e))
        assert_exact(to_np(gc), rc, "counts")
        assert_tol(to_np(gs), rs, "sumw")
        assert_tol(to_np(g2), r2, "sumw2")


def test_tables_at_the_shared_memory_limits(hk):
    """The largest tables each entry accepts (include/hepk.h states the limits; the padded copies of the edges count),
    and one step beyond: refused with HEPK_ERR_UNSUPPORTED, never a launch with too little shared memory."""
    rng = np.random.default_rng(5)
    # lookup_interp: 16 bytes of shared memory per knot, 200 KB
    for nk, log in ((12_800, False), (12_800, True)):
        xs = (np.geomspace(1.0, 1e5, nk) if log else np.linspace(0.0, 1000.0, nk)).astype(np.float32)
        ys = rng.uniform(0.9, 1.1, nk).astype(np.float32)
        x = values(xs[::37], rng, 200_001)
        assert_tol(to_np(hk.lookup_interp(cu(x), cu(xs), cu(ys))), hepo.lookup_interp(x, xs, ys), "lookup_interp, 12,800 knots")
    xs = np.linspace(0.0, 1000.0, 12_801).astype(np.float32)
    with pytest.raises(hk.HepkError):
        hk.lookup_interp(cu(xs), cu(xs), cu(xs))
    # lookup_binned: 2 (nx + 1) + 2 (ny + 1) + nx ny floats, 200 KB
    ex, ey = np.linspace(-5.0, 5.0, 201).astype(np.float32), np.geomspace(10.0, 5000.0, 241).astype(np.float32)
    table = rng.uniform(0.5, 1.5, (200, 240)).astype(np.float32)
    x, y = values(ex, rng, 200_001), values(ey, rng, 200_001)
    assert_exact(to_np(hk.lookup_binned(cu(x), cu(y), cu(ex), cu(ey), cu(table))), hepo.lookup_binned(x, y, ex, ey, table),
                 "lookup_binned, 200 x 240 table")
    ex2 = np.linspace(-5.0, 5.0, 221).astype(np.float32)
    with pytest.raises(hk.HepkError):
        hk.lookup_binned(cu(x), cu(y), cu(ex2), cu(ey), cu(np.zeros((220, 240), np.float32)))
    # fill_histogram_2d: (nx + 2) (ny + 2) = 16384 slots
    ex, ey = np.linspace(-3.0, 3.0, 127).astype(np.float32), np.geomspace(20.0, 2000.0, 127).astype(np.float32)
    x, y = values(ex, rng, 300_001), values(ey, rng, 300_001)
    w = rng.normal(1.0, 0.1, x.size).astype(np.float32)
    sw_ref, ct_ref = hepo.fill_histogram_2d(x, y, w, ex, ey)
    sw, ct = hk.fill_histogram_2d(cu(x), cu(y), cu(w), cu(ex), cu(ey))
    assert_exact(to_np(ct), ct_ref, "fill_histogram_2d counts, 16384 slots")
    assert_tol(to_np(sw), sw_ref, "fill_histogram_2d sumw, 16384 slots")
    with pytest.raises(hk.HepkError):
        hk.fill_histogram_2d(cu(x), cu(y), None, cu(np.linspace(-3.0, 3.0, 128).astype(np.float32)), cu(ey))
