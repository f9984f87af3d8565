"""Parity of the SURVEY.md 8(f-2) second half (PAPER.md:L134 event weights from lookups, PAPER.md:L109 weighted fills with
the sum of squared weights) through the C ABI against the CPU oracle on the same seeded inputs."""
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
    return None if a is None else torch.from_numpy(np.ascontiguousarray(a)).cuda()


@pytest.mark.parametrize("n", [0, 1, 1023, 2_000_003])
@pytest.mark.parametrize("axis", ["uniform", "log", "irregular"])
def test_event_weight_lookup_bit_exact(hk, n, axis):
    rng = np.random.default_rng(n + len(axis))
    if axis == "uniform":
        edges = np.linspace(0, 60, 31).astype(np.float32)
    elif axis == "log":
        edges = np.geomspace(1, 500, 26).astype(np.float32)
    else:
        edges = np.sort(rng.uniform(0, 60, 18)).astype(np.float32)
    nb = edges.size - 1
    table = rng.uniform(0.5, 1.5, nb).astype(np.float32)
    x = rng.uniform(float(edges[0]) - 5, float(edges[-1]) + 5, n).astype(np.float32)
    if n > 100:
        x[:nb + 1] = edges                                # exactly on every edge
        x[100:110] = np.nan
        x[110] = np.inf
        x[111] = -np.inf
    w = rng.normal(1, 0.2, n).astype(np.float32)
    want = hepo.event_weight_lookup(w, x, edges, table)
    got = hk.event_weight_lookup(cu(w), cu(x), cu(edges), cu(table))
    assert_exact(to_np(got), want, "w * table[B(x)]")
    assert_exact(to_np(hk.event_weight_lookup(None, cu(x), cu(edges), cu(table))), hepo.event_weight_lookup(None, x, edges, table))
    if n > 8:      # misaligned views take the scalar path; in place is allowed
        xm, wm = cu(x)[1:], cu(w)[1:].clone()
        hk.event_weight_lookup(wm, xm, cu(edges), cu(table), out=wm)
        assert_exact(to_np(wm), want[1:], "in place, misaligned")


@pytest.mark.parametrize("n", [0, 1, 1000, 3_000_001])
@pytest.mark.parametrize("weights", ["normal", "none", "wide", "negative"])
def test_fill_histogram_w2(hk, n, weights):
    rng = np.random.default_rng(n + 3)
    edges = np.linspace(0, 1000, 101).astype(np.float32)
    x = rng.exponential(200, n).astype(np.float32) - 20
    if n > 50:
        x[:30] = edges[:30]
        x[30:40] = np.nan
    w = None
    if weights == "normal":
        w = rng.normal(1, 0.1, n).astype(np.float32)
    elif weights == "wide":
        w = (rng.normal(1, 0.1, n) * 10.0 ** rng.integers(-3, 4, n)).astype(np.float32)
    elif weights == "negative":
        w = (rng.normal(1, 0.1, n) * rng.choice([-1.0, 1.0], n, p=[0.2, 0.8])).astype(np.float32)
    base_sw = rng.uniform(0, 5, 102).astype(np.float32)
    base_ct = rng.integers(0, 9, 102).astype(np.int64)
    rs, r2, rc = hepo.fill_histogram_w2(x, w, edges, sumw=base_sw.copy(), sumw2=base_sw.copy(), counts=base_ct.copy())
    gs, g2, gc = hk.fill_histogram_w2(cu(x), cu(w), cu(edges), sumw=cu(base_sw), sumw2=cu(base_sw), counts=cu(base_ct))
    assert_exact(to_np(gc), rc, "counts (accumulate)")
    assert_tol(to_np(g2), r2, "sumw2")
    if weights == "negative":
        ra, _, _ = hepo.fill_histogram_w2(x, np.abs(w), edges)
        err = np.abs(to_np(gs).astype(np.float64) - rs)
        assert (err <= 1e-5 * (np.abs(ra) + base_sw) + 1e-6).all()
    else:
        assert_tol(to_np(gs), rs, "sumw")
    # any subset of the outputs
    _, o2, _ = hk.fill_histogram_w2(cu(x), cu(w), cu(edges), want=("sumw2",))
    assert_tol(to_np(o2), hepo.fill_histogram_w2(x, w, edges)[1], "sumw2 alone")


def test_fill_histogram_w2_one_hot_bin_does_not_overflow(hk):
    """4 M entries of weight ~1 in ONE bin: fixed-point bins must be moved out before they leave the int32 range."""
    n = 4_000_000
    rng = np.random.default_rng(1)
    x = np.full(n, 55.5, np.float32)
    w = rng.normal(1, 0.05, n).astype(np.float32)
    edges = np.linspace(0, 100, 11).astype(np.float32)
    rs, r2, rc = hepo.fill_histogram_w2(x, w, edges)
    gs, g2, gc = hk.fill_histogram_w2(cu(x), cu(w), cu(edges))
    assert_exact(to_np(gc), rc)
    assert_tol(to_np(gs), rs, "sumw")
    assert_tol(to_np(g2), r2, "sumw2")


@pytest.mark.parametrize("n,nx,ny", [(0, 5, 4), (1000, 5, 4), (2_000_003, 20, 30), (500_001, 90, 90)])
def test_fill_histogram_2d_w2(hk, n, nx, ny):
    rng = np.random.default_rng(n + nx)
    ex = np.linspace(-2.5, 2.5, nx + 1).astype(np.float32)
    ey = np.geomspace(20, 600, ny + 1).astype(np.float32)
    x = rng.uniform(-2.7, 2.7, n).astype(np.float32)
    y = (20 + rng.exponential(60, n)).astype(np.float32) - 3
    w = rng.normal(1, 0.1, n).astype(np.float32)
    rs, r2, rc = hepo.fill_histogram_2d_w2(x, y, w, ex, ey)
    gs, g2, gc = hk.fill_histogram_2d_w2(cu(x), cu(y), cu(w), cu(ex), cu(ey))
    assert_exact(to_np(gc), rc)
    assert_tol(to_np(gs), rs, "sumw")
    assert_tol(to_np(g2), r2, "sumw2")
    s0, _, c0 = hk.fill_histogram_2d_w2(cu(x), cu(y), None, cu(ex), cu(ey), want=("sumw", "counts"))
    assert_exact(to_np(s0), to_np(c0).astype(np.float32), "unit weights: sumw == counts")


def test_fill_histogram_2d_w2_too_large_is_refused(hk):
    ex = torch.linspace(0, 1, 121, device="cuda"); ey = torch.linspace(0, 1, 121, device="cuda")
    x = torch.rand(100, device="cuda")
    with pytest.raises(hk.HepkError, match="shared memory"):
        hk.fill_histogram_2d_w2(x, x, None, ex, ey)
