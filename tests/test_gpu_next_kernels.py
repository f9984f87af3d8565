"""Parity of the SURVEY.md 8(f-1) CUDA kernels (hepk_get_in_offsets, hepk_set_in_offsets, hepk_select_opposite_sign,
through the C ABI) against the CPU oracle on the same seeded inputs.  All three are exact class: bit-exact."""
import numpy as np
import pytest
import torch

import hepgen
from oracle import hepo
from _util import assert_exact, to_np

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def hk():
    from paper_1906_06242_b200 import binding
    binding.lib()
    return binding


def cu(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def charges(rng, m):
    q = rng.choice([-1, 1], m).astype(np.int32)
    q[rng.random(m) < 0.01] = 0
    return q


@pytest.mark.parametrize("config,n", [(0, None), (2, 300_011)])
def test_get_and_set_in_offsets(hk, config, n):
    wl = hepgen.generate(config, n_events=n)
    rng = np.random.default_rng(7)
    j = wl.jets
    N, M = wl.n_events, j.pt.size
    mc = (rng.random(M) < 0.7).astype(np.uint8)
    mr = (rng.random(N) < 0.85).astype(np.uint8)
    vals = rng.normal(size=N).astype(np.float32)
    d_pt, d_off, d_mc, d_mr = cu(j.pt), cu(j.offsets), cu(mc), cu(mr)
    for index in (0, 1, 5, 39, 200):
        for rows, cont in ((None, None), (mr, mc)):
            want = hepo.get_in_offsets(j.pt, j.offsets, index, rows, cont, fill=-1.5)
            got = hk.get_in_offsets(d_pt, d_off, index, None if rows is None else d_mr, None if cont is None else d_mc, fill=-1.5)
            assert_exact(to_np(got), want, f"get index={index} masks={rows is not None}")
            want = hepo.set_in_offsets(j.pt, j.offsets, index, values=vals, mask_rows=rows, mask_content=cont)
            buf = d_pt.clone()
            hk.set_in_offsets(buf, d_off, index, values=cu(vals), mask_rows=None if rows is None else d_mr,
                              mask_content=None if cont is None else d_mc)
            assert_exact(to_np(buf), want, f"set index={index}")
    want = hepo.set_in_offsets(j.pt, j.offsets, 0, value=3.25)
    buf = d_pt.clone()
    hk.set_in_offsets(buf, d_off, 0, value=3.25)
    assert_exact(to_np(buf), want, "set scalar")
    torch.cuda.synchronize()


def test_get_in_offsets_content_base_and_edges(hk):
    wl = hepgen.generate(2, n_events=5_000, seed=3)
    j = wl.jets
    e0, e1 = 1_000, 4_321
    g0, g1 = int(j.offsets[e0]), int(j.offsets[e1])
    want = hepo.get_in_offsets(j.pt[g0:g1], j.offsets[e0:e1 + 1], 2, fill=0.0, content_base=g0)
    got = hk.get_in_offsets(cu(j.pt[g0:g1]), cu(j.offsets[e0:e1 + 1]), 2, fill=0.0, content_base=g0)
    assert_exact(to_np(got), want)
    assert_exact(want, hepo.get_in_offsets(j.pt, j.offsets, 2, fill=0.0)[e0:e1])
    empty = np.zeros(1, np.int64)                               # no events at all
    assert hk.get_in_offsets(cu(np.zeros(0, np.float32)), cu(empty), 0).numel() == 0
    off = np.zeros(101, np.int64)                               # 100 empty events
    got = hk.get_in_offsets(cu(np.zeros(0, np.float32)), cu(off), 0, fill=9.0)
    assert (to_np(got) == 9.0).all()
    with pytest.raises(hk.HepkError):
        hk.get_in_offsets(cu(j.pt), cu(j.offsets), -1)


@pytest.mark.parametrize("config,n", [(0, None), (2, 400_003)])
def test_select_opposite_sign(hk, config, n):
    wl = hepgen.generate(config, n_events=n)
    rng = np.random.default_rng(8)
    m = wl.muons
    N, M = wl.n_events, m.pt.size
    pt = m.pt.copy()
    pt[rng.random(M) < 0.1] = np.float32(33.0)                  # ties
    pt[rng.random(M) < 0.001] = np.float32(np.nan)
    q = charges(rng, M)
    mc = (rng.random(M) < 0.8).astype(np.uint8)
    mr = (rng.random(N) < 0.9).astype(np.uint8)
    for rows, cont in ((None, None), (mr, mc)):
        want = hepo.select_opposite_sign(pt, q, m.offsets, rows, cont)
        got = hk.select_opposite_sign(cu(pt), cu(q), cu(m.offsets), None if rows is None else cu(rows),
                                      None if cont is None else cu(cont))
        assert_exact(to_np(got), want)
        per = np.add.reduceat(np.concatenate([want, [0]]).astype(np.int64), m.offsets[:-1])[:N]
        per = np.where(np.diff(m.offsets) > 0, per, 0)
        assert set(np.unique(per)) <= {0, 2}
    # the same on the jets of config 2 (long rows, 30-40 objects)
    j = wl.jets
    qj = charges(rng, j.pt.size)
    assert_exact(to_np(hk.select_opposite_sign(cu(j.pt), cu(qj), cu(j.offsets))), hepo.select_opposite_sign(j.pt, qj, j.offsets))


def test_lookup_interp(hk):
    from _util import assert_tol
    wl = hepgen.generate(2, n_events=200_003)
    rng = np.random.default_rng(9)
    xs = np.sort(rng.uniform(20, 600, 30)).astype(np.float32)
    ys = rng.uniform(0.9, 1.1, 30).astype(np.float32)
    x = wl.jets.pt.copy()
    x[:40] = np.resize(xs, 40)                               # exactly on knots
    x[40:44] = [np.nan, -np.inf, np.inf, 0.0]
    want = hepo.lookup_interp(x, xs, ys)
    got = to_np(hk.lookup_interp(cu(x), cu(xs), cu(ys)))
    assert_tol(got, want, "lookup_interp")
    assert_exact(got[:40], want[:40], "knots are exact")
    two = hk.lookup_interp(cu(x), cu(xs[:2]), cu(ys[:2]))    # the smallest table
    assert_tol(to_np(two), hepo.lookup_interp(x, xs[:2], ys[:2]))
    with pytest.raises(hk.HepkError):
        hk.lookup_interp(cu(x), cu(xs[:1]), cu(ys[:1]))


@pytest.mark.parametrize("n", [0, 1, 1000, 1_000_003])
def test_fill_histogram_2d(hk, n):
    from _util import assert_tol
    rng = np.random.default_rng(10)
    x = rng.normal(0, 1.5, n).astype(np.float32)
    y = (20 + rng.exponential(30, n)).astype(np.float32)
    if n > 10:
        x[:3] = np.nan
        y[3:6] = [np.inf, -np.inf, 500.0]
        x[6], y[6] = np.float32(2.5), np.float32(20.0)       # on the last x edge -> x overflow
    w = rng.normal(1, 0.1, n).astype(np.float32)
    ex = np.linspace(-2.5, 2.5, 21).astype(np.float32)
    ey = np.geomspace(20, 500, 31).astype(np.float32)         # non-uniform axis
    for weights in (w, None):
        sw_ref, ct_ref = hepo.fill_histogram_2d(x, y, weights, ex, ey)
        sw, ct = hk.fill_histogram_2d(cu(x), cu(y), None if weights is None else cu(w), cu(ex), cu(ey))
        assert_exact(to_np(ct), ct_ref, "2d counts")
        assert_tol(to_np(sw), sw_ref, "2d sumw")
        hk.fill_histogram_2d(cu(x), cu(y), None if weights is None else cu(w), cu(ex), cu(ey), sumw=sw, counts=ct)   # accumulates
        assert_exact(to_np(ct), 2 * ct_ref)
        assert_tol(to_np(sw), 2.0 * sw_ref.astype(np.float64))
    _, only = hk.fill_histogram_2d(cu(x), cu(y), None, cu(ex), cu(ey), want_sumw=False)
    assert_exact(to_np(only), hepo.fill_histogram_2d(x, y, None, ex, ey)[1])


def _triplet_check(got_m, got_i, ref_m, ref_i, pt, eta, phi, mass, off, sel, target):
    """Tolerance-class comparison of an argmin: the distance reached must equal the oracle's within tolerance, the
    returned triplet must be a valid one whose float64 mass is the returned mass; indices equal except at near-ties."""
    n = off.size - 1
    p, e, f, m = (a.astype(np.float64) for a in (pt, eta, phi, mass))
    vec = np.stack([np.sqrt(p ** 2 * np.cosh(e) ** 2 + m ** 2), p * np.cos(f), p * np.sin(f), p * np.sinh(e)], axis=1)
    none = ref_i[:, 0] < 0
    assert_exact(got_i[none], ref_i[none], "events without a triplet")
    assert (got_m[none] == 0).all()
    ok = ~none
    gi = got_i[ok].astype(np.int64) + off[:-1][ok, None]
    assert (got_i[ok][:, 0] < got_i[ok][:, 1]).all() and (got_i[ok][:, 1] < got_i[ok][:, 2]).all()
    assert (gi < off[1:][ok, None]).all()
    if sel is not None:
        assert sel[gi].all()
    v = vec[gi].sum(axis=1)
    M = np.sqrt(np.maximum(v[:, 0] ** 2 - v[:, 1] ** 2 - v[:, 2] ** 2 - v[:, 3] ** 2, 0.0))
    tol = 1e-5 * np.maximum(M, 1.0) + 1e-6
    assert np.all(np.abs(got_m[ok] - M) <= tol), "returned mass is the mass of the returned triplet"
    assert np.all(np.abs(np.abs(M - target) - np.abs(ref_m[ok].astype(np.float64) - target)) <= 2 * tol), "distance reached"
    same = (got_i[ok] == ref_i[ok]).all(axis=1).mean()
    assert same > 0.999, same


@pytest.mark.parametrize("config,n", [(0, None), (2, 200_003)])
def test_triplet_mass(hk, config, n):
    wl = hepgen.generate(config, n_events=n)
    j = wl.jets
    rng = np.random.default_rng(12)
    sel = (j.pt > 30) & (np.abs(j.eta) < 2.4)
    mr = (rng.random(wl.n_events) < 0.9).astype(np.uint8)
    for rows, cont in ((None, None), (mr, sel.astype(np.uint8))):
        ref_m, ref_i = hepo.triplet_mass(j.pt, j.eta, j.phi, j.mass, j.offsets, 172.0, rows, cont)
        got_m, got_i = hk.triplet_mass(cu(j.pt), cu(j.eta), cu(j.phi), cu(j.mass), cu(j.offsets), 172.0,
                                       None if rows is None else cu(rows), None if cont is None else cu(cont))
        _triplet_check(to_np(got_m), to_np(got_i), ref_m, ref_i, j.pt, j.eta, j.phi, j.mass, j.offsets,
                       None if cont is None else cont.astype(bool), 172.0)
        if rows is not None:
            assert (to_np(got_m)[mr == 0] == 0).all()


def test_triplet_mass_long_events(hk):
    """Events larger than the kernel's shared-memory cache (64 selected jets) and exact ties."""
    rng = np.random.default_rng(13)
    counts = np.array([0, 2, 3, 120, 5, 97, 96, 1, 40], np.int64)
    off = np.zeros(counts.size + 1, np.int64)
    off[1:] = np.cumsum(counts)
    m = int(off[-1])
    pt = (20 + rng.exponential(30, m)).astype(np.float32)
    eta = rng.uniform(-2.5, 2.5, m).astype(np.float32)
    phi = rng.uniform(-np.pi, np.pi, m).astype(np.float32)
    mass = rng.exponential(10, m).astype(np.float32)
    pt[off[4]:off[5]] = 45.0; eta[off[4]:off[5]] = 0.3; phi[off[4]:off[5]] = 1.0; mass[off[4]:off[5]] = 4.0   # five identical jets: all triplets tie
    ref_m, ref_i = hepo.triplet_mass(pt, eta, phi, mass, off, 172.0)
    got_m, got_i = hk.triplet_mass(cu(pt), cu(eta), cu(phi), cu(mass), cu(off), 172.0)
    gm, gi = to_np(got_m), to_np(got_i)
    assert list(gi[4]) == [0, 1, 2] and list(ref_i[4]) == [0, 1, 2]             # first triplet wins an exact tie
    _triplet_check(gm, gi, ref_m, ref_i, pt, eta, phi, mass, off, None, 172.0)
    only_m, none = hk.triplet_mass(cu(pt), cu(eta), cu(phi), cu(mass), cu(off), 172.0, want_indices=False)
    assert none is None
    assert_exact(to_np(only_m), gm)


def test_validate_offsets(hk):
    wl = hepgen.generate(2, n_events=300_001)
    off = wl.jets.offsets
    m = wl.jets.pt.size
    assert hk.validate_offsets(cu(off), m) == 0 == hepo.validate_offsets(off, m)
    assert hk.validate_offsets(cu(off), m - 1) == 1
    assert hk.validate_offsets(cu(off + 7), m, content_base=8) == 1
    rng = np.random.default_rng(14)
    broken = off.copy()
    broken[rng.choice(np.arange(1, off.size - 1), 1000, replace=False)] -= 10_000_000
    assert hk.validate_offsets(cu(broken), m) == hepo.validate_offsets(broken, m) > 0
