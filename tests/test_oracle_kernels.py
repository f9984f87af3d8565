"""Pins of the CPU oracle's single kernels against things other than itself:
hand-worked values (tests/golden/), closed forms, invariants, numpy library routines and brute force.
CPU only."""
import math
import os

import numpy as np
import pytest

import hepgen
from oracle import hepo

GOLDEN = os.path.join(os.path.dirname(__file__), "golden")
PI_F = np.float32(3.14159274101257324)


def _read_golden(name):
    out = {}
    with open(os.path.join(GOLDEN, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            key, *vals = line.split()
            out[key] = [float(v) for v in vals]
    return out


# --------------------------------------------------------------------------- c1 select_mask
def test_select_mask_strict_and_f32_constants():
    # 2.4f = 0x4019999A; |eta| == 2.4f exactly must fail (strict <); pt == 30 must fail (strict >)
    eta24 = np.float32(2.4)
    assert eta24.view(np.uint32) == 0x4019999A
    below = np.nextafter(eta24, np.float32(0))
    pt = np.array([30.0, np.nextafter(np.float32(30), np.float32(31)), 100, 100, 100, 100, np.nan, 100], np.float32)
    eta = np.array([0, 0, eta24, -eta24, below, -below, 0, np.nan], np.float32)
    m = hepo.select_mask(pt, eta, 30.0, 2.4)
    assert m.tolist() == [0, 1, 0, 0, 1, 1, 0, 0]


def test_select_mask_brute_force_and_limits():
    rng = np.random.default_rng(1)
    pt = (20 + rng.exponential(30, 5000)).astype(np.float32)
    eta = rng.uniform(-2.5, 2.5, 5000).astype(np.float32)
    m = hepo.select_mask(pt, eta, 30.0, 2.4)
    expect = [1 if (p > np.float32(30.0) and abs(e) < np.float32(2.4)) else 0 for p, e in zip(pt, eta)]
    assert m.tolist() == expect
    assert m.sum() <= pt.size
    assert hepo.select_mask(pt, eta, -np.inf, np.inf).all()          # all finite -> all ones
    assert (hepo.select_mask(pt, None, 30.0, 0.0) == (pt > 30)).all()  # eta NULL drops the eta term


# --------------------------------------------------------------------------- c2 segmented reductions
def test_listing1_golden():
    g = _read_golden("listing1_tiny_events.txt")
    off = np.array(g["offsets"], np.int64)
    pt = np.array(g["pt"], np.float32)
    mc = np.array(g["mask_content"], np.uint8)
    mr = np.array(g["mask_rows"], np.uint8)
    for op in ("sum", "count", "max", "min", "argmax"):
        got = hepo.segmented_reduce(op, pt, off, mr, mc)
        np.testing.assert_array_equal(got.astype(np.float64), np.array(g[f"{op}_masked"]), err_msg=op)
        got = hepo.segmented_reduce(op, pt, off)
        np.testing.assert_array_equal(got.astype(np.float64), np.array(g[f"{op}_all"]), err_msg=op)


def _random_jagged(rng, n_events, lam=5, p_empty_tail=True):
    counts = rng.poisson(lam, n_events)
    if p_empty_tail:
        counts[-3:] = 0          # trailing empty rows (np.add.reduceat breaks there; the oracle must not)
    off = np.zeros(n_events + 1, np.int64)
    off[1:] = np.cumsum(counts)
    return off, int(off[-1])


def test_segmented_invariants_and_numpy():
    rng = np.random.default_rng(2)
    off, m = _random_jagged(rng, 3000)
    data = (20 + rng.exponential(30, m)).astype(np.float32)
    mask = (rng.random(m) < 0.7).astype(np.uint8)
    rows = (rng.random(3000) < 0.9).astype(np.uint8)
    n_per = np.diff(off)

    # count with all-true masks == offsets diff (north_star invariant)
    np.testing.assert_array_equal(hepo.segmented_reduce("count", data, off), n_per)
    s_all = hepo.segmented_reduce("sum", data, off)
    s_msk = hepo.segmented_reduce("sum", data, off, None, mask)
    assert (s_msk <= s_all).all()                                   # masked sum <= unmasked sum (data >= 0)
    # np.add.reduceat on non-empty rows only
    ne = n_per > 0
    ra = np.add.reduceat((data.astype(np.float64) * mask), off[:-1][ne])
    # reduceat spans to the next listed index, which is the next non-empty row start: correct here
    np.testing.assert_allclose(s_msk[ne], ra.astype(np.float32), rtol=1e-6)
    assert (s_msk[~ne] == 0).all()
    # total of per-event sums == masked total
    assert math.isclose(s_msk.astype(np.float64).sum(), (data.astype(np.float64) * mask).sum(), rel_tol=1e-6)

    mx = hepo.segmented_reduce("max", data, off, rows, mask)
    mn = hepo.segmented_reduce("min", data, off, rows, mask)
    ct = hepo.segmented_reduce("count", data, off, rows, mask)
    am = hepo.segmented_reduce("argmax", data, off, rows, mask)
    nz = ct > 0
    assert (mx[nz] >= mn[nz]).all()
    assert np.isneginf(mx[~nz]).all() and np.isposinf(mn[~nz]).all() and (am[~nz] == -1).all()
    assert (ct[rows == 0] == 0).all()
    # data[offsets[e] + argmax] == max bitwise, and it is selected
    g = off[:-1][nz] + am[nz]
    np.testing.assert_array_equal(data[g], mx[nz])
    assert mask[g].all()
    # brute force per event
    for e in range(0, 3000, 37):
        sel = [i for i in range(off[e], off[e + 1]) if mask[i]] if rows[e] else []
        assert ct[e] == len(sel)
        if sel:
            vals = data[sel]
            assert mx[e] == vals.max() and mn[e] == vals.min()
            assert am[e] == sel[int(np.argmax(vals))] - off[e]     # np.argmax returns the first maximum


def test_argmax_first_index_tie_rule_and_nan():
    off = np.array([0, 4, 8, 10], np.int64)
    data = np.array([7, 7, 7, 7, 1, 9, 9, 2, np.nan, 3], np.float32)
    np.testing.assert_array_equal(hepo.segmented_reduce("argmax", data, off), [0, 1, 1])
    mask = np.array([0, 0, 1, 1, 1, 0, 1, 1, 1, 1], np.uint8)
    np.testing.assert_array_equal(hepo.segmented_reduce("argmax", data, off, None, mask), [2, 2, 1])
    np.testing.assert_array_equal(hepo.segmented_reduce("max", data, off), [7, 9, 3])     # NaN skipped
    np.testing.assert_array_equal(hepo.segmented_reduce("min", data, off), [7, 1, 3])
    assert np.isnan(hepo.segmented_reduce("sum", data, off)[2])                            # sum propagates NaN


def test_segmented_content_base():
    rng = np.random.default_rng(3)
    off, m = _random_jagged(rng, 500)
    data = rng.normal(0, 1, m).astype(np.float32)
    e0 = 123
    base = int(off[e0])
    for op in ("sum", "max", "min", "count", "argmax"):
        whole = hepo.segmented_reduce(op, data, off)
        part = hepo.segmented_reduce(op, data[base:], off[e0:], content_base=base)
        np.testing.assert_array_equal(whole[e0:], part)


def test_sum_is_float64_accumulated():
    # 1 + 2^-24 * k pattern: a float32 running sum would lose the small terms, float64 keeps them
    data = np.array([1.0] + [2.0 ** -24] * 4096, np.float32)
    off = np.array([0, data.size], np.int64)
    got = hepo.segmented_reduce("sum", data, off)[0]
    assert got == np.float32(1.0 + 4096 * 2.0 ** -24)


# --------------------------------------------------------------------------- c3 deltar_mask
def _dr2_f64(e1, p1, e2, p2):
    dphi = (float(p1) - float(p2) + math.pi) % (2 * math.pi) - math.pi
    return (float(e1) - float(e2)) ** 2 + dphi ** 2


def test_deltar_special_cases():
    off1 = np.array([0, 1], np.int64)
    off2 = np.array([0, 1], np.int64)
    one = lambda a: np.array([a], np.float32)
    # same (eta, phi) -> matched for any dr_max > 0
    assert hepo.deltar_mask(one(1.2), one(-0.7), off1, None, one(1.2), one(-0.7), off2, None, 1e-3)[0] == 1
    # dr_max = 0 -> none matched (strict <)
    assert hepo.deltar_mask(one(1.2), one(-0.7), off1, None, one(1.2), one(-0.7), off2, None, 0.0)[0] == 0
    # phi wrap: +3.1 vs -3.1 -> raw dphi 6.2, wrapped -0.083 -> matched at 0.4
    assert hepo.deltar_mask(one(0), one(3.1), off1, None, one(0), one(-3.1), off2, None, 0.4)[0] == 1
    assert hepo.deltar_mask(one(0), one(-3.1), off1, None, one(0), one(3.1), off2, None, 0.4)[0] == 1
    # without the wrap the same pair is 6.2 apart: check it is NOT matched at 0.05 but is at 0.1
    assert hepo.deltar_mask(one(0), one(3.1), off1, None, one(0), one(-3.1), off2, None, 0.05)[0] == 0
    assert hepo.deltar_mask(one(0), one(3.1), off1, None, one(0), one(-3.1), off2, None, 0.1)[0] == 1
    # deta alone: 0.39 matched, 0.41 not
    assert hepo.deltar_mask(one(0.39), one(0), off1, None, one(0), one(0), off2, None, 0.4)[0] == 1
    assert hepo.deltar_mask(one(0.41), one(0), off1, None, one(0), one(0), off2, None, 0.4)[0] == 0
    # empty collection 2 -> zero; unselected objects -> zero / ignored
    assert hepo.deltar_mask(one(0), one(0), off1, None, np.zeros(0, np.float32), np.zeros(0, np.float32),
                            np.array([0, 0], np.int64), None, 0.4)[0] == 0
    assert hepo.deltar_mask(one(0), one(0), off1, np.array([0], np.uint8), one(0), one(0), off2, None, 0.4)[0] == 0
    assert hepo.deltar_mask(one(0), one(0), off1, None, one(0), one(0), off2, np.array([0], np.uint8), 0.4)[0] == 0


def test_deltar_threshold_is_float32_product():
    # thr = 0.4f*0.4f = 0.1600000113..., not float32(0.16) = 0.1599999964...: a pair with dr2 == float32(0.16)
    # exactly must be matched.  deta^2 with deta = 0.4f is exactly the threshold -> NOT matched (strict).
    off = np.array([0, 1], np.int64)
    d = np.float32(0.4)
    z = np.zeros(1, np.float32)
    assert hepo.deltar_mask(np.array([d]), z, off, None, z, z, off, None, 0.4)[0] == 0
    dm = np.nextafter(d, np.float32(0))
    assert hepo.deltar_mask(np.array([dm]), z, off, None, z, z, off, None, 0.4)[0] == 1


def test_deltar_brute_force_same_event_only_and_symmetry():
    wl = hepgen.generate(0, n_events=4000, seed=11)
    j, mu = wl.jets, wl.muons
    rng = np.random.default_rng(5)
    selj = (rng.random(j.n_objects) < 0.8).astype(np.uint8)
    selm = (rng.random(mu.n_objects) < 0.8).astype(np.uint8)
    got = hepo.deltar_mask(j.eta, j.phi, j.offsets, selj, mu.eta, mu.phi, mu.offsets, selm, 0.4)
    thr64 = float(np.float32(0.4) * np.float32(0.4))
    n_checked = n_close = 0
    pairs_fwd = set()
    for e in range(wl.n_events):
        for a in range(j.offsets[e], j.offsets[e + 1]):
            want, near = 0, False
            for b in range(mu.offsets[e], mu.offsets[e + 1]):
                if not (selj[a] and selm[b]):
                    continue
                d2 = _dr2_f64(j.eta[a], j.phi[a], mu.eta[b], mu.phi[b])
                assert d2 >= 0
                if abs(d2 - thr64) < 1e-5:
                    near = True
                if d2 < thr64:
                    want = 1
                    pairs_fwd.add((e, a - j.offsets[e], b - mu.offsets[e]))
            if near:
                n_close += 1
                continue           # float64 vs float32 may differ within ~1e-7 of the threshold
            assert got[a] == want, (e, a)
            n_checked += 1
    assert n_checked > 15000 and n_close < 5 and got.sum() > 50
    # symmetry: swapping the collections and OR-reducing matches the same set of events/objects
    rev = hepo.deltar_mask(mu.eta, mu.phi, mu.offsets, selm, j.eta, j.phi, j.offsets, selj, 0.4)
    ev_j = np.repeat(np.arange(wl.n_events), np.diff(j.offsets))
    ev_m = np.repeat(np.arange(wl.n_events), np.diff(mu.offsets))
    assert set(ev_j[got == 1]) == set(ev_m[rev == 1])
    assert set(ev_j[got == 1]) == {p[0] for p in pairs_fwd}


# --------------------------------------------------------------------------- c4 pair_invmass
def _mass(pt, eta, phi, m):
    off = np.array([0, len(pt)], np.int64)
    return hepo.pair_invmass(np.array(pt, np.float32), np.array(eta, np.float32), np.array(phi, np.float32),
                             np.array(m, np.float32), off)


def test_pair_mass_closed_forms():
    # back-to-back massless equal-pt pair: M = 2 pt cosh(deta/2)  (north_star closed form)
    pt, deta = 50.0, 1.3
    phi1 = np.float32(0.3)
    phi2 = np.float32(float(phi1) - math.pi)
    m, i1, i2 = _mass([pt, pt], [0.2 + deta, 0.2], [phi1, phi2], [0, 0])
    assert (i1[0], i2[0]) == (0, 1)
    # float32 inputs: use the same rounded values in the closed form
    de = float(np.float32(0.2 + deta)) - float(np.float32(0.2))
    dphi = float(phi1) - float(phi2)
    expect = math.sqrt(2 * pt * pt * (math.cosh(de) - math.cos(dphi)))
    assert math.isclose(m[0], expect, rel_tol=2e-7)
    assert math.isclose(m[0], 2 * pt * math.cosh(deta / 2), rel_tol=1e-6)
    assert math.isclose(2 * 50 * math.cosh(0.65), 121.87933, rel_tol=1e-7)        # SURVEY.md 8(c4) worked value
    # any massless pair: M^2 = 2 pt1 pt2 (cosh deta - cos dphi)
    m, _, _ = _mass([80, 45], [1.0, -0.5], [0.4, 2.0], [0, 0])
    e1, e2 = float(np.float32(1.0)), float(np.float32(-0.5))
    p1, p2 = float(np.float32(0.4)), float(np.float32(2.0))
    assert math.isclose(m[0], math.sqrt(2 * 80 * 45 * (math.cosh(e1 - e2) - math.cos(p1 - p2))), rel_tol=2e-7)
    # two identical four-vectors: M = 2 m
    m, _, _ = _mass([60, 60], [0.7, 0.7], [1.1, 1.1], [12.5, 12.5])
    assert math.isclose(m[0], 25.0, rel_tol=1e-6)
    # eta = 0, dphi = pi, equal pt and mass: M = 2 sqrt(pt^2 + m^2)
    m, _, _ = _mass([40, 40], [0, 0], [0.0, np.float32(math.pi)], [9, 9])
    assert math.isclose(m[0], 2 * math.sqrt(40 ** 2 + 9 ** 2), rel_tol=1e-6)
    # a single massive particle pair at rest relative to each other in eta, collinear: M = m1 + m2 when
    # both have equal velocity; here equal pt/m ratio -> M = m1 + m2
    m, _, _ = _mass([30, 60], [0.3, 0.3], [-1.0, -1.0], [5, 10])
    assert math.isclose(m[0], 15.0, rel_tol=1e-6)


def test_pair_mass_invariances_and_ordering():
    rng = np.random.default_rng(7)
    wl = hepgen.generate(0, n_events=2000, seed=3)
    j = wl.jets
    mask = (rng.random(j.n_objects) < 0.7).astype(np.uint8)
    m, i1, i2 = hepo.pair_invmass(j.pt, j.eta, j.phi, j.mass, j.offsets, mask)
    # common phi rotation (stay inside float range; tolerance covers input re-rounding)
    m_rot, _, _ = hepo.pair_invmass(j.pt, j.eta, (j.phi + np.float32(0.25)), j.mass, j.offsets, mask)
    np.testing.assert_allclose(m_rot, m, rtol=2e-5, atol=1e-4)
    # reversing the order of particles inside every event leaves the mass unchanged (swap symmetry + top-2 by value)
    idx = np.concatenate([np.arange(j.offsets[e + 1] - 1, j.offsets[e] - 1, -1) for e in range(wl.n_events)]).astype(np.int64)
    m_rev, r1, r2 = hepo.pair_invmass(j.pt[idx], j.eta[idx], j.phi[idx], j.mass[idx], j.offsets, mask[idx])
    np.testing.assert_allclose(m_rev, m, rtol=1e-6, atol=1e-6)
    # ordering: pt[i1] >= pt[i2] >= every other selected pt; fewer than two selected -> 0 and -1
    cnt = hepo.segmented_reduce("count", j.pt, j.offsets, None, mask)
    am = hepo.segmented_reduce("argmax", j.pt, j.offsets, None, mask)
    np.testing.assert_array_equal(i1, am)                            # i1 is the c2 argmax
    for e in range(wl.n_events):
        sel = [k for k in range(j.offsets[e + 1] - j.offsets[e]) if mask[j.offsets[e] + k]]
        if cnt[e] < 2:
            assert m[e] == 0 and i2[e] == -1
            assert i1[e] == (sel[0] if sel else -1)
            continue
        p = j.pt[j.offsets[e]:j.offsets[e + 1]]
        others = [p[k] for k in sel if k not in (i1[e], i2[e])]
        assert p[i1[e]] >= p[i2[e]] and all(p[i2[e]] >= o for o in others)
        assert m[e] >= j.mass[j.offsets[e] + i1[e]] + j.mass[j.offsets[e] + i2[e]] - 1e-3   # M >= m1 + m2


def test_pair_mass_top2_ties():
    # equal values: lower index leads, next one is subleading
    m, i1, i2 = _mass([40, 70, 70, 70], [0, 0.5, -0.5, 1.0], [0, 1, 2, 3], [1, 2, 3, 4])
    assert (i1[0], i2[0]) == (1, 2)
    m, i1, i2 = _mass([70, 40, 70], [0, 0.5, -0.5], [0, 1, 2], [1, 2, 3])
    assert (i1[0], i2[0]) == (0, 2)


# --------------------------------------------------------------------------- c5 lookup_binned
def test_lookup_bin_finder_vs_searchsorted():
    rng = np.random.default_rng(9)
    cal = hepgen.calibration_table(rng)
    pe, ee = cal["pt_edges"], cal["eta_edges"]
    nx, ny = pe.size - 1, ee.size - 1
    x = np.concatenate([(20 + rng.exponential(300, 20000)).astype(np.float32), pe, [np.float32(5), np.float32(1e5), np.float32(np.nan)]]).astype(np.float32)
    y = np.concatenate([rng.uniform(-2.6, 2.6, 20000).astype(np.float32), ee, np.float32([0, 0, 0])])[: x.size].astype(np.float32)
    y = np.resize(y, x.size).astype(np.float32)
    # table T[i][j] = i*ny + j returns the flat bin id (checks row-major indexing order)
    T = np.arange(nx * ny, dtype=np.float32).reshape(nx, ny)
    got = hepo.lookup_binned(x, y, pe, ee, T)
    bx = np.clip(np.searchsorted(pe, x, side="right") - 1, 0, nx - 1)     # NaN sorts last -> clipped to nx-1
    by = np.clip(np.searchsorted(ee, y, side="right") - 1, 0, ny - 1)
    np.testing.assert_array_equal(got, (bx * ny + by).astype(np.float32))
    # a constant table returns the constant; 1-D form
    assert (hepo.lookup_binned(x, y, pe, ee, np.full((nx, ny), 1.25, np.float32)) == np.float32(1.25)).all()
    got1 = hepo.lookup_binned(x, None, pe, None, np.arange(nx, dtype=np.float32))
    np.testing.assert_array_equal(got1, bx.astype(np.float32))
    # value exactly on an interior edge goes to the upper bin; last edge clamps to the last bin
    assert hepo.lookup_binned(pe[3:4], None, pe, None, np.arange(nx, dtype=np.float32))[0] == 3
    assert hepo.lookup_binned(pe[-1:], None, pe, None, np.arange(nx, dtype=np.float32))[0] == nx - 1


# --------------------------------------------------------------------------- c6 fill_histogram
def test_fill_histogram_vs_numpy():
    rng = np.random.default_rng(10)
    edges = hepgen.hist_axes(["ht"])["ht"]
    nb = edges.size - 1
    x = np.concatenate([rng.exponential(250, 50000) - 20, edges.astype(np.float64), [np.nan, np.inf, -np.inf]]).astype(np.float32)
    w = rng.normal(1, 0.1, x.size).astype(np.float32)
    sumw, counts = hepo.fill_histogram(x, w, edges)
    # layout identity with searchsorted/bincount (NaN sorts past the last edge -> overflow)
    slot = np.searchsorted(edges, x, side="right")
    np.testing.assert_array_equal(counts, np.bincount(slot, minlength=nb + 2))
    np.testing.assert_allclose(sumw, np.bincount(slot, weights=w.astype(np.float64), minlength=nb + 2), rtol=1e-6)
    # totals: sum of all slots == sum of weights / n (north_star invariant)
    assert counts.sum() == x.size
    assert math.isclose(sumw.astype(np.float64).sum(), w.astype(np.float64).sum(), rel_tol=1e-6)
    # interior bins == np.histogram except x == last edge (numpy closes the last bin; ours -> overflow)
    fin = np.isfinite(x)
    h = np.histogram(x[fin], edges)[0]
    n_last = int((x == edges[-1]).sum())
    assert n_last == 1
    h[-1] -= n_last
    np.testing.assert_array_equal(counts[1:-1], h)
    assert counts[-1] == (x[fin] >= edges[-1]).sum() + 2                # +2: the NaN and +inf entries
    assert counts[0] == (x[fin] < edges[0]).sum() + 1                   # +1: the -inf entry
    # weights NULL => sumw == counts
    s1, c1 = hepo.fill_histogram(x, None, edges)
    np.testing.assert_array_equal(s1, c1.astype(np.float32))
    # filling in two calls == one call on the concatenation (accumulating in/out arrays)
    sa, ca = hepo.fill_histogram(x[:20000], w[:20000], edges)
    sa, ca = hepo.fill_histogram(x[20000:], w[20000:], edges, sa, ca)
    np.testing.assert_array_equal(ca, counts)
    np.testing.assert_allclose(sa, sumw, rtol=1e-6)


def test_fill_histogram_nonuniform_edges_brute_force():
    rng = np.random.default_rng(12)
    edges = np.sort(rng.uniform(0, 10, 18)).astype(np.float32)
    x = np.concatenate([rng.uniform(-1, 11, 3000).astype(np.float32), edges])
    _, counts = hepo.fill_histogram(x, None, edges)
    nb = edges.size - 1
    want = np.zeros(nb + 2, np.int64)
    for v in x:
        if v < edges[0]:
            want[0] += 1
        elif v >= edges[nb]:
            want[nb + 1] += 1
        else:
            b = max(k for k in range(nb) if edges[k] <= v)
            want[1 + b] += 1
    np.testing.assert_array_equal(counts, want)


def test_invalid_arguments_return_error():
    with pytest.raises(ValueError):
        hepo.fill_histogram(np.zeros(3, np.float32), None, np.zeros(1, np.float32))     # nbins = 0
