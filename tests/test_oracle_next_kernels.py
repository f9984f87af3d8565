"""Pins of the oracle's SURVEY.md 8(f-1) kernels (get_in_offsets, set_in_offsets, select_opposite_sign) against
what the paper's one-line definitions and plain numpy fix: brute force in Python on
small jagged arrays, library special cases, invariants."""
import numpy as np

from oracle import hepo


def _jagged(rng, n, lam, cap=12):
    counts = np.minimum(rng.poisson(lam, n), cap)
    off = np.zeros(n + 1, np.int64)
    off[1:] = np.cumsum(counts)
    return off


def test_get_in_offsets_brute_force_and_numpy():
    rng = np.random.default_rng(0)
    off = _jagged(rng, 500, 3.0)
    m = int(off[-1])
    data = rng.normal(size=m).astype(np.float32)
    mc = rng.random(m) < 0.7
    mr = rng.random(500) < 0.8
    for index in (0, 1, 4):
        got = hepo.get_in_offsets(data, off, index, fill=-7.0)
        # positional, no masks: numpy fancy indexing where the row is long enough
        want = np.full(500, -7.0, np.float32)
        ok = np.diff(off) > index
        want[ok] = data[off[:-1][ok] + index]
        np.testing.assert_array_equal(got, want)
        got = hepo.get_in_offsets(data, off, index, mask_rows=mr, mask_content=mc, fill=np.float32(99.0))
        for e in range(500):                                   # brute force: index-th selected element of the row
            sel = [i for i in range(off[e], off[e + 1]) if mc[i]]
            exp = data[sel[index]] if (mr[e] and len(sel) > index) else np.float32(99.0)
            assert got[e] == exp, (e, index)
    # index 0 on pt-sorted rows is the row maximum (the paper's "leading jet pT" use)
    srt = data.copy()
    for e in range(500):
        srt[off[e]:off[e + 1]] = np.sort(srt[off[e]:off[e + 1]])[::-1]
    lead = hepo.get_in_offsets(srt, off, 0, fill=-np.inf)
    np.testing.assert_array_equal(lead, hepo.segmented_reduce("max", srt, off))


def test_set_in_offsets_roundtrip_and_untouched():
    rng = np.random.default_rng(1)
    off = _jagged(rng, 400, 2.5)
    m = int(off[-1])
    data = rng.normal(size=m).astype(np.float32)
    vals = rng.normal(size=400).astype(np.float32)
    mc = rng.random(m) < 0.6
    for index in (0, 2):
        new = hepo.set_in_offsets(data, off, index, values=vals, mask_content=mc)
        # what was set is read back by get_in_offsets; rows without that element read the fill
        back = hepo.get_in_offsets(new, off, index, mask_content=mc, fill=np.float32(1e9))
        had = hepo.get_in_offsets(data, off, index, mask_content=mc, fill=np.float32(1e9)) != np.float32(1e9)
        np.testing.assert_array_equal(back[had], vals[had])
        assert (back[~had] == np.float32(1e9)).all()
        # exactly one element per such row changed, nothing else
        changed = new != data
        assert changed.sum() <= had.sum()
        for e in range(400):
            assert changed[off[e]:off[e + 1]].sum() <= 1
    new = hepo.set_in_offsets(data, off, 0, value=5.0, mask_rows=np.zeros(400, bool))
    np.testing.assert_array_equal(new, data)                   # every row masked: untouched
    new = hepo.set_in_offsets(data, off, 0, value=5.0)
    ne = np.diff(off) > 0
    assert (new[off[:-1][ne]] == 5.0).all() and (new != data).sum() <= ne.sum()


def test_select_opposite_sign_brute_force_and_hand_cases():
    # hand cases: (pt, charge) per event
    ev = [
        ([50, 40, 30], [+1, +1, -1]),          # lead 0, partner 2 (40 has the same sign)
        ([10, 60, 20, 60], [-1, +1, -1, -1]),  # lead = first 60 (index 1), partner = second 60 (index 3, opposite, highest)
        ([30, 20], [+1, +1]),                  # no opposite pair
        ([], []),
        ([25], [-1]),
        ([5, 5, 5], [+1, -1, -1]),             # all equal: lead 0, partner = first opposite (index 1)
    ]
    want = [[1, 0, 1], [0, 1, 0, 1], [0, 0], [], [0], [1, 1, 0]]
    pt = np.concatenate([np.asarray(p, np.float32) for p, _ in ev])
    q = np.concatenate([np.asarray(c, np.int32) for _, c in ev])
    off = np.zeros(len(ev) + 1, np.int64)
    off[1:] = np.cumsum([len(p) for p, _ in ev])
    got = hepo.select_opposite_sign(pt, q, off)
    np.testing.assert_array_equal(got, np.concatenate([np.asarray(w, np.uint8) for w in want]))
    # brute force on random events: sort by (-pt, index), first element + first later element of opposite sign
    rng = np.random.default_rng(2)
    off = _jagged(rng, 800, 2.2, cap=8)
    m = int(off[-1])
    pt = (20 + rng.exponential(30, m)).astype(np.float32)
    pt[rng.random(m) < 0.2] = np.float32(45.0)                 # plenty of ties
    q = rng.choice([-1, 1], m).astype(np.int32)
    mc = rng.random(m) < 0.8
    mr = rng.random(800) < 0.9
    got = hepo.select_opposite_sign(pt, q, off, mask_rows=mr, mask_content=mc)
    for e in range(800):
        exp = np.zeros(off[e + 1] - off[e], np.uint8)
        idx = [i for i in range(off[e], off[e + 1]) if mc[i]]
        order = sorted(idx, key=lambda i: (-float(pt[i]), i))
        if mr[e] and order:
            lead = order[0]
            part = next((i for i in order[1:] if q[i] * q[lead] < 0), None)
            if part is not None:
                exp[lead - off[e]] = exp[part - off[e]] = 1
        np.testing.assert_array_equal(got[off[e]:off[e + 1]], exp, err_msg=str(e))
    # invariants: 0 or 2 per event, and the two have opposite signs
    per = np.add.reduceat(np.concatenate([got, [0]]).astype(np.int64), off[:-1])[:800] if m else np.zeros(800)
    per = np.where(np.diff(off) > 0, per, 0)
    assert set(np.unique(per)) <= {0, 2}


def test_lookup_interp_against_numpy_and_closed_forms():
    rng = np.random.default_rng(3)
    xs = np.sort(rng.uniform(20, 3000, 40)).astype(np.float32)
    ys = rng.uniform(0.9, 1.1, 40).astype(np.float32)
    x = np.concatenate([rng.uniform(0, 3500, 20_000), xs, [np.nan, -np.inf, np.inf]]).astype(np.float32)
    got = hepo.lookup_interp(x, xs, ys).astype(np.float64)
    want = np.interp(x.astype(np.float64), xs.astype(np.float64), ys.astype(np.float64))
    fin = ~np.isnan(x)
    assert np.all(np.abs(got[fin] - want[fin]) <= 1e-6 * np.abs(want[fin]))      # float32 rounding of the float64 value
    assert np.isnan(got[~fin]).all()
    np.testing.assert_array_equal(hepo.lookup_interp(xs, xs, ys), ys)             # exact at the knots
    # a straight line is reproduced, and constant extrapolation holds the end values
    line = (2.0 + 0.5 * xs.astype(np.float64)).astype(np.float32)
    mid = (0.5 * (xs[:-1].astype(np.float64) + xs[1:])).astype(np.float32)
    g = hepo.lookup_interp(mid, xs, line).astype(np.float64)
    assert np.all(np.abs(g - (2.0 + 0.5 * mid.astype(np.float64))) <= 2e-6 * np.abs(g))
    assert hepo.lookup_interp(np.float32([1.0]), xs, ys)[0] == ys[0] and hepo.lookup_interp(np.float32([1e9]), xs, ys)[0] == ys[-1]


def test_fill_histogram_2d_against_numpy_and_marginals():
    rng = np.random.default_rng(4)
    n = 50_000
    x = rng.normal(0, 1.5, n).astype(np.float32)
    y = rng.exponential(40, n).astype(np.float32)
    x[:5] = np.nan
    w = rng.normal(1, 0.1, n).astype(np.float32)
    ex = np.linspace(-2.5, 2.5, 21).astype(np.float32)
    ey = np.geomspace(5, 300, 13).astype(np.float32)
    sw, ct = hepo.fill_histogram_2d(x, y, w, ex, ey)
    assert ct.shape == (22, 14) and ct.sum() == n
    assert abs(sw.astype(np.float64).sum() - w.astype(np.float64).sum()) <= 1e-5 * n
    # inner bins == numpy (right-open bins; no entry sits exactly on a last edge here)
    h, _, _ = np.histogram2d(x, y, bins=[ex, ey])
    np.testing.assert_array_equal(ct[1:-1, 1:-1], h.astype(np.int64))
    hw, _, _ = np.histogram2d(x[5:], y[5:], bins=[ex, ey], weights=w[5:].astype(np.float64))
    assert np.all(np.abs(sw[1:-1, 1:-1] - hw) <= 1e-5 * np.abs(hw) + 1e-6)
    # marginals == the one-dimensional histograms of each axis (flow bins included, NaN -> overflow)
    sx, cx = hepo.fill_histogram(x, w, ex)
    sy, cy = hepo.fill_histogram(y, w, ey)
    np.testing.assert_array_equal(ct.sum(axis=1), cx)
    np.testing.assert_array_equal(ct.sum(axis=0), cy)
    assert np.all(np.abs(sw.astype(np.float64).sum(axis=1) - sx) <= 1e-5 * np.abs(sx) + 1e-5)
    assert ct[-1, :].sum() >= 5                                                    # the NaNs went to x overflow
    # two calls == one call on the concatenation
    sw2, ct2 = hepo.fill_histogram_2d(x[: n // 2], y[: n // 2], w[: n // 2], ex, ey)
    hepo.fill_histogram_2d(x[n // 2:], y[n // 2:], w[n // 2:], ex, ey, sumw=sw2, counts=ct2)
    np.testing.assert_array_equal(ct2, ct)
    assert np.all(np.abs(sw2 - sw) <= 1e-5 * np.abs(sw) + 1e-6)


def test_triplet_mass_closed_forms_and_brute_force():
    import itertools
    # closed form: three massless jets at eta = 0, phi = 0, 2pi/3, 4pi/3 with equal pt: total momentum 0, M = 3 pt
    phi = np.float32([0.0, 2 * np.pi / 3, 4 * np.pi / 3 - 2 * np.pi])
    pt = np.float32([50, 50, 50]); z = np.zeros(3, np.float32)
    m, idx = hepo.triplet_mass(pt, z, phi, z, np.int64([0, 3]), 172.0)
    assert abs(m[0] - 150.0) < 1e-3 and list(idx[0]) == [0, 1, 2]
    # three identical four-vectors: M = 3 m
    m, _ = hepo.triplet_mass(np.float32([40] * 3), np.float32([0.7] * 3), np.float32([1.1] * 3), np.float32([5.0] * 3), np.int64([0, 3]), 172.0)
    assert abs(m[0] - 15.0) < 1e-4
    # fewer than three (selected) objects
    m, idx = hepo.triplet_mass(pt, z, phi, z, np.int64([0, 2, 3]), 172.0)
    assert (m == 0).all() and (idx == -1).all()
    m, idx = hepo.triplet_mass(pt, z, phi, z, np.int64([0, 3]), 172.0, mask_content=np.uint8([1, 0, 1]))
    assert m[0] == 0 and (idx == -1).all()
    # brute force with numpy float64 four-vectors on random events
    rng = np.random.default_rng(6)
    off = _jagged(rng, 300, 4.5, cap=9)
    n = int(off[-1])
    pt = (20 + rng.exponential(30, n)).astype(np.float32)
    eta = rng.uniform(-2.5, 2.5, n).astype(np.float32)
    phi = rng.uniform(-np.pi, np.pi, n).astype(np.float32)
    mass = rng.exponential(10, n).astype(np.float32)
    mc = rng.random(n) < 0.8
    got_m, got_i = hepo.triplet_mass(pt, eta, phi, mass, off, 172.0, mask_content=mc)
    p64, e64, f64, m64 = (a.astype(np.float64) for a in (pt, eta, phi, mass))
    vec = np.stack([np.sqrt(p64 ** 2 * np.cosh(e64) ** 2 + m64 ** 2), p64 * np.cos(f64), p64 * np.sin(f64), p64 * np.sinh(e64)], axis=1)
    for e in range(300):
        sel = [i for i in range(off[e], off[e + 1]) if mc[i]]
        if len(sel) < 3:
            assert got_m[e] == 0 and (got_i[e] == -1).all()
            continue
        best = None
        for tri in itertools.combinations(sel, 3):
            v = vec[list(tri)].sum(axis=0)
            M = np.sqrt(max(v[0] ** 2 - v[1] ** 2 - v[2] ** 2 - v[3] ** 2, 0.0))
            if best is None or abs(M - 172.0) < best[0]:
                best = (abs(M - 172.0), M, tri)
        assert abs(got_m[e] - best[1]) <= 1e-5 * best[1] + 1e-6
        assert tuple(got_i[e] + off[e]) == best[2]
    # invariance of the chosen mass under a common phi rotation
    rot = ((phi + np.float32(0.9) + np.pi) % (2 * np.pi) - np.pi).astype(np.float32)
    rm, _ = hepo.triplet_mass(pt, eta, rot, mass, off, 172.0, mask_content=mc)
    assert np.all(np.abs(rm - got_m) <= 2e-4 * np.abs(got_m) + 1e-4)


def test_validate_offsets_against_numpy():
    rng = np.random.default_rng(8)
    off = _jagged(rng, 1000, 3.0)
    m = int(off[-1])
    assert hepo.validate_offsets(off, m) == 0
    assert hepo.validate_offsets(off, m - 1) == 1                       # last offset beyond the columns
    assert hepo.validate_offsets(off + 5, m, content_base=5) == 0
    assert hepo.validate_offsets(off + 5, m, content_base=6) == 1       # first offset before content_base
    broken = off.copy()
    idx = rng.choice(np.arange(1, 1000), 25, replace=False)
    broken[idx] -= 1000
    want = int((np.diff(broken) < 0).sum()) + int(broken[0] < 0) + int(broken[-1] > m)
    assert hepo.validate_offsets(broken, m) == want and want >= 10
