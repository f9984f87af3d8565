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
