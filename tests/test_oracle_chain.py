"""Pins of the oracle's fused chain: it must equal calling the single-function
oracles in sequence (T4), satisfy the chain invariants, and match a hand-worked tiny event.  CPU only."""
import math

import numpy as np
import pytest

import hepgen
from oracle import hepo


def compose_from_singles(wl):
    """The chain written as a sequence of single-kernel oracle calls (PAPER.md:L129-139 steps)."""
    j, mu, el = wl.jets, wl.muons, wl.electrons
    c = wl.cuts
    N = wl.n_events
    if wl.calib is not None:
        corr = hepo.lookup_binned(j.pt, j.eta, wl.calib["pt_edges"], wl.calib["eta_edges"], wl.calib["table"])
        scales = wl.calib["scales"]
    else:
        corr, scales = None, [None]
    msel = hepo.select_mask(mu.pt, None, c["lep_pt_min"], 0.0)
    esel = hepo.select_mask(el.pt, None, c["lep_pt_min"], 0.0) if el is not None else None
    out = {k: [] for k in ("njet", "argmax", "ht", "maxpt", "minpt", "mjj", "subpt", "jet_mask")}
    hists = {}
    for v, s in enumerate(scales):
        if corr is None:
            ptv = j.pt
        else:
            cv = corr * np.float32(s)              # float32 multiply: table x scale
            ptv = j.pt * cv                        # float32 multiply: applied to pt
            assert ptv.dtype == np.float32
        jsel = hepo.select_mask(ptv, j.eta, c["jet_pt_min"], c["jet_abs_eta_max"])
        matched = hepo.deltar_mask(j.eta, j.phi, j.offsets, jsel, mu.eta, mu.phi, mu.offsets, msel, c["dr_max"])
        if el is not None:
            matched |= hepo.deltar_mask(j.eta, j.phi, j.offsets, jsel, el.eta, el.phi, el.offsets, esel, c["dr_max"])
        clean = (jsel & (1 - matched)).astype(np.uint8)
        njet = hepo.segmented_reduce("count", ptv, j.offsets, None, clean)
        ht = hepo.segmented_reduce("sum", ptv, j.offsets, None, clean)
        maxpt = hepo.segmented_reduce("max", ptv, j.offsets, None, clean)
        minpt = hepo.segmented_reduce("min", ptv, j.offsets, None, clean)
        argmax = hepo.segmented_reduce("argmax", ptv, j.offsets, None, clean)
        mjj, i1, i2 = hepo.pair_invmass(ptv, j.eta, j.phi, j.mass, j.offsets, clean)
        subpt = np.where(i2 >= 0, ptv[np.minimum(j.offsets[:-1] + np.maximum(i2, 0), max(j.n_objects - 1, 0))], np.float32(0)).astype(np.float32) \
            if j.n_objects else np.zeros(N, np.float32)
        np.testing.assert_array_equal(i1, argmax)
        vals = dict(njet=njet, argmax=argmax, ht=ht, maxpt=maxpt, minpt=minpt, mjj=mjj, subpt=subpt, jet_mask=clean)
        for k in out:
            out[k].append(vals[k])
        for name in wl.hists:
            x = vals[name].astype(np.float32)
            for w in range(wl.weights.shape[0]):
                hists[(v, name, w)] = hepo.fill_histogram(x, wl.weights[w], wl.axes[name])
    return {k: np.stack(a) for k, a in out.items()}, hists


def check_chain_equals_composition(wl):
    res = hepo.analysis_chain(wl)
    comp, hists = compose_from_singles(wl)
    for k in ("njet", "argmax", "maxpt", "minpt", "jet_mask", "ht", "mjj", "subpt"):
        np.testing.assert_array_equal(res[k], comp[k], err_msg=k)      # same arithmetic in both -> bitwise
    for name in wl.hists:
        sw, ct = hepo.hist_view(res, name, wl)
        for v in range(sw.shape[0]):
            for w in range(sw.shape[1]):
                s_ref, c_ref = hists[(v, name, w)]
                np.testing.assert_array_equal(ct[v], c_ref, err_msg=f"{name} counts v{v}")
                np.testing.assert_array_equal(sw[v, w], s_ref, err_msg=f"{name} sumw v{v} w{w}")
    return res


@pytest.mark.parametrize("config,n", [(0, 3000), (1, 3000), (2, 3000), (3, 2000), (4, 1500)])
def test_chain_equals_composition_of_single_oracles(config, n):
    wl = hepgen.generate(config, n_events=n)
    res = check_chain_equals_composition(wl)
    j = wl.jets
    V = res["njet"].shape[0]
    # invariants
    assert (res["njet"] <= np.diff(j.offsets)[None, :]).all()
    tot_w = wl.weights.astype(np.float64).sum(axis=1)
    for name in wl.hists:
        sw, ct = hepo.hist_view(res, name, wl)
        assert (ct.sum(axis=1) == wl.n_events).all()                   # every event lands in exactly one slot
        np.testing.assert_allclose(sw.astype(np.float64).sum(axis=2), np.broadcast_to(tot_w, (V, tot_w.size)), rtol=1e-6)
    # events with no clean jets: HT 0 -> first bin, maxpt -inf -> underflow, minpt +inf -> overflow
    empty = res["njet"][0] == 0
    assert empty.any()
    assert (res["ht"][0][empty] == 0).all() and np.isneginf(res["maxpt"][0][empty]).all()
    assert np.isposinf(res["minpt"][0][empty]).all() and (res["argmax"][0][empty] == -1).all()
    assert (res["mjj"][0][res["njet"][0] < 2] == 0).all() and (res["subpt"][0][res["njet"][0] < 2] == 0).all()
    assert (res["mjj"][0][res["njet"][0] >= 2] > 0).all()
    if "maxpt" in wl.hists:
        _, ct = hepo.hist_view(res, "maxpt", wl)
        assert ct[0, 0] == empty.sum()


def test_variant_invariants_config3():
    wl = hepgen.generate(3, n_events=4000)
    res = hepo.analysis_chain(wl)
    sc = wl.calib["scales"].tolist()
    nom, up2, dn2, up5, dn5 = (sc.index(np.float32(x)) for x in (1.0, 1.02, 0.98, 1.05, 0.95))
    nj = res["njet"]
    assert (nj[up5] >= nj[up2]).all() and (nj[up2] >= nj[nom]).all()
    assert (nj[nom] >= nj[dn2]).all() and (nj[dn2] >= nj[dn5]).all()
    assert (nj[up5] > nj[dn5]).any()
    # HT_v <= sum over all jets of pt_v
    corr = hepo.lookup_binned(wl.jets.pt, wl.jets.eta, wl.calib["pt_edges"], wl.calib["eta_edges"], wl.calib["table"])
    for v, s in enumerate(wl.calib["scales"]):
        ptv = wl.jets.pt * (corr * np.float32(s))
        tot = hepo.segmented_reduce("sum", ptv, wl.jets.offsets)
        assert (res["ht"][v] <= tot * (1 + 1e-6)).all()


def test_unit_table_variant0_equals_uncalibrated_bitwise():
    wl = hepgen.generate(3, n_events=3000)
    wl.calib["table"][:] = 1.0
    res_c = hepo.analysis_chain(wl)
    wl0 = hepgen.generate(3, n_events=3000)
    wl0.calib = None
    res_0 = hepo.analysis_chain(wl0)
    for k in ("njet", "argmax", "ht", "maxpt", "minpt", "mjj", "subpt", "jet_mask"):
        np.testing.assert_array_equal(res_c[k][0], res_0[k][0], err_msg=k)
    for name in wl.hists:
        np.testing.assert_array_equal(hepo.hist_view(res_c, name, wl)[0][0], hepo.hist_view(res_0, name, wl0)[0][0])


def test_chain_hand_worked_event():
    """Three events worked by hand against BASELINE.json config 0's chain definition."""
    wl = hepgen.generate(0, n_events=3)
    f = lambda *a: np.array(a, np.float32)
    # event 0: 4 jets; event 1: no jets; event 2: 2 jets
    wl.jets = hepgen.Collection(np.array([0, 4, 4, 6], np.int64),
                                pt=f(100, 50, 29, 80, 45, 31),
                                eta=f(0.0, 1.0, 0.5, 2.45, -1.0, 2.0),
                                phi=f(0.0, math.pi, 1.0, 2.0, 0.5, -3.0),
                                mass=f(0, 0, 5, 5, 10, 10))
    # event 0: one muon at (1.0, 3.0) -> dR to jet 1 = |pi - 3.0| = 0.14 -> jet 1 dropped; event 2: soft muon (pt 15) on top of jet 0 ignored
    wl.muons = hepgen.Collection(np.array([0, 1, 1, 2], np.int64), pt=f(40, 15), eta=f(1.0, -1.0), phi=f(3.0, 0.5),
                                 mass=f(0.1057, 0.1057))
    wl.electrons = None
    wl.weights = f(2.0, 3.0, 0.5).reshape(1, 3)
    res = hepo.analysis_chain(wl)
    # event 0: jet0 clean (pt 100); jet1 pt 50 matched -> dropped; jet2 pt 29 fails pt; jet3 |eta| 2.45 fails eta
    assert res["jet_mask"][0].tolist() == [1, 0, 0, 0, 1, 1]
    assert res["njet"][0].tolist() == [1, 0, 2]
    assert res["ht"][0].tolist() == [100.0, 0.0, 76.0]
    assert res["maxpt"][0].tolist() == [100.0, -np.inf, 45.0]
    assert res["minpt"][0].tolist() == [100.0, np.inf, 31.0]
    assert res["argmax"][0].tolist() == [0, -1, 0]
    assert res["subpt"][0].tolist() == [0.0, 0.0, 31.0]
    assert res["mjj"][0][0] == 0 and res["mjj"][0][1] == 0
    # event 2 mass by the textbook formula
    def p4(pt, eta, phi, m):
        return (math.sqrt((pt * math.cosh(eta)) ** 2 + m * m), pt * math.cos(phi), pt * math.sin(phi), pt * math.sinh(eta))
    a, b = p4(45, -1.0, 0.5, 10), p4(31, 2.0, -3.0, 10)
    s = [x + y for x, y in zip(a, b)]
    assert math.isclose(res["mjj"][0][2], math.sqrt(s[0] ** 2 - s[1] ** 2 - s[2] ** 2 - s[3] ** 2), rel_tol=1e-6)
    # HT histogram (100 bins of width 10 on [0,1000]): 100 -> bin 10 (slot 11) weight 2; 0 -> slot 1 weight 3; 76 -> slot 8 weight .5
    sw, ct = hepo.hist_view(res, "ht", wl)
    want = np.zeros(102, np.float32)
    want[11], want[1], want[8] = 2.0, 3.0, 0.5
    np.testing.assert_array_equal(sw[0, 0], want)
    np.testing.assert_array_equal(ct[0], (want > 0).astype(np.int64))


def test_chain_event_range_matches_whole():
    wl = hepgen.generate(2, n_events=2000)
    whole = hepo.analysis_chain(wl)
    a = hepo.analysis_chain(wl, 0, 777)
    b = hepo.analysis_chain(wl, 777, 2000, hist_sumw=a["hist_sumw"].copy(), hist_counts=a["hist_counts"].copy())
    for k in ("njet", "ht", "mjj", "argmax"):
        np.testing.assert_array_equal(np.concatenate([a[k], b[k]], axis=1), whole[k])
    np.testing.assert_array_equal(b["hist_counts"], whole["hist_counts"])
    np.testing.assert_allclose(b["hist_sumw"], whole["hist_sumw"], rtol=1e-6)
