"""ctypes wrapper of the CPU oracle (oracle/libhepo.so).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this module.  numpy arrays in, numpy arrays out; no arithmetic of the method lives here
(argument marshalling only).
"""
from __future__ import annotations

import ctypes as C

import numpy as np

from . import build as _build

OBSERVABLES = ("njet", "ht", "maxpt", "minpt", "mjj", "subpt")
N_OBS = len(OBSERVABLES)

_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.hepo_chain_desc_size.restype = C.c_size_t
        assert _lib.hepo_chain_desc_size() == C.sizeof(ChainDesc), "hepo_chain_desc layout mismatch"
    return _lib


def _p(a, dtype):
    """Pointer to a C-contiguous numpy array of the given dtype (or NULL)."""
    if a is None:
        return None
    assert isinstance(a, np.ndarray) and a.dtype == dtype and a.flags.c_contiguous, (a.dtype, dtype)
    return a.ctypes.data_as(C.c_void_p)


def _f32(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _u8(a):
    if a is None:
        return None
    a = np.asarray(a)
    if a.dtype == np.bool_:
        a = a.view(np.uint8)
    return np.ascontiguousarray(a, dtype=np.uint8)


def _i64(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.int64)


def _check(rc):
    if rc != 0:
        raise ValueError(f"oracle call failed with status {rc}")


def select_mask(pt, eta, pt_min, abs_eta_max):
    pt, eta = _f32(pt), _f32(eta)
    out = np.empty(pt.shape[0], dtype=np.uint8)
    _check(lib().hepo_select_mask(_p(pt, np.float32), _p(eta, np.float32), C.c_int64(pt.shape[0]),
                                  C.c_float(pt_min), C.c_float(abs_eta_max), _p(out, np.uint8)))
    return out


def segmented_reduce(op, data, offsets, mask_rows=None, mask_content=None, content_base=0):
    data, offsets = _f32(data), _i64(offsets)
    mask_rows, mask_content = _u8(mask_rows), _u8(mask_content)
    n = offsets.shape[0] - 1
    out = np.empty(n, dtype=np.int32 if op in ("count", "argmax") else np.float32)
    fn = getattr(lib(), f"hepo_segmented_reduce_{op}")
    _check(fn(_p(data, np.float32), _p(offsets, np.int64), C.c_int64(n), C.c_int64(content_base),
              _p(mask_rows, np.uint8), _p(mask_content, np.uint8), _p(out, out.dtype)))
    return out


def deltar_mask(eta1, phi1, offsets1, sel1, eta2, phi2, offsets2, sel2, dr_max, base1=0, base2=0):
    eta1, phi1, eta2, phi2 = _f32(eta1), _f32(phi1), _f32(eta2), _f32(phi2)
    offsets1, offsets2 = _i64(offsets1), _i64(offsets2)
    sel1, sel2 = _u8(sel1), _u8(sel2)
    n = offsets1.shape[0] - 1
    out = np.zeros(eta1.shape[0], dtype=np.uint8)
    _check(lib().hepo_deltar_mask(_p(eta1, np.float32), _p(phi1, np.float32), _p(offsets1, np.int64), C.c_int64(base1),
                                  _p(sel1, np.uint8), _p(eta2, np.float32), _p(phi2, np.float32),
                                  _p(offsets2, np.int64), C.c_int64(base2), _p(sel2, np.uint8),
                                  C.c_int64(n), C.c_float(dr_max), _p(out, np.uint8)))
    return out


def pair_invmass(pt, eta, phi, mass, offsets, mask_content=None, content_base=0):
    pt, eta, phi, mass = _f32(pt), _f32(eta), _f32(phi), _f32(mass)
    offsets, mask_content = _i64(offsets), _u8(mask_content)
    n = offsets.shape[0] - 1
    m = np.empty(n, dtype=np.float32)
    i1 = np.empty(n, dtype=np.int32)
    i2 = np.empty(n, dtype=np.int32)
    _check(lib().hepo_pair_invmass(_p(pt, np.float32), _p(eta, np.float32), _p(phi, np.float32), _p(mass, np.float32),
                                   _p(offsets, np.int64), C.c_int64(n), C.c_int64(content_base),
                                   _p(mask_content, np.uint8), _p(m, np.float32), _p(i1, np.int32), _p(i2, np.int32)))
    return m, i1, i2


def get_in_offsets(data, offsets, index, mask_rows=None, mask_content=None, fill=0.0, content_base=0):
    data, offsets = _f32(data), _i64(offsets)
    mask_rows, mask_content = _u8(mask_rows), _u8(mask_content)
    n = offsets.shape[0] - 1
    out = np.empty(n, dtype=np.float32)
    _check(lib().hepo_get_in_offsets(_p(data, np.float32), _p(offsets, np.int64), C.c_int64(n), C.c_int64(content_base),
                                     _p(mask_rows, np.uint8), _p(mask_content, np.uint8), C.c_int32(index),
                                     C.c_float(fill), _p(out, np.float32)))
    return out


def set_in_offsets(data, offsets, index, values=None, value=0.0, mask_rows=None, mask_content=None, content_base=0):
    """Returns a modified copy of `data`."""
    data, offsets, values = _f32(data).copy(), _i64(offsets), _f32(values)
    mask_rows, mask_content = _u8(mask_rows), _u8(mask_content)
    n = offsets.shape[0] - 1
    _check(lib().hepo_set_in_offsets(_p(data, np.float32), _p(offsets, np.int64), C.c_int64(n), C.c_int64(content_base),
                                     _p(mask_rows, np.uint8), _p(mask_content, np.uint8), C.c_int32(index),
                                     _p(values, np.float32), C.c_float(value)))
    return data


def select_opposite_sign(pt, charge, offsets, mask_rows=None, mask_content=None, content_base=0):
    pt, offsets = _f32(pt), _i64(offsets)
    charge = np.ascontiguousarray(charge, dtype=np.int32)
    mask_rows, mask_content = _u8(mask_rows), _u8(mask_content)
    n = offsets.shape[0] - 1
    out = np.zeros(pt.shape[0], dtype=np.uint8)
    _check(lib().hepo_select_opposite_sign(_p(pt, np.float32), _p(charge, np.int32), _p(offsets, np.int64), C.c_int64(n),
                                           C.c_int64(content_base), _p(mask_rows, np.uint8), _p(mask_content, np.uint8),
                                           _p(out, np.uint8)))
    return out


def lookup_binned(x, y, edges_x, edges_y, table):
    x, y, edges_x, edges_y = _f32(x), _f32(y), _f32(edges_x), _f32(edges_y)
    table = _f32(table)
    out = np.empty(x.shape[0], dtype=np.float32)
    nx = edges_x.shape[0] - 1
    ny = 0 if edges_y is None else edges_y.shape[0] - 1
    _check(lib().hepo_lookup_binned(_p(x, np.float32), _p(y, np.float32), C.c_int64(x.shape[0]),
                                    _p(edges_x, np.float32), C.c_int32(nx), _p(edges_y, np.float32), C.c_int32(ny),
                                    _p(table, np.float32), _p(out, np.float32)))
    return out


def fill_histogram(data, weights, edges, sumw=None, counts=None):
    """Returns (sumw float32[nbins+2], counts int64[nbins+2]); both accumulate into the arrays passed in."""
    data, weights, edges = _f32(data), _f32(weights), _f32(edges)
    nbins = edges.shape[0] - 1
    if sumw is None:
        sumw = np.zeros(nbins + 2, dtype=np.float32)
    if counts is None:
        counts = np.zeros(nbins + 2, dtype=np.int64)
    _check(lib().hepo_fill_histogram(_p(data, np.float32), _p(weights, np.float32), C.c_int64(data.shape[0]),
                                     _p(edges, np.float32), C.c_int32(nbins), _p(sumw, np.float32), _p(counts, np.int64)))
    return sumw, counts


def fill_histogram_w2(data, weights, edges, sumw=None, sumw2=None, counts=None):
    """Returns (sumw, sumw2 float32[nbins+2], counts int64[nbins+2]); all accumulate into the arrays passed in."""
    data, weights, edges = _f32(data), _f32(weights), _f32(edges)
    nbins = edges.shape[0] - 1
    if sumw is None:
        sumw = np.zeros(nbins + 2, dtype=np.float32)
    if sumw2 is None:
        sumw2 = np.zeros(nbins + 2, dtype=np.float32)
    if counts is None:
        counts = np.zeros(nbins + 2, dtype=np.int64)
    _check(lib().hepo_fill_histogram_w2(_p(data, np.float32), _p(weights, np.float32), C.c_int64(data.shape[0]),
                                        _p(edges, np.float32), C.c_int32(nbins), _p(sumw, np.float32),
                                        _p(sumw2, np.float32), _p(counts, np.int64)))
    return sumw, sumw2, counts


def event_weight_lookup(w_in, x, edges, table):
    w_in, x, edges, table = _f32(w_in), _f32(x), _f32(edges), _f32(table)
    out = np.empty(x.shape[0], dtype=np.float32)
    _check(lib().hepo_event_weight_lookup(_p(w_in, np.float32), _p(x, np.float32), C.c_int64(x.shape[0]),
                                          _p(edges, np.float32), C.c_int32(edges.shape[0] - 1), _p(table, np.float32),
                                          _p(out, np.float32)))
    return out


def lookup_interp(x, xs, ys):
    x, xs, ys = _f32(x), _f32(xs), _f32(ys)
    out = np.empty(x.shape[0], dtype=np.float32)
    _check(lib().hepo_lookup_interp(_p(x, np.float32), C.c_int64(x.shape[0]), _p(xs, np.float32), _p(ys, np.float32),
                                    C.c_int32(xs.shape[0]), _p(out, np.float32)))
    return out


def fill_histogram_2d(x, y, weights, edges_x, edges_y, sumw=None, counts=None):
    """Returns (sumw float32[nx+2][ny+2], counts int64[nx+2][ny+2]); both accumulate into the arrays passed in."""
    x, y, weights, edges_x, edges_y = _f32(x), _f32(y), _f32(weights), _f32(edges_x), _f32(edges_y)
    nx, ny = edges_x.shape[0] - 1, edges_y.shape[0] - 1
    if sumw is None:
        sumw = np.zeros((nx + 2, ny + 2), dtype=np.float32)
    if counts is None:
        counts = np.zeros((nx + 2, ny + 2), dtype=np.int64)
    _check(lib().hepo_fill_histogram_2d(_p(x, np.float32), _p(y, np.float32), _p(weights, np.float32), C.c_int64(x.shape[0]),
                                        _p(edges_x, np.float32), C.c_int32(nx), _p(edges_y, np.float32), C.c_int32(ny),
                                        _p(sumw, np.float32), _p(counts, np.int64)))
    return sumw, counts


def fill_histogram_2d_w2(x, y, weights, edges_x, edges_y, sumw=None, sumw2=None, counts=None):
    """Returns (sumw, sumw2 float32[nx+2][ny+2], counts int64[nx+2][ny+2]); all accumulate."""
    x, y, weights, edges_x, edges_y = _f32(x), _f32(y), _f32(weights), _f32(edges_x), _f32(edges_y)
    nx, ny = edges_x.shape[0] - 1, edges_y.shape[0] - 1
    if sumw is None:
        sumw = np.zeros((nx + 2, ny + 2), dtype=np.float32)
    if sumw2 is None:
        sumw2 = np.zeros((nx + 2, ny + 2), dtype=np.float32)
    if counts is None:
        counts = np.zeros((nx + 2, ny + 2), dtype=np.int64)
    _check(lib().hepo_fill_histogram_2d_w2(_p(x, np.float32), _p(y, np.float32), _p(weights, np.float32), C.c_int64(x.shape[0]),
                                           _p(edges_x, np.float32), C.c_int32(nx), _p(edges_y, np.float32), C.c_int32(ny),
                                           _p(sumw, np.float32), _p(sumw2, np.float32), _p(counts, np.int64)))
    return sumw, sumw2, counts


def triplet_mass(pt, eta, phi, mass, offsets, target, mask_rows=None, mask_content=None, content_base=0):
    """Returns (mass float32[n_events], indices int32[n_events][3])."""
    pt, eta, phi, mass, offsets = _f32(pt), _f32(eta), _f32(phi), _f32(mass), _i64(offsets)
    mask_rows, mask_content = _u8(mask_rows), _u8(mask_content)
    n = offsets.shape[0] - 1
    out = np.zeros(n, dtype=np.float32)
    idx = np.full((n, 3), -1, dtype=np.int32)
    _check(lib().hepo_triplet_mass(_p(pt, np.float32), _p(eta, np.float32), _p(phi, np.float32), _p(mass, np.float32),
                                   _p(offsets, np.int64), C.c_int64(n), C.c_int64(content_base), _p(mask_rows, np.uint8),
                                   _p(mask_content, np.uint8), C.c_float(target), _p(out, np.float32), _p(idx, np.int32)))
    return out, idx


def validate_offsets(offsets, n_objects, content_base=0):
    """Number of violations of the jagged-layout preconditions (0 = valid)."""
    offsets = _i64(offsets)
    bad = C.c_int64(0)
    _check(lib().hepo_validate_offsets(_p(offsets, np.int64), C.c_int64(offsets.shape[0] - 1), C.c_int64(content_base),
                                       C.c_int64(n_objects), C.byref(bad)))
    return bad.value


class Collection(C.Structure):
    _fields_ = [("offsets", C.c_void_p), ("content_base", C.c_int64), ("n_objects", C.c_int64),
                ("pt", C.c_void_p), ("eta", C.c_void_p), ("phi", C.c_void_p), ("mass", C.c_void_p)]


class ChainDesc(C.Structure):
    _fields_ = [
        ("n_events", C.c_int64),
        ("jets", Collection), ("muons", Collection), ("electrons", Collection),
        ("jet_pt_min", C.c_float), ("jet_abs_eta_max", C.c_float), ("lep_pt_min", C.c_float), ("dr_max", C.c_float),
        ("calib_pt_edges", C.c_void_p), ("calib_npt", C.c_int32),
        ("calib_eta_edges", C.c_void_p), ("calib_neta", C.c_int32),
        ("calib_table", C.c_void_p), ("calib_scales", C.c_void_p),
        ("n_variants", C.c_int32), ("n_wvar", C.c_int32),
        ("weights", C.c_void_p),
        ("axis_edges", C.c_void_p * N_OBS), ("axis_nbins", C.c_int32 * N_OBS),
        ("out_njet", C.c_void_p), ("out_argmax", C.c_void_p),
        ("out_ht", C.c_void_p), ("out_maxpt", C.c_void_p), ("out_minpt", C.c_void_p),
        ("out_mjj", C.c_void_p), ("out_subpt", C.c_void_p),
        ("out_jet_mask", C.c_void_p),
        ("hist_sumw", C.c_void_p), ("hist_counts", C.c_void_p),
        ("evw_x", C.c_void_p), ("evw_edges", C.c_void_p), ("evw_nbins", C.c_int32), ("evw_table", C.c_void_p),
        ("hist_sumw2", C.c_void_p),
    ]


def _coll(c, keep, e0=0, e1=None):
    s = Collection()
    if c is None:
        return s
    offsets = _i64(c.offsets)
    if e1 is None:
        e1 = offsets.shape[0] - 1
    keep.append(offsets)
    s.offsets = offsets.ctypes.data + 8 * e0
    s.content_base = 0
    s.n_objects = c.pt.shape[0]
    for name in ("pt", "eta", "phi", "mass"):
        a = _f32(getattr(c, name))
        keep.append(a)
        setattr(s, name, a.ctypes.data)
    return s


def hist_layout(hists, axes, n_variants, n_wvar):
    """Slot bookkeeping shared by callers: returns (obs_prefix dict, slots_per_variant)."""
    prefix, tot = {}, 0
    for name in OBSERVABLES:
        if name in hists:
            prefix[name] = tot
            tot += axes[name].shape[0] - 1 + 2
    return prefix, tot


def max_threads():
    return int(lib().hepo_omp_max_threads())


def analysis_chain(wl, e0=0, e1=None, want_mask=True, hist_sumw=None, hist_counts=None, evw=None, want_sumw2=False,
                   hist_sumw2=None, threads=1):
    """Run the oracle chain on events [e0, e1) of a hepgen.Workload.

    Returns a dict with per-event outputs [V][n], jet_mask [V][Mj] (whole collection; only rows of the
    event range are written), hist_sumw (flat float32) and hist_counts (flat int64), plus 'layout'.
    evw: optional dict(x=float32[n_events], edges=float32[nb+1], table=float32[nb]) — the per-event weight factor
    from a lookup; want_sumw2: also return hist_sumw2; threads != 1: the OpenMP timing leg (<= 0: all cores).
    """
    keep = []
    if e1 is None:
        e1 = wl.n_events
    n = e1 - e0
    d = ChainDesc()
    d.n_events = n
    d.jets = _coll(wl.jets, keep, e0, e1)
    d.muons = _coll(wl.muons, keep, e0, e1)
    d.electrons = _coll(wl.electrons, keep, e0, e1)
    d.jet_pt_min = wl.cuts["jet_pt_min"]
    d.jet_abs_eta_max = wl.cuts["jet_abs_eta_max"]
    d.lep_pt_min = wl.cuts["lep_pt_min"]
    d.dr_max = wl.cuts["dr_max"]
    V = 1
    if wl.calib is not None:
        pe, ee = _f32(wl.calib["pt_edges"]), _f32(wl.calib["eta_edges"])
        tb, sc = _f32(wl.calib["table"]), _f32(wl.calib["scales"])
        keep += [pe, ee, tb, sc]
        d.calib_pt_edges, d.calib_npt = pe.ctypes.data, pe.shape[0] - 1
        d.calib_eta_edges, d.calib_neta = ee.ctypes.data, ee.shape[0] - 1
        d.calib_table, d.calib_scales = tb.ctypes.data, sc.ctypes.data
        V = sc.shape[0]
    d.n_variants = V
    W = wl.weights.shape[0]
    d.n_wvar = W
    wts = np.ascontiguousarray(wl.weights[:, e0:e1], dtype=np.float32)
    keep.append(wts)
    d.weights = wts.ctypes.data
    for o, name in enumerate(OBSERVABLES):
        if name in wl.hists:
            ed = _f32(wl.axes[name])
            keep.append(ed)
            d.axis_edges[o] = ed.ctypes.data
            d.axis_nbins[o] = ed.shape[0] - 1
    out = {
        "njet": np.empty((V, n), np.int32), "argmax": np.empty((V, n), np.int32),
        "ht": np.empty((V, n), np.float32), "maxpt": np.empty((V, n), np.float32),
        "minpt": np.empty((V, n), np.float32), "mjj": np.empty((V, n), np.float32),
        "subpt": np.empty((V, n), np.float32),
    }
    for k, a in out.items():
        setattr(d, "out_" + k, a.ctypes.data)
    if want_mask:
        out["jet_mask"] = np.zeros((V, wl.jets.pt.shape[0]), np.uint8)
        d.out_jet_mask = out["jet_mask"].ctypes.data
    prefix, spv = hist_layout(wl.hists, wl.axes, V, W)
    if hist_sumw is None:
        hist_sumw = np.zeros(V * W * spv, np.float32)
    if hist_counts is None:
        hist_counts = np.zeros(V * spv, np.int64)
    d.hist_sumw, d.hist_counts = hist_sumw.ctypes.data, hist_counts.ctypes.data
    if evw is not None:
        ex = np.ascontiguousarray(np.asarray(evw["x"], dtype=np.float32)[e0:e1])
        ee, et = _f32(evw["edges"]), _f32(evw["table"])
        keep += [ex, ee, et]
        d.evw_x, d.evw_edges, d.evw_nbins, d.evw_table = ex.ctypes.data, ee.ctypes.data, ee.shape[0] - 1, et.ctypes.data
    if want_sumw2 or hist_sumw2 is not None:
        if hist_sumw2 is None:
            hist_sumw2 = np.zeros(V * W * spv, np.float32)
        d.hist_sumw2 = hist_sumw2.ctypes.data
        out["hist_sumw2"] = hist_sumw2
    if threads == 1:
        _check(lib().hepo_analysis_chain(C.byref(d)))
    else:
        _check(lib().hepo_analysis_chain_omp(C.byref(d), C.c_int32(threads)))
    out["hist_sumw"], out["hist_counts"] = hist_sumw, hist_counts
    out["layout"] = dict(prefix=prefix, slots_per_variant=spv, n_variants=V, n_wvar=W)
    return out


def hist_view(res, name, wl):
    """(sumw [V][W][nbins+2], counts [V][nbins+2]) views of one observable's histograms."""
    lay = res["layout"]
    V, W, spv = lay["n_variants"], lay["n_wvar"], lay["slots_per_variant"]
    nb2 = wl.axes[name].shape[0] - 1 + 2
    p = lay["prefix"][name]
    sw = res["hist_sumw"].reshape(V, W * spv)[:, W * p: W * p + W * nb2].reshape(V, W, nb2)
    ct = res["hist_counts"].reshape(V, spv)[:, p: p + nb2]
    return sw, ct
