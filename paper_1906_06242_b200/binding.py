"""Thin Python binding of libhepk.so (include/hepk.h): argument marshalling only.

Every function has the name of its C entry point without the `hepk_` prefix and takes torch CUDA
tensors (device memory and streams are all PyTorch is used for).  Every step of the path runs inside
the CUDA library; there is no CPU or PyTorch fallback — if the library is missing or a call fails,
an exception is raised.
"""
from __future__ import annotations

import ctypes as C
import os
from dataclasses import dataclass

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
# HEPK_LIBRARY overrides the path of the shared library (e.g. a build with other compile flags)
LIB_PATH = os.environ.get("HEPK_LIBRARY") or os.path.join(_HERE, "csrc", "libhepk.so")

OBSERVABLES = ("njet", "ht", "maxpt", "minpt", "mjj", "subpt")
N_OBS = 6
MAX_VARIANTS = 64
MAX_WVAR = 16
VARIANT_AUTO, VARIANT_WARP_PER_EVENT, VARIANT_BLOCK_PER_TILE = 0, 1, 2


class HepkError(RuntimeError):
    pass


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
        ("calib_table", C.c_void_p),
        ("calib_scales", C.c_float * MAX_VARIANTS),
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
        ("weights_stride", C.c_int64), ("out_stride", C.c_int64),
        ("tune_cap_jets", C.c_int32), ("tune_cap_leptons", C.c_int32),
        ("tune_ctas_per_sm", C.c_int32), ("tune_warps_per_cta", C.c_int32), ("tune_warps_per_sm", C.c_int32),
        ("tune_variants_per_pass", C.c_int32), ("tune_generic_build", C.c_int32),
    ]


_lib = None


def lib():
    """Load libhepk.so; fails loudly if it has not been built (python -m paper_1906_06242_b200.build)."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise HepkError(f"{LIB_PATH} is missing: build it with `python -m paper_1906_06242_b200.build` "
                            "(there is no CPU fallback)")
        L = C.CDLL(LIB_PATH)
        L.hepk_last_error.restype = C.c_char_p
        L.hepk_version.restype = C.c_int32
        L.hepk_chain_workspace_bytes.restype = C.c_size_t
        L.hepk_chain_workspace_bytes.argtypes = [C.POINTER(ChainDesc)]
        L.hepk_chain_host_workspace_bytes.restype = C.c_size_t
        L.hepk_chain_host_workspace_bytes.argtypes = [C.POINTER(ChainDesc), C.c_int64]
        _lib = L
    return _lib


def _check(rc, name):
    if rc != 0:
        raise HepkError(f"hepk_{name} failed ({rc}): {lib().hepk_last_error().decode()}")


def _ptr(t, dtype=None):
    if t is None:
        return None
    assert isinstance(t, torch.Tensor) and t.is_cuda and t.is_contiguous(), "expected a contiguous CUDA tensor"
    if dtype is not None:
        assert t.dtype == dtype, (t.dtype, dtype)
    if t.numel() == 0:          # torch gives empty tensors a NULL data_ptr; the C ABI wants a valid (unread) pointer
        return C.c_void_p(_empty_buffer(t.device).data_ptr())
    return C.c_void_p(t.data_ptr())


_EMPTY = {}


def _empty_buffer(device):
    if device not in _EMPTY:
        _EMPTY[device] = torch.zeros(16, dtype=torch.uint8, device=device)
    return _EMPTY[device]


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _mask(t):
    if t is not None and t.dtype == torch.bool:
        t = t.view(torch.uint8)
    return t


def version():
    return lib().hepk_version()


def last_error():
    return lib().hepk_last_error().decode()


def kernel_launches():
    """Kernels this library has enqueued in this process so far."""
    L = lib()
    L.hepk_kernel_launches.restype = C.c_int64
    return int(L.hepk_kernel_launches())


def probe_shared_atomics(warps_per_sm=16, nbins=32768):
    """Measured red.shared.add.s32 rate of the device (lane-atomics per second, random addresses)."""
    scratch = torch.zeros(4096, dtype=torch.int32, device="cuda")
    r = C.c_double(0.0)
    _check(lib().hepk_probe_shared_atomics(C.c_int32(warps_per_sm), C.c_int32(nbins), C.c_void_p(scratch.data_ptr()), C.byref(r)),
           "probe_shared_atomics")
    return r.value


def profile_begin():
    _check(lib().hepk_profile_begin(), "profile_begin")


def profile_end():
    """(summed milliseconds of the fused chain kernel, number of timed launches) since profile_begin()."""
    ms, n = C.c_double(0.0), C.c_int32(0)
    _check(lib().hepk_profile_end(C.byref(ms), C.byref(n)), "profile_end")
    return ms.value, n.value


def select_mask(pt, eta, pt_min, abs_eta_max, out=None, stream=None):
    n = pt.numel()
    if out is None:
        out = torch.empty(n, dtype=torch.uint8, device=pt.device)
    _check(lib().hepk_select_mask(_ptr(pt, torch.float32), _ptr(eta, torch.float32), C.c_int64(n), C.c_float(pt_min),
                                  C.c_float(abs_eta_max), _ptr(out, torch.uint8), _stream(stream)), "select_mask")
    return out


def _segmented(op, data, offsets, mask_rows, mask_content, content_base, out, variant, stream):
    n = offsets.numel() - 1
    dt = torch.int32 if op in ("count", "argmax") else torch.float32
    if out is None:
        out = torch.empty(n, dtype=dt, device=offsets.device)
    fn = getattr(lib(), f"hepk_segmented_reduce_{op}")
    _check(fn(_ptr(data, torch.float32), _ptr(offsets, torch.int64), C.c_int64(n), C.c_int64(content_base),
              _ptr(_mask(mask_rows), torch.uint8), _ptr(_mask(mask_content), torch.uint8), _ptr(out, dt),
              C.c_int32(variant), _stream(stream)), f"segmented_reduce_{op}")
    return out


def segmented_reduce_sum(data, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, variant=0, stream=None):
    return _segmented("sum", data, offsets, mask_rows, mask_content, content_base, out, variant, stream)


def segmented_reduce_max(data, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, variant=0, stream=None):
    return _segmented("max", data, offsets, mask_rows, mask_content, content_base, out, variant, stream)


def segmented_reduce_min(data, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, variant=0, stream=None):
    return _segmented("min", data, offsets, mask_rows, mask_content, content_base, out, variant, stream)


def segmented_reduce_count(data, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, variant=0, stream=None):
    return _segmented("count", data, offsets, mask_rows, mask_content, content_base, out, variant, stream)


def segmented_reduce_argmax(data, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, variant=0, stream=None):
    return _segmented("argmax", data, offsets, mask_rows, mask_content, content_base, out, variant, stream)


def deltar_mask(eta1, phi1, offsets1, sel1, eta2, phi2, offsets2, sel2, dr_max, base1=0, base2=0, out=None, stream=None):
    n = offsets1.numel() - 1
    if out is None:
        out = torch.zeros(eta1.numel(), dtype=torch.uint8, device=eta1.device)
    _check(lib().hepk_deltar_mask(_ptr(eta1, torch.float32), _ptr(phi1, torch.float32), _ptr(offsets1, torch.int64),
                                  C.c_int64(base1), _ptr(_mask(sel1), torch.uint8),
                                  _ptr(eta2, torch.float32), _ptr(phi2, torch.float32), _ptr(offsets2, torch.int64),
                                  C.c_int64(base2), _ptr(_mask(sel2), torch.uint8),
                                  C.c_int64(n), C.c_float(dr_max), _ptr(out, torch.uint8), _stream(stream)), "deltar_mask")
    return out


def pair_invmass(pt, eta, phi, mass, offsets, mask_content=None, content_base=0, want_indices=True, stream=None):
    n = offsets.numel() - 1
    dev = offsets.device
    m = torch.empty(n, dtype=torch.float32, device=dev)
    i1 = torch.empty(n, dtype=torch.int32, device=dev) if want_indices else None
    i2 = torch.empty(n, dtype=torch.int32, device=dev) if want_indices else None
    _check(lib().hepk_pair_invmass(_ptr(pt, torch.float32), _ptr(eta, torch.float32), _ptr(phi, torch.float32),
                                   _ptr(mass, torch.float32), _ptr(offsets, torch.int64), C.c_int64(n),
                                   C.c_int64(content_base), _ptr(_mask(mask_content), torch.uint8),
                                   _ptr(m, torch.float32), _ptr(i1, torch.int32), _ptr(i2, torch.int32),
                                   _stream(stream)), "pair_invmass")
    return m, i1, i2


def get_in_offsets(data, offsets, index, mask_rows=None, mask_content=None, fill=0.0, content_base=0, out=None, stream=None):
    n = offsets.numel() - 1
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=offsets.device)
    _check(lib().hepk_get_in_offsets(_ptr(data, torch.float32), _ptr(offsets, torch.int64), C.c_int64(n), C.c_int64(content_base),
                                     _ptr(_mask(mask_rows), torch.uint8), _ptr(_mask(mask_content), torch.uint8),
                                     C.c_int32(index), C.c_float(fill), _ptr(out, torch.float32), _stream(stream)),
           "get_in_offsets")
    return out


def set_in_offsets(data, offsets, index, values=None, value=0.0, mask_rows=None, mask_content=None, content_base=0, stream=None):
    """In place on `data`; returns it."""
    n = offsets.numel() - 1
    _check(lib().hepk_set_in_offsets(_ptr(data, torch.float32), _ptr(offsets, torch.int64), C.c_int64(n), C.c_int64(content_base),
                                     _ptr(_mask(mask_rows), torch.uint8), _ptr(_mask(mask_content), torch.uint8),
                                     C.c_int32(index), _ptr(values, torch.float32), C.c_float(value), _stream(stream)),
           "set_in_offsets")
    return data


def select_opposite_sign(pt, charge, offsets, mask_rows=None, mask_content=None, content_base=0, out=None, stream=None):
    n = offsets.numel() - 1
    if out is None:
        out = torch.empty(pt.numel(), dtype=torch.uint8, device=pt.device)
    _check(lib().hepk_select_opposite_sign(_ptr(pt, torch.float32), _ptr(charge, torch.int32), _ptr(offsets, torch.int64),
                                           C.c_int64(n), C.c_int64(content_base), _ptr(_mask(mask_rows), torch.uint8),
                                           _ptr(_mask(mask_content), torch.uint8), _ptr(out, torch.uint8), _stream(stream)),
           "select_opposite_sign")
    return out


def lookup_interp(x, xs, ys, out=None, stream=None):
    n = x.numel()
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=x.device)
    _check(lib().hepk_lookup_interp(_ptr(x, torch.float32), C.c_int64(n), _ptr(xs, torch.float32), _ptr(ys, torch.float32),
                                    C.c_int32(xs.numel()), _ptr(out, torch.float32), _stream(stream)), "lookup_interp")
    return out


def fill_histogram_2d(x, y, weights, edges_x, edges_y, sumw=None, counts=None, want_sumw=True, want_counts=True, stream=None):
    """Returns (sumw float32[nx+2][ny+2] or None, counts int64[nx+2][ny+2] or None); both accumulate."""
    nx, ny = edges_x.numel() - 1, edges_y.numel() - 1
    dev = x.device
    if sumw is None and want_sumw:
        sumw = torch.zeros((nx + 2, ny + 2), dtype=torch.float32, device=dev)
    if counts is None and want_counts:
        counts = torch.zeros((nx + 2, ny + 2), dtype=torch.int64, device=dev)
    L = lib()
    L.hepk_hist2d_workspace_bytes.restype = C.c_size_t
    nbytes = L.hepk_hist2d_workspace_bytes(C.c_int32(nx), C.c_int32(ny))
    ws = torch.empty(max(int(nbytes), 8), dtype=torch.uint8, device=dev)
    _check(L.hepk_fill_histogram_2d(_ptr(x, torch.float32), _ptr(y, torch.float32), _ptr(weights, torch.float32),
                                    C.c_int64(x.numel()), _ptr(edges_x, torch.float32), C.c_int32(nx),
                                    _ptr(edges_y, torch.float32), C.c_int32(ny), _ptr(sumw, torch.float32),
                                    _ptr(counts, torch.int64), C.c_void_p(ws.data_ptr()), C.c_size_t(ws.numel()),
                                    _stream(stream)), "fill_histogram_2d")
    return sumw, counts


def _hist_ws(nx, ny, dev):
    L = lib()
    L.hepk_hist_workspace_bytes.restype = C.c_size_t
    return torch.empty(max(int(L.hepk_hist_workspace_bytes(C.c_int32(nx), C.c_int32(ny))), 8), dtype=torch.uint8, device=dev)


def fill_histogram_w2(data, weights, edges, sumw=None, sumw2=None, counts=None, want=("sumw", "sumw2", "counts"), stream=None):
    """Returns (sumw, sumw2 float32[nbins+2], counts int64[nbins+2]); arrays not in `want` and not given are None."""
    nbins = edges.numel() - 1
    dev = edges.device
    if sumw is None and "sumw" in want:
        sumw = torch.zeros(nbins + 2, dtype=torch.float32, device=dev)
    if sumw2 is None and "sumw2" in want:
        sumw2 = torch.zeros(nbins + 2, dtype=torch.float32, device=dev)
    if counts is None and "counts" in want:
        counts = torch.zeros(nbins + 2, dtype=torch.int64, device=dev)
    ws = _hist_ws(nbins, 0, dev)
    _check(lib().hepk_fill_histogram_w2(_ptr(data, torch.float32), _ptr(weights, torch.float32), C.c_int64(data.numel()),
                                        _ptr(edges, torch.float32), C.c_int32(nbins), _ptr(sumw, torch.float32),
                                        _ptr(sumw2, torch.float32), _ptr(counts, torch.int64), C.c_void_p(ws.data_ptr()),
                                        C.c_size_t(ws.numel()), _stream(stream)), "fill_histogram_w2")
    return sumw, sumw2, counts


def static_hist_scratch_bytes():
    L = lib()
    L.hepk_static_hist_scratch_bytes.restype = C.c_size_t
    return int(L.hepk_static_hist_scratch_bytes())


def fill_histogram_w2_static(data, weights, edges, sumw, sumw2, counts, stream=None):
    """hepk_fill_histogram_w2_static: the caller passes every array (each may be None); nothing is allocated, here
    or in the library.  Calls on one device share the library's scratch array: do not let two overlap on the GPU."""
    _check(lib().hepk_fill_histogram_w2_static(_ptr(data, torch.float32), _ptr(weights, torch.float32), C.c_int64(data.numel()),
                                               _ptr(edges, torch.float32), C.c_int32(edges.numel() - 1),
                                               _ptr(sumw, torch.float32), _ptr(sumw2, torch.float32), _ptr(counts, torch.int64),
                                               _stream(stream)), "fill_histogram_w2_static")
    return sumw, sumw2, counts


def fill_histogram_2d_w2(x, y, weights, edges_x, edges_y, sumw=None, sumw2=None, counts=None,
                         want=("sumw", "sumw2", "counts"), stream=None):
    nx, ny = edges_x.numel() - 1, edges_y.numel() - 1
    dev = x.device
    if sumw is None and "sumw" in want:
        sumw = torch.zeros((nx + 2, ny + 2), dtype=torch.float32, device=dev)
    if sumw2 is None and "sumw2" in want:
        sumw2 = torch.zeros((nx + 2, ny + 2), dtype=torch.float32, device=dev)
    if counts is None and "counts" in want:
        counts = torch.zeros((nx + 2, ny + 2), dtype=torch.int64, device=dev)
    ws = _hist_ws(nx, ny, dev)
    _check(lib().hepk_fill_histogram_2d_w2(_ptr(x, torch.float32), _ptr(y, torch.float32), _ptr(weights, torch.float32),
                                           C.c_int64(x.numel()), _ptr(edges_x, torch.float32), C.c_int32(nx),
                                           _ptr(edges_y, torch.float32), C.c_int32(ny), _ptr(sumw, torch.float32),
                                           _ptr(sumw2, torch.float32), _ptr(counts, torch.int64), C.c_void_p(ws.data_ptr()),
                                           C.c_size_t(ws.numel()), _stream(stream)), "fill_histogram_2d_w2")
    return sumw, sumw2, counts


def event_weight_lookup(w_in, x, edges, table, out=None, stream=None):
    n = x.numel()
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=x.device)
    _check(lib().hepk_event_weight_lookup(_ptr(w_in, torch.float32), _ptr(x, torch.float32), C.c_int64(n),
                                          _ptr(edges, torch.float32), C.c_int32(edges.numel() - 1), _ptr(table, torch.float32),
                                          _ptr(out, torch.float32), _stream(stream)), "event_weight_lookup")
    return out


def triplet_mass(pt, eta, phi, mass, offsets, target, mask_rows=None, mask_content=None, content_base=0, want_indices=True,
                 stream=None):
    """Returns (mass float32[n_events], indices int32[n_events][3] or None)."""
    n = offsets.numel() - 1
    out = torch.empty(n, dtype=torch.float32, device=offsets.device)
    idx = torch.empty((n, 3), dtype=torch.int32, device=offsets.device) if want_indices else None
    _check(lib().hepk_triplet_mass(_ptr(pt, torch.float32), _ptr(eta, torch.float32), _ptr(phi, torch.float32),
                                   _ptr(mass, torch.float32), _ptr(offsets, torch.int64), C.c_int64(n), C.c_int64(content_base),
                                   _ptr(_mask(mask_rows), torch.uint8), _ptr(_mask(mask_content), torch.uint8),
                                   C.c_float(target), _ptr(out, torch.float32), _ptr(idx, torch.int32), _stream(stream)),
           "triplet_mass")
    return out, idx


def validate_offsets(offsets, n_objects, content_base=0, stream=None):
    """Number of violations of the jagged-layout preconditions (synchronises to read the count back)."""
    out = torch.zeros(1, dtype=torch.int64, device=offsets.device)
    _check(lib().hepk_validate_offsets(_ptr(offsets, torch.int64), C.c_int64(offsets.numel() - 1), C.c_int64(content_base),
                                       C.c_int64(n_objects), _ptr(out, torch.int64), _stream(stream)), "validate_offsets")
    return int(out.item())


def lookup_binned(x, y, edges_x, edges_y, table, out=None, stream=None):
    n = x.numel()
    if out is None:
        out = torch.empty(n, dtype=torch.float32, device=x.device)
    nx = edges_x.numel() - 1
    ny = 0 if edges_y is None else edges_y.numel() - 1
    _check(lib().hepk_lookup_binned(_ptr(x, torch.float32), _ptr(y, torch.float32), C.c_int64(n),
                                    _ptr(edges_x, torch.float32), C.c_int32(nx), _ptr(edges_y, torch.float32), C.c_int32(ny),
                                    _ptr(table, torch.float32), _ptr(out, torch.float32), _stream(stream)), "lookup_binned")
    return out


def fill_histogram(data, weights, edges, sumw=None, counts=None, want_sumw=True, want_counts=True, stream=None):
    """Accumulates into sumw float32[nbins+2] / counts int64[nbins+2] (created zeroed when not given)."""
    nbins = edges.numel() - 1
    if sumw is None and want_sumw:
        sumw = torch.zeros(nbins + 2, dtype=torch.float32, device=edges.device)
    if counts is None and want_counts:
        counts = torch.zeros(nbins + 2, dtype=torch.int64, device=edges.device)
    _check(lib().hepk_fill_histogram(_ptr(data, torch.float32), _ptr(weights, torch.float32), C.c_int64(data.numel()),
                                     _ptr(edges, torch.float32), C.c_int32(nbins), _ptr(sumw, torch.float32),
                                     _ptr(counts, torch.int64), _stream(stream)), "fill_histogram")
    return sumw, counts


# ------------------------------------------------------------------------------------------ fused chain
@dataclass
class DeviceCollection:
    offsets: torch.Tensor          # int64 [n_events+1]
    pt: torch.Tensor
    eta: torch.Tensor
    phi: torch.Tensor
    mass: torch.Tensor | None = None
    content_base: int = 0


@dataclass
class ChainInputs:
    """Device-resident inputs of one chain call (tensors only; no arithmetic)."""
    n_events: int
    jets: DeviceCollection
    muons: DeviceCollection
    electrons: DeviceCollection | None
    weights: torch.Tensor | None            # float32 [n_wvar][n_events]
    cuts: dict                              # jet_pt_min, jet_abs_eta_max, lep_pt_min, dr_max
    hists: tuple                            # names from OBSERVABLES
    axes: dict                              # name -> float32 device tensor of edges
    calib: dict | None = None               # pt_edges, eta_edges, table (device), scales (list of float)
    evw: dict | None = None                 # event-weight lookup: x [n_events], edges [nb+1], table [nb] (device float32)

    @property
    def n_variants(self):
        return 1 if self.calib is None else len(self.calib["scales"])

    @property
    def n_wvar(self):
        return 1 if self.weights is None else int(self.weights.shape[0])


def upload(wl, device="cuda"):
    """hepgen.Workload (numpy, host) -> ChainInputs (torch, device).  A plain host->device copy."""
    def coll(c):
        if c is None:
            return None
        t = lambda a: torch.from_numpy(a).to(device)
        return DeviceCollection(t(c.offsets), t(c.pt), t(c.eta), t(c.phi), t(c.mass))
    calib = None
    if wl.calib is not None:
        calib = dict(pt_edges=torch.from_numpy(wl.calib["pt_edges"]).to(device),
                     eta_edges=torch.from_numpy(wl.calib["eta_edges"]).to(device),
                     table=torch.from_numpy(wl.calib["table"]).to(device).contiguous(),
                     scales=[float(s) for s in wl.calib["scales"]])
    return ChainInputs(n_events=wl.n_events, jets=coll(wl.jets), muons=coll(wl.muons), electrons=coll(wl.electrons),
                       weights=torch.from_numpy(wl.weights).to(device).contiguous(), cuts=dict(wl.cuts),
                       hists=tuple(wl.hists), axes={k: torch.from_numpy(v).to(device) for k, v in wl.axes.items()},
                       calib=calib)


def hist_layout(hists, axes):
    prefix, tot = {}, 0
    for name in OBSERVABLES:
        if name in hists:
            prefix[name] = tot
            tot += axes[name].numel() - 1 + 2
    return prefix, tot


def _fill_collection(s, c):
    if c is None:
        return
    s.offsets = c.offsets.data_ptr()
    s.content_base = c.content_base
    s.n_objects = c.pt.numel()
    s.pt, s.eta, s.phi = c.pt.data_ptr(), c.eta.data_ptr(), c.phi.data_ptr()
    s.mass = c.mass.data_ptr() if c.mass is not None else None
    for t in (c.offsets, c.pt, c.eta, c.phi):
        assert t.is_cuda and (t.numel() <= 1 or t.stride(0) == 1)
    assert c.offsets.dtype == torch.int64 and c.pt.dtype == torch.float32


class ChainPlan:
    """Pre-built descriptor, outputs and workspace for repeated hepk_analysis_chain calls on fixed buffers."""

    EVENT_OUTPUTS = ("njet", "argmax", "ht", "maxpt", "minpt", "mjj", "subpt")

    def __init__(self, inp: ChainInputs, want_event_outputs=True, want_mask=False, want_hists=True, want_counts=True,
                 want_sumw2=False, tune=None, out_into=None, out_col=0):
        """want_event_outputs: True (all seven), False (none) or a tuple of names from EVENT_OUTPUTS.
        out_into: dict name -> tensor [V][N_total] of a larger workload; this plan (a shard of it) then writes its
        per-event outputs at columns [out_col, out_col + n_events) of those arrays instead of allocating its own."""
        self.inp = inp
        dev = inp.jets.pt.device
        N, V, W = inp.n_events, inp.n_variants, inp.n_wvar
        d = ChainDesc()
        d.n_events = N
        _fill_collection(d.jets, inp.jets)
        _fill_collection(d.muons, inp.muons)
        _fill_collection(d.electrons, inp.electrons)
        d.jet_pt_min = inp.cuts["jet_pt_min"]
        d.jet_abs_eta_max = inp.cuts["jet_abs_eta_max"]
        d.lep_pt_min = inp.cuts["lep_pt_min"]
        d.dr_max = inp.cuts["dr_max"]
        if inp.calib is not None:
            d.calib_pt_edges = inp.calib["pt_edges"].data_ptr()
            d.calib_npt = inp.calib["pt_edges"].numel() - 1
            d.calib_eta_edges = inp.calib["eta_edges"].data_ptr()
            d.calib_neta = inp.calib["eta_edges"].numel() - 1
            d.calib_table = inp.calib["table"].data_ptr()
            for i, s in enumerate(inp.calib["scales"]):
                d.calib_scales[i] = s
        d.n_variants, d.n_wvar = V, W
        if inp.weights is not None:
            wt = inp.weights                   # [W][N], rows contiguous; a column slice of a larger array is fine
            assert wt.dtype == torch.float32 and wt.shape == (W, N) and (N <= 1 or wt.stride(1) == 1)
            d.weights = wt.data_ptr()
            d.weights_stride = wt.stride(0) if W > 1 else 0
        self.out = {}
        if want_event_outputs:
            names = self.EVENT_OUTPUTS if want_event_outputs is True else tuple(want_event_outputs)
            for k in names:
                assert k in self.EVENT_OUTPUTS, k
                dt = torch.int32 if k in ("njet", "argmax") else torch.float32
                if out_into is not None:
                    whole = out_into[k]
                    assert whole.dtype == dt and whole.is_contiguous() and whole.shape[0] == V
                    self.out[k] = whole[:, out_col: out_col + N]
                    d.out_stride = whole.shape[1]
                    setattr(d, "out_" + k, whole.data_ptr() + 4 * out_col)
                else:
                    self.out[k] = torch.empty((V, N), dtype=dt, device=dev)
                    setattr(d, "out_" + k, self.out[k].data_ptr())
        if want_mask:
            self.out["jet_mask"] = torch.zeros((V, inp.jets.pt.numel()), dtype=torch.uint8, device=dev)
            d.out_jet_mask = self.out["jet_mask"].data_ptr()
        self.prefix, self.spv = hist_layout(inp.hists, inp.axes)
        if want_hists:
            for o, name in enumerate(OBSERVABLES):
                if name in inp.hists:
                    d.axis_edges[o] = inp.axes[name].data_ptr()
                    d.axis_nbins[o] = inp.axes[name].numel() - 1
            self.out["hist_sumw"] = torch.zeros(V * W * self.spv, dtype=torch.float32, device=dev)
            d.hist_sumw = self.out["hist_sumw"].data_ptr()
            if want_counts:
                self.out["hist_counts"] = torch.zeros(V * self.spv, dtype=torch.int64, device=dev)
                d.hist_counts = self.out["hist_counts"].data_ptr()
            if want_sumw2:
                self.out["hist_sumw2"] = torch.zeros(V * W * self.spv, dtype=torch.float32, device=dev)
                d.hist_sumw2 = self.out["hist_sumw2"].data_ptr()
        if inp.evw is not None:
            for k in ("x", "edges", "table"):
                t = inp.evw[k]
                assert t.is_cuda and t.is_contiguous() and t.dtype == torch.float32, k
            assert inp.evw["x"].numel() == N and inp.evw["table"].numel() == inp.evw["edges"].numel() - 1
            self._keep = inp.evw
            d.evw_x, d.evw_edges = inp.evw["x"].data_ptr(), inp.evw["edges"].data_ptr()
            d.evw_nbins, d.evw_table = inp.evw["table"].numel(), inp.evw["table"].data_ptr()
        for k, v in (tune or {}).items():
            setattr(d, "tune_" + k, int(v))
        self.desc = d
        nbytes = lib().hepk_chain_workspace_bytes(C.byref(d))
        self.workspace = torch.empty(max(nbytes, 8), dtype=torch.uint8, device=dev)
        self.V, self.W = V, W

    def zero_hists(self):
        for k in ("hist_sumw", "hist_sumw2", "hist_counts"):
            if k in self.out:
                self.out[k].zero_()

    def zero_hists_on(self, stream):
        with torch.cuda.stream(stream):
            self.zero_hists()

    def run(self, stream=None):
        _check(lib().hepk_analysis_chain(C.byref(self.desc), C.c_void_p(self.workspace.data_ptr()),
                                         C.c_size_t(self.workspace.numel()), _stream(stream)), "analysis_chain")
        return self.out

    def hist_view(self, name):
        """(sumw [V][W][nbins+2], counts [V][nbins+2]) views of one observable's histograms."""
        nb2 = self.inp.axes[name].numel() - 1 + 2
        p, V, W, spv = self.prefix[name], self.V, self.W, self.spv
        sw = self.out["hist_sumw"].view(V, W * spv)[:, W * p: W * p + W * nb2].reshape(V, W, nb2)
        ct = self.out["hist_counts"].view(V, spv)[:, p: p + nb2] if "hist_counts" in self.out else None
        return sw, ct


def analysis_chain(inp: ChainInputs, stream=None, **plan_kwargs):
    """One-shot hepk_analysis_chain: builds the plan, runs it, returns (outputs dict, plan)."""
    plan = ChainPlan(inp, **plan_kwargs)
    plan.run(stream)
    return plan.out, plan


# ------------------------------------------------------------------------------------------ host streaming
class HostChainPlan:
    """hepk_analysis_chain_host on a hepgen-style workload held in PINNED host memory.

    All inputs and outputs are host tensors; the C library does the host->device copies, the kernels and the
    device->host copies.  `wl` needs the attributes of hepgen.Workload (numpy arrays)."""

    def __init__(self, wl, batch_events, want_event_outputs=True, want_hists=True, want_counts=True, want_sumw2=False,
                 evw=None, device="cuda"):
        """evw: optional dict(x, edges, table) of numpy float32 arrays (the event-weight lookup)."""
        pin = lambda a: torch.from_numpy(a).pin_memory()
        self.keep = []
        self.h2d_bytes = 0
        d = ChainDesc()
        N = wl.n_events
        d.n_events = N

        def coll(s, c, with_mass):
            if c is None:
                return
            off = pin(c.offsets)
            self.keep.append(off)
            s.offsets, s.content_base, s.n_objects = off.data_ptr(), 0, c.pt.shape[0]
            self.h2d_bytes += off.numel() * 8
            for name in ("pt", "eta", "phi") + (("mass",) if with_mass else ()):
                t = pin(getattr(c, name))
                self.keep.append(t)
                setattr(s, name, t.data_ptr())
                self.h2d_bytes += t.numel() * 4
        coll(d.jets, wl.jets, True)
        coll(d.muons, wl.muons, False)
        coll(d.electrons, wl.electrons, False)
        d.jet_pt_min, d.jet_abs_eta_max = wl.cuts["jet_pt_min"], wl.cuts["jet_abs_eta_max"]
        d.lep_pt_min, d.dr_max = wl.cuts["lep_pt_min"], wl.cuts["dr_max"]
        V = 1
        if wl.calib is not None:
            pe, ee, tb = pin(wl.calib["pt_edges"]), pin(wl.calib["eta_edges"]), pin(wl.calib["table"])
            self.keep += [pe, ee, tb]
            d.calib_pt_edges, d.calib_npt = pe.data_ptr(), pe.numel() - 1
            d.calib_eta_edges, d.calib_neta = ee.data_ptr(), ee.numel() - 1
            d.calib_table = tb.data_ptr()
            V = len(wl.calib["scales"])
            for i, s in enumerate(wl.calib["scales"]):
                d.calib_scales[i] = float(s)
        W = int(wl.weights.shape[0])
        d.n_variants, d.n_wvar = V, W
        wt = pin(wl.weights)
        self.keep.append(wt)
        d.weights = wt.data_ptr()
        self.h2d_bytes += wt.numel() * 4
        self.out = {}
        self.d2h_bytes = 0
        if want_event_outputs:
            names = ChainPlan.EVENT_OUTPUTS if want_event_outputs is True else tuple(want_event_outputs)
            for k in names:
                dt = torch.int32 if k in ("njet", "argmax") else torch.float32
                self.out[k] = torch.empty((V, N), dtype=dt).pin_memory()
                setattr(d, "out_" + k, self.out[k].data_ptr())
                self.d2h_bytes += self.out[k].numel() * 4
        axes = {k: pin(v) for k, v in wl.axes.items()}
        self.axes = axes
        self.prefix, self.spv = hist_layout(wl.hists, axes)
        if want_hists:
            for o, name in enumerate(OBSERVABLES):
                if name in wl.hists:
                    d.axis_edges[o] = axes[name].data_ptr()
                    d.axis_nbins[o] = axes[name].numel() - 1
            self.out["hist_sumw"] = torch.zeros(V * W * self.spv, dtype=torch.float32).pin_memory()
            d.hist_sumw = self.out["hist_sumw"].data_ptr()
            self.d2h_bytes += self.out["hist_sumw"].numel() * 4
            if want_counts:
                self.out["hist_counts"] = torch.zeros(V * self.spv, dtype=torch.int64).pin_memory()
                d.hist_counts = self.out["hist_counts"].data_ptr()
                self.d2h_bytes += self.out["hist_counts"].numel() * 8
            if want_sumw2:
                self.out["hist_sumw2"] = torch.zeros(V * W * self.spv, dtype=torch.float32).pin_memory()
                d.hist_sumw2 = self.out["hist_sumw2"].data_ptr()
                self.d2h_bytes += self.out["hist_sumw2"].numel() * 4
        if evw is not None:
            ex, ee, et = (pin(evw[k]) for k in ("x", "edges", "table"))
            self.keep += [ex, ee, et]
            d.evw_x, d.evw_edges, d.evw_nbins, d.evw_table = ex.data_ptr(), ee.data_ptr(), et.numel(), et.data_ptr()
            self.h2d_bytes += ex.numel() * 4
        self.desc, self.V, self.W = d, V, W
        self.batch_events = int(batch_events)
        nbytes = lib().hepk_chain_host_workspace_bytes(C.byref(d), C.c_int64(self.batch_events))
        if nbytes == 0:
            raise HepkError("hepk_chain_host_workspace_bytes returned 0 (bad descriptor)")
        self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=device)

    def zero_hists(self):
        for k in ("hist_sumw", "hist_sumw2", "hist_counts"):
            if k in self.out:
                self.out[k].zero_()

    def run(self, overlap=True, stream=None):
        _check(lib().hepk_analysis_chain_host(C.byref(self.desc), C.c_int64(self.batch_events), C.c_int32(1 if overlap else 0),
                                              C.c_void_p(self.workspace.data_ptr()), C.c_size_t(self.workspace.numel()),
                                              _stream(stream)), "analysis_chain_host")
        return self.out

    def hist_view(self, name):
        nb2 = self.axes[name].numel() - 1 + 2
        p, V, W, spv = self.prefix[name], self.V, self.W, self.spv
        sw = self.out["hist_sumw"].view(V, W * spv)[:, W * p: W * p + W * nb2].reshape(V, W, nb2)
        ct = self.out["hist_counts"].view(V, spv)[:, p: p + nb2] if "hist_counts" in self.out else None
        return sw, ct
