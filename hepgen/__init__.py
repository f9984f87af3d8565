"""Seeded synthetic collider events (jagged arrays) for the BASELINE.json configs.

This module is the ONLY code shared by the CPU oracle (`oracle/`) and the CUDA
path (`paper_1906_06242_b200/`).  It holds no arithmetic of the method: it only
draws random numbers and lays them out as the paper's jagged arrays
(section II: "a contiguous offset array of size N+1 and a
contiguous data array of size M for each particle feature").

The events stand in for the CMS Open Data top-pair workload the paper measures
on, which is not available here.  Recipe: SURVEY.md section 8(d),
restated in DESIGN.md "Input recipe".
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

__all__ = ["CONFIGS", "Workload", "Collection", "generate", "concat", "hist_axes", "calibration_table",
           "OBSERVABLES"]

# Fixed observable order used by the fused chain on both sides (names only; no arithmetic here).
OBSERVABLES = ("njet", "ht", "maxpt", "minpt", "mjj", "subpt")

# Axis ranges, 100 bins each.  HT [0,1000] and leading-jet pt [0,500] are from BASELINE.json
# configs 0/1; the other four are the SURVEY.md 8(c7) proposal for config 4's "30 variables".
_AXIS_RANGE = {
    "njet": (0.0, 50.0),
    "ht": (0.0, 1000.0),
    "maxpt": (0.0, 500.0),
    "minpt": (0.0, 200.0),
    "mjj": (0.0, 1000.0),
    "subpt": (0.0, 300.0),
}

# BASELINE.json "configs" 0..4.
CONFIGS = {
    0: dict(n_events=10_000, seed=0, lam_jet=5.0, cap_jet=20, tail=False, lam_mu=1.0, lam_el=None,
            n_wvar=1, calib=False, hists=("ht",)),
    1: dict(n_events=1_000_000, seed=1, lam_jet=5.0, cap_jet=20, tail=False, lam_mu=1.0, lam_el=None,
            n_wvar=1, calib=False, hists=("ht", "maxpt")),
    2: dict(n_events=10_000_000, seed=2, lam_jet=8.0, cap_jet=40, tail=True, lam_mu=1.5, lam_el=1.0,
            n_wvar=1, calib=False, hists=("ht", "maxpt")),
    3: dict(n_events=10_000_000, seed=3, lam_jet=8.0, cap_jet=40, tail=True, lam_mu=1.5, lam_el=1.0,
            n_wvar=1, calib=True, hists=("ht", "maxpt")),
    4: dict(n_events=5_000_000, seed=4, lam_jet=8.0, cap_jet=40, tail=True, lam_mu=1.5, lam_el=1.0,
            n_wvar=10, calib=True, hists=OBSERVABLES, n_batches=10),
}

CUTS = dict(jet_pt_min=30.0, jet_abs_eta_max=2.4, lep_pt_min=20.0, dr_max=0.4)
SCALES = (1.0, 1.02, 0.98, 1.05, 0.95)   # BASELINE.json config 3: table x {1, 1+-0.02, 1+-0.05}
LEPTON_CAP = 6
MUON_MASS = 0.1057
ELECTRON_MASS = 0.000511


@dataclass
class Collection:
    offsets: np.ndarray   # int64 [n_events+1]
    pt: np.ndarray        # float32 [n_objects]
    eta: np.ndarray
    phi: np.ndarray
    mass: np.ndarray

    @property
    def n_objects(self) -> int:
        return int(self.pt.shape[0])


@dataclass
class Workload:
    config: int
    n_events: int
    seed: int
    batch: int
    jets: Collection
    muons: Collection
    electrons: Collection | None
    weights: np.ndarray                 # float32 [n_wvar][n_events]
    cuts: dict
    hists: tuple                        # names of histogrammed observables, in OBSERVABLES order
    axes: dict                          # name -> float32 edges [nbins+1]
    calib: dict | None = None           # pt_edges, eta_edges, table [npt][neta], scales
    meta: dict = field(default_factory=dict)


def hist_axes(names, nbins: int = 100) -> dict:
    """float32(linspace(lo, hi, nbins+1)) per observable, generated once and given to both sides."""
    return {n: np.linspace(_AXIS_RANGE[n][0], _AXIS_RANGE[n][1], nbins + 1).astype(np.float32)
            for n in names}


def calibration_table(rng: np.random.Generator) -> dict:
    """BASELINE.json config 3: 50 log-spaced pt bins 20..3000 GeV x 20 uniform eta bins, U(0.9,1.1)."""
    return dict(
        pt_edges=np.geomspace(20.0, 3000.0, 51).astype(np.float32),
        eta_edges=np.linspace(-2.5, 2.5, 21).astype(np.float32),
        table=rng.uniform(0.9, 1.1, size=(50, 20)).astype(np.float32),
        scales=np.asarray(SCALES, dtype=np.float32),
    )


def _collection(rng, counts, mass_kind) -> Collection:
    offsets = np.zeros(counts.shape[0] + 1, dtype=np.int64)
    np.cumsum(counts, out=offsets[1:])
    m = int(offsets[-1])
    pt = (20.0 + rng.exponential(30.0, m)).astype(np.float32)
    eta = rng.uniform(-2.5, 2.5, m).astype(np.float32)
    phi = rng.uniform(-math.pi, math.pi, m).astype(np.float32)
    if mass_kind == "jet":
        mass = rng.exponential(10.0, m).astype(np.float32)
    else:
        mass = np.full(m, mass_kind, dtype=np.float32)
    return Collection(offsets, pt, eta, phi, mass)


def generate(config: int, n_events: int | None = None, seed: int | None = None, batch: int = 0,
             **overrides) -> Workload:
    """Draw one batch of events for BASELINE.json config `config`.

    Fixed draw order (determinism is what matters: parity is always CUDA-vs-oracle on the same
    arrays): jet counts, tail flags+counts, muon counts, electron counts, jets (pt, eta, phi,
    mass), muons, electrons, weights, calibration table.
    """
    cfg = dict(CONFIGS[config])
    cfg.update(overrides)
    n = int(cfg["n_events"] if n_events is None else n_events)
    seed = int(cfg["seed"] if seed is None else seed)
    rng = np.random.Generator(np.random.PCG64(np.random.SeedSequence([seed, batch])))

    n_jet = np.minimum(rng.poisson(cfg["lam_jet"], n), cfg["cap_jet"]).astype(np.int64)
    if cfg["tail"]:
        # "1% heavy tail at 30-40 jets": 1% of events get a uniform integer count in [30, 40].
        tail = rng.random(n) < 0.01
        tail_counts = rng.integers(30, 41, n)
        n_jet[tail] = tail_counts[tail]
    n_mu = np.minimum(rng.poisson(cfg["lam_mu"], n), LEPTON_CAP).astype(np.int64)
    n_el = None
    if cfg["lam_el"] is not None:
        n_el = np.minimum(rng.poisson(cfg["lam_el"], n), LEPTON_CAP).astype(np.int64)

    jets = _collection(rng, n_jet, "jet")
    muons = _collection(rng, n_mu, MUON_MASS)
    electrons = _collection(rng, n_el, ELECTRON_MASS) if n_el is not None else None
    weights = rng.normal(1.0, 0.1, size=(cfg["n_wvar"], n)).astype(np.float32)
    calib = calibration_table(rng) if cfg["calib"] else None

    return Workload(config=config, n_events=n, seed=seed, batch=batch, jets=jets, muons=muons,
                    electrons=electrons, weights=weights, cuts=dict(CUTS), hists=tuple(cfg["hists"]),
                    axes=hist_axes(cfg["hists"]), calib=calib,
                    meta=dict(lam_jet=cfg["lam_jet"], cap_jet=cfg["cap_jet"], tail=cfg["tail"]))


def concat(workloads) -> Workload:
    """Several batches of one config laid end to end as ONE workload (offsets shifted, columns concatenated): the
    host-resident input of a streamed run (BASELINE.json config 4: 10 batches of 5 M events).  Layout only."""
    first = workloads[0]

    def cat(get):
        cols = [get(w) for w in workloads]
        if cols[0] is None:
            return None
        offs, base = [cols[0].offsets], int(cols[0].offsets[-1])
        for c in cols[1:]:
            offs.append(c.offsets[1:] + base)
            base += int(c.offsets[-1])
        return Collection(np.concatenate(offs), *(np.concatenate([getattr(c, k) for c in cols]) for k in ("pt", "eta", "phi", "mass")))

    return Workload(config=first.config, n_events=sum(w.n_events for w in workloads), seed=first.seed, batch=first.batch,
                    jets=cat(lambda w: w.jets), muons=cat(lambda w: w.muons), electrons=cat(lambda w: w.electrons),
                    weights=np.ascontiguousarray(np.concatenate([w.weights for w in workloads], axis=1)), cuts=dict(first.cuts),
                    hists=first.hists, axes=first.axes, calib=first.calib, meta=dict(first.meta))
