/*
 * hepo.h — CPU ORACLE for the columnar HEP kernels of arXiv:1906.06242.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this library.  It shares no code with the CUDA
 * path (paper_1906_06242_b200/, include/hepk.h) and neither includes the other.
 *
 * Every function is a plain per-event loop in the paper's own order (Listing 1,
 * loop over events, skip masked rows, loop over the event's particles
 * between offsets[iev] and offsets[iev+1], skip masked particles).  All pointers are HOST
 * pointers.  Return value: 0 = OK, -1 = invalid argument.
 *
 * Two result classes:
 *   exact class     masks, counts, indices, bin slots, max/min: float32 expression tree,
 *                   one IEEE round-to-nearest op per node, no FMA contraction
 *                   (build with -ffp-contract=off, no -ffast-math);
 *   tolerance class sums, masses, weighted bins: float64 accumulation from the float32
 *                   inputs, rounded once to float32.
 *
 * Pinned by tests/test_oracle_*.py (closed forms, brute force, numpy special cases,
 * invariants).  Conventions the paper is silent on (empty-event sentinels, out-of-range lookup
 * policy, NaN routing, electron cut, the 30 variables of config 4) are DESIGN.md readings and
 * are marked "parity unpinned" there and below.
 */
#ifndef HEPO_H
#define HEPO_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* PAPER.md:L132 "object selection based on cuts on objects: jet, lepton selection based on pT, eta".
 * out[i] = (pt[i] > pt_min) && (|eta[i]| < abs_eta_max); eta == NULL drops the second term. */
int32_t hepo_select_mask(const float* pt, const float* eta, int64_t n, float pt_min, float abs_eta_max,
                         uint8_t* out_mask);

/* Listing 1 and the generic kernels sum/max/min_in_offsets.
 * Element for global index g is data[g - content_base].  mask_rows / mask_content may be NULL (all true).
 * Outputs are overwritten for every event.  Empty values: sum 0.0f, count 0, max -inf, min +inf,
 * argmax -1 (parity unpinned: the paper does not say). */
int32_t hepo_segmented_reduce_sum(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out);
int32_t hepo_segmented_reduce_max(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out);
int32_t hepo_segmented_reduce_min(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out);
int32_t hepo_segmented_reduce_count(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                    const uint8_t* mask_rows, const uint8_t* mask_content, int32_t* out);
int32_t hepo_segmented_reduce_argmax(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                     const uint8_t* mask_rows, const uint8_t* mask_content, int32_t* out);

/* mask_deltar_first: out_matched[j] = 1 iff object j of collection 1 is selected and some
 * selected object of collection 2 in the same event has dR^2 = deta^2 + dphi^2 < dr_max^2. */
int32_t hepo_deltar_mask(const float* eta1, const float* phi1, const int64_t* offsets1, int64_t base1, const uint8_t* sel1,
                         const float* eta2, const float* phi2, const int64_t* offsets2, int64_t base2, const uint8_t* sel2,
                         int64_t n_events, float dr_max, uint8_t* out_matched);

/* Invariant mass of the two highest-pt selected particles per event (coordinates pT, eta, phi, M:
 * PAPER.md:L11; candidate-mass step: PAPER.md:L136; "first two ... ordered by pT": PAPER.md:L105). */
int32_t hepo_pair_invmass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_content,
                          float* out_mass, int32_t* out_i1, int32_t* out_i2);

/* get_bin_contents: out[i] = table[bin_x(x[i]) * ny + bin_y(y[i])]; y == NULL -> 1-D. */
int32_t hepo_lookup_binned(const float* x, const float* y, int64_t n,
                           const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                           const float* table, float* out);

/* fill_histogram.  sumw/counts have nbins+2 slots [under, bins..., over] and accumulate. */
int32_t hepo_fill_histogram(const float* data, const float* weights, int64_t n,
                            const float* edges, int32_t nbins, float* sumw, int64_t* counts);

/* fill_histogram with the sum of squared weights: sumw2[slot] += w*w, float64
 * accumulation of the float32 weight's square, rounded once; weights == NULL: w = 1 (sumw2 == sumw == counts).
 * sumw, sumw2, counts each nullable, all accumulate. */
int32_t hepo_fill_histogram_w2(const float* data, const float* weights, int64_t n,
                               const float* edges, int32_t nbins, float* sumw, float* sumw2, int64_t* counts);

/* Event weight from a histogram lookup ("event weight computation based on
 * histogram lookups: pileup, lepton efficiency corrections"): w_out[e] = w_in[e] * table[B(x[e])], one float32
 * multiply, B the clamped bin of hepo_lookup_binned; w_in == NULL: w_in = 1. */
int32_t hepo_event_weight_lookup(const float* w_in, const float* x, int64_t n,
                                 const float* edges, int32_t nbins, const float* table, float* w_out);

/* ---- fused chain (PAPER.md:L129-139 for the analysis steps) ---- */
enum { HEPO_OBS_NJET = 0, HEPO_OBS_HT, HEPO_OBS_MAXPT, HEPO_OBS_MINPT, HEPO_OBS_MJJ, HEPO_OBS_SUBPT, HEPO_N_OBS };

typedef struct {
    const int64_t* offsets;   /* [n_events+1]; NULL = collection absent */
    int64_t content_base;
    int64_t n_objects;
    const float* pt;
    const float* eta;
    const float* phi;
    const float* mass;        /* only read for jets */
} hepo_collection;

typedef struct {
    int64_t n_events;
    hepo_collection jets, muons, electrons;
    float jet_pt_min, jet_abs_eta_max, lep_pt_min, dr_max;
    /* calibration; calib_table == NULL -> none and n_variants must be 1 */
    const float* calib_pt_edges;  int32_t calib_npt;
    const float* calib_eta_edges; int32_t calib_neta;
    const float* calib_table;     /* [npt][neta] */
    const float* calib_scales;    /* [n_variants] */
    int32_t n_variants;
    int32_t n_wvar;
    const float* weights;         /* [n_wvar][n_events]; NULL -> weight 1 */
    const float* axis_edges[HEPO_N_OBS];   /* NULL -> observable not histogrammed */
    int32_t axis_nbins[HEPO_N_OBS];
    /* per-event outputs, each [n_variants][n_events], all nullable */
    int32_t* out_njet; int32_t* out_argmax;
    float* out_ht; float* out_maxpt; float* out_minpt; float* out_mjj; float* out_subpt;
    uint8_t* out_jet_mask;        /* [n_variants][jets.n_objects] clean-jet mask */
    /* histograms (accumulate): sumw [V][active obs o][n_wvar][nbins_o+2]; counts [V][active obs o][nbins_o+2] */
    float* hist_sumw; int64_t* hist_counts;
    /* optional per-event weight factor from a 1-D lookup on a per-event column,
     * factor[e] = evw_table[B(evw_x[e])] (clamped bin of hepo_lookup_binned), multiplied into every weight column
     * with ONE float32 multiply before the fill (weights NULL: 1.0f * factor).  evw_table == NULL: none. */
    const float* evw_x;           /* [n_events] */
    const float* evw_edges;       /* [evw_nbins+1] */
    int32_t evw_nbins;
    const float* evw_table;       /* [evw_nbins] */
    /* sum of squared (final) weights per slot, layout of hist_sumw, accumulates; NULL = not wanted */
    float* hist_sumw2;
} hepo_chain_desc;

int32_t hepo_analysis_chain(const hepo_chain_desc* d);
size_t  hepo_chain_desc_size(void);

/* The same computation on n_threads host threads (<= 0: all; OpenMP `parallel for` over contiguous event blocks,
 * PAPER.md:L66-68 `prange`), per-thread private histograms merged in thread order.  TIMING BASELINE for bench.py;
 * hepo_analysis_chain stays the checker.  Per-event outputs and counts equal the single-thread results exactly,
 * sumw / sumw2 up to the order of the float64 additions. */
int32_t hepo_analysis_chain_omp(const hepo_chain_desc* d, int32_t n_threads);
int32_t hepo_omp_max_threads(void);

/* ---- the remaining generic kernels of the paper's list ------------------------------
 *
 * get_in_offsets ("given jagged data with offsets, retrieves the n-th elements for all rows ...
 * to create a contiguous array of e.g. the leading jet pT").  out[e] = the index-th element of row e, counting
 * only elements with mask_content set (mask_content == NULL: every element); rows with mask_rows clear or with
 * fewer than index+1 counted elements get `fill`.  index >= 0.  (Counting through the content mask and the
 * fill value are readings: the paper says neither.  parity unpinned for those two conventions.) */
int32_t hepo_get_in_offsets(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index, float fill,
                            float* out);

/* set_in_offsets ("as above, but sets the n-th element to a value ... to selectively mask
 * objects in a collection").  data[position of the index-th counted element of row e] = values ? values[e]
 * : value, for rows with mask_rows set (or NULL) that have that element; everything else is left untouched. */
int32_t hepo_set_in_offsets(float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index,
                            const float* values, float value);

/* select_opposite_sign_muons ("given a collection of objects with charge (i.e. muons),
 * masks all but the first two objects ordered by pT which are of opposite charge").  Per event, over the
 * objects with mask_content set: the leading object by pt (first index among equal pt) and the highest-pt
 * object whose charge has the opposite sign (charge * charge_lead < 0; first index among equal pt) get 1,
 * everything else 0; an event without such a pair (or with mask_rows clear) gets all 0.  NaN pt is skipped. */
int32_t hepo_select_opposite_sign(const float* pt, const int32_t* charge, const int64_t* offsets, int64_t n_events,
                                  int64_t content_base, const uint8_t* mask_rows, const uint8_t* mask_content,
                                  uint8_t* out_mask);

/* ---- lookup / histogram variants ------------------------------------------------------
 *
 * Linear-interpolated correction ("systematic corrections based on linear interpolations").
 * Knots xs[0..nk) ascending with values ys[0..nk):  out = ys[b] + (x - xs[b]) * (ys[b+1] - ys[b]) / (xs[b+1] - xs[b])
 * for xs[b] <= x < xs[b+1], evaluated in float64 and rounded once; x <= xs[0] -> ys[0], x >= xs[nk-1] -> ys[nk-1]
 * (constant extrapolation), NaN -> NaN.  Tolerance class.  nk >= 2. */
int32_t hepo_lookup_interp(const float* x, int64_t n, const float* xs, const float* ys, int32_t nk, float* out);

/* Two-dimensional weighted histogram ("Extension to multidimensional histograms is
 * straightforward").  Slot = sx * (ny + 2) + sy with sx, sy the one-dimensional slots of hepo_fill_histogram
 * (under/overflow kept per axis, NaN -> overflow); sumw [nx+2][ny+2] accumulates in float64 per call and is added
 * to the float32 array; counts int64 [nx+2][ny+2]. */
int32_t hepo_fill_histogram_2d(const float* x, const float* y, const float* weights, int64_t n,
                               const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                               float* sumw, int64_t* counts);
int32_t hepo_fill_histogram_2d_w2(const float* x, const float* y, const float* weights, int64_t n,
                                  const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                                  float* sumw, float* sumw2, int64_t* counts);

/* ---- jet-triplet candidate -------------------------------------------------------------
 *
 * PAPER.md:L136 "high-level variable reconstruction: top quark candidate from jet triplet with invariant mass
 * closest to M = 172 GeV".  Per event, over all triplets i < j < k of the objects with mask_content set (local
 * indices): M_ijk = sqrt(max(0, (E_i+E_j+E_k)^2 - |p_i+p_j+p_k|^2)) from the four-vectors of hepo_pair_invmass
 * (float64), and the triplet minimising |M_ijk - target| is kept; among equal distances the lexicographically
 * first (i, j, k).  out_mass = (float)M of that triplet, out_idx[3*e..] its local indices; fewer than three
 * selected objects (or mask_rows clear): mass 0.0f, indices -1.  (The formula, the tie rule and the "< 3" value
 * are readings: the paper gives one phrase.)  Tolerance class; which triplet wins is decided in float64 here. */
int32_t hepo_triplet_mass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base,
                          const uint8_t* mask_rows, const uint8_t* mask_content, float target,
                          float* out_mass, int32_t* out_idx);

/* Precondition check of a jagged layout ("a contiguous offsets array of size N+1" indexing
 * contiguous data arrays): returns in *n_bad the number of violations among
 *   offsets[0] >= content_base,  offsets[e] <= offsets[e+1] for every e,  offsets[n_events] - content_base <= n_objects. */
int32_t hepo_validate_offsets(const int64_t* offsets, int64_t n_events, int64_t content_base, int64_t n_objects, int64_t* n_bad);

#ifdef __cplusplus
}
#endif
#endif
