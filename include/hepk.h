/*
 * hepk.h — C ABI of libhepk.so: B200-native (sm_100a) columnar HEP analysis kernels.
 *
 * The operations are the data-parallel hot path of "Processing Columnar Collider Data with
 * GPU-Accelerated Kernels" (arXiv:1906.06242).  Citations are PAPER.md:L<line> of the paper text.
 *
 * Data model (section II): N events with M particles in total are stored as a
 * contiguous int64 `offsets` array of N+1 non-decreasing entries plus one contiguous float32
 * array of M entries per particle feature (pt, eta, phi, mass).  Several collections (jets,
 * muons, electrons) each carry their own offsets.
 *
 * Conventions for every entry point unless stated otherwise
 *   - Pointers are CALLER-OWNED DEVICE pointers (cudaMalloc / torch CUDA tensors).  The library
 *     never allocates or frees user-visible memory; scratch comes from a caller workspace.
 *     Pointers marked HOST are host pointers.
 *   - `stream` is a cudaStream_t passed as void* (NULL = legacy default stream).  Calls enqueue work
 *     and return; there is no implicit synchronisation.
 *   - Return value: HEPK_OK (0), HEPK_ERR_INVALID (-1: NULL required pointer, negative size, bad
 *     enum), HEPK_ERR_UNSUPPORTED (-2: size beyond what the kernels support), HEPK_ERR_CUDA (-3:
 *     a CUDA runtime call failed).  hepk_last_error() returns a thread-local message.
 *     No exceptions, no abort.  Arguments are validated on the host only (pointers and sizes);
 *     monotone offsets are a precondition.
 *   - Jagged convention: the element for global particle index g lives at col[g - content_base];
 *     content_base is normally offsets[0] = 0, and lets a streamed batch pass a slice of a global
 *     offsets array without rebasing it.
 *   - Masks are uint8_t (0 / non-zero), numpy-bool compatible; a NULL mask means "all true"
 *     (boolean masks for events and particles).
 *   - Reduction outputs are OVERWRITTEN for every event; histogram outputs ACCUMULATE (the
 *     caller zeroes them), because the paper's histogram contents are in/out.
 *   - Arithmetic contract: masks, counts, indices, bin slots, max/min are evaluated in
 *     float32 with one IEEE round-to-nearest operation per node and no FMA contraction, so they
 *     are bit-exact against the CPU oracle; sums, masses and weighted bins are float32 results
 *     within 1e-5 relative (1e-6 absolute floor) of the exactly rounded value.
 */
#ifndef HEPK_H
#define HEPK_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define HEPK_OK               0
#define HEPK_ERR_INVALID     (-1)
#define HEPK_ERR_UNSUPPORTED (-2)
#define HEPK_ERR_CUDA        (-3)

#define HEPK_MAX_VARIANTS 64
#define HEPK_MAX_WVAR     16

/* Library version (major*10000 + minor*100 + patch). */
int32_t hepk_version(void);
/* Thread-local message of the last failing call on this thread ("" if none).  HOST string. */
const char* hepk_last_error(void);

/* ---------------------------------------------------------------------------------------------
 * Object selection ("object selection based on cuts on objects: jet, lepton selection
 * based on pT, eta").
 *   out_mask[i] = (pt[i] > pt_min) && (fabsf(eta[i]) < abs_eta_max)     for i in [0, n)
 * eta == NULL drops the eta term.  Both inequalities are strict; NaN compares false.
 * pt, eta: float32[n]; out_mask: uint8[n].  Any 4-byte aligned pointers are accepted; 16-byte aligned
 * pointers take the 128-bit vector path. */
int32_t hepk_select_mask(const float* pt, const float* eta, int64_t n,
                         float pt_min, float abs_eta_max, uint8_t* out_mask, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Segmented (per-event) reductions: Listing 1 "sum_ht" generalised to the
 * kernels sum_in_offsets / max_in_offsets / min_in_offsets; counting objects
 * "by summing masks"; argmax for leading-object quantities.
 *   for each event e: if mask_rows && !mask_rows[e] -> empty value; else reduce data[g - content_base]
 *   over g in [offsets[e], offsets[e+1]) with mask_content[g - content_base] != 0.
 * data: float32[M]; offsets: int64[n_events+1]; mask_rows: uint8[n_events] or NULL;
 * mask_content: uint8[M] or NULL.
 * out: float32[n_events] for sum / max / min; int32[n_events] for count / argmax.
 * Empty values: sum 0.0f, count 0, max -inf, min +inf, argmax -1.  argmax is the index LOCAL to
 * the event (g - offsets[e]); equal values: the smallest index wins; NaN elements are skipped by
 * max / min / argmax and propagated by sum.  count ignores `data` (may be NULL).
 * variant: 0 = auto (= 2), 1 = warp-per-event (lanes stride over the event's particles, shuffle
 * reduction), 2 = block-per-tile (every warp of a persistent block streams tiles of 64 events through
 * its own double-buffered shared-memory stage with TMA bulk copies; one lane per event, the whole warp
 * for the elements of an event beyond the 16th).  count / max / min / argmax are bitwise identical
 * across variants; sums are accumulated in float64 and rounded once (tolerance class).  The calls
 * enqueue and return (nothing is read back from the device). */
#define HEPK_VARIANT_AUTO            0
#define HEPK_VARIANT_WARP_PER_EVENT  1
#define HEPK_VARIANT_BLOCK_PER_TILE  2
int32_t hepk_segmented_reduce_sum(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content,
                                  float* out, int32_t variant, void* stream);
int32_t hepk_segmented_reduce_max(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content,
                                  float* out, int32_t variant, void* stream);
int32_t hepk_segmented_reduce_min(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content,
                                  float* out, int32_t variant, void* stream);
int32_t hepk_segmented_reduce_count(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                    const uint8_t* mask_rows, const uint8_t* mask_content,
                                    int32_t* out, int32_t variant, void* stream);
int32_t hepk_segmented_reduce_argmax(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                     const uint8_t* mask_rows, const uint8_t* mask_content,
                                     int32_t* out, int32_t variant, void* stream);

/* ---------------------------------------------------------------------------------------------
 * dR matching, mask_deltar_first ("given two collections of objects, masks all objects
 * in the first collection that are closer than a predefined value in dR^2 = deta^2 + dphi^2 to an
 * object in the second collection"; nested per-event loop PAPER.md:L112).
 *   out_matched[j] = 1 iff (sel1 == NULL || sel1[j]) and some m in the same event with
 *   (sel2 == NULL || sel2[m]) has dr2(j, m) < dr_max*dr_max (float32 product, strict <), else 0.
 *   dr2: deta = eta1-eta2; dphi = phi1-phi2; if (dphi > PI_F) dphi -= 2PI_F; else if (dphi <= -PI_F)
 *   dphi += 2PI_F; dr2 = deta*deta + dphi*dphi — float32, one rounding per operation.
 * eta1, phi1: float32[M1]; offsets1: int64[n_events+1]; sel1: uint8[M1] or NULL; likewise collection 2.
 * out_matched: uint8[M1], written for every object of collection 1 inside the event range.
 * The cleaned-jet mask is formed by the caller: clean = sel1 & !matched. */
int32_t hepk_deltar_mask(const float* eta1, const float* phi1, const int64_t* offsets1, int64_t base1, const uint8_t* sel1,
                         const float* eta2, const float* phi2, const int64_t* offsets2, int64_t base2, const uint8_t* sel2,
                         int64_t n_events, float dr_max, uint8_t* out_matched, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Leading-pair invariant mass (particle coordinates pT, eta, phi, M: PAPER.md:L11; candidate mass
 * from jets: PAPER.md:L136; "first two jets ordered by pT": PAPER.md:L105).
 *   i1 = argmax of pt over selected particles of the event (rule of segmented_reduce_argmax),
 *   i2 = argmax over the selected particles excluding i1;
 *   out_mass[e] = sqrt(max(0, (E1+E2)^2 - |p1+p2|^2)) with px = pt cos(phi), py = pt sin(phi),
 *   pz = pt sinh(eta), E = sqrt(pt^2 cosh^2(eta) + m^2); fewer than two selected -> 0.0f, missing index -1.
 * pt, eta, phi, mass: float32[M]; mask_content: uint8[M] or NULL; out_mass: float32[n_events];
 * out_i1, out_i2: int32[n_events] local indices, each may be NULL. */
int32_t hepk_pair_invmass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_content,
                          float* out_mass, int32_t* out_i1, int32_t* out_i2, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Binned lookup, get_bin_contents ("given a data array and a lookup histogram, retrieves
 * the bin contents corresponding to each data array element"; jet energy corrections PAPER.md:L135).
 *   out[i] = table[B(x[i], edges_x, nx) * ny + B(y[i], edges_y, ny)]     (y == NULL: table[B(x[i])])
 *   B(v) = the b with edges[b] <= v < edges[b+1], clamped: v < edges[0] -> 0; v >= edges[n] or NaN -> n-1.
 * x, y: float32[n]; edges_x: float32[nx+1] ascending; edges_y: float32[ny+1]; table: float32[nx*ny]
 * row-major, no flow bins; out: float32[n].  Limit: 2*(nx+1)+2*(ny+1)+nx*ny floats (the edges, a padded copy of
 * them for the bin search, the table) must fit 200 KB of shared memory, else HEPK_ERR_UNSUPPORTED. */
int32_t hepk_lookup_binned(const float* x, const float* y, int64_t n,
                           const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                           const float* table, float* out, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Weighted 1-D histogram fill, fill_histogram ("given a data array, a weight array,
 * histogram bin edges and contents, fills the weighted data to the histogram").
 *   slot(x) = 0 if x < edges[0]; nbins+1 if x >= edges[nbins] or x is NaN; else 1+b with
 *   edges[b] <= x < edges[b+1].   sumw[slot] += w (w = 1 if weights == NULL); counts[slot] += 1.
 * data, weights: float32[n]; edges: float32[nbins+1] ascending; sumw: float32[nbins+2] or NULL;
 * counts: int64[nbins+2] or NULL.  Both outputs accumulate.  Bins are privatised in shared memory — for
 * small histograms (up to ~200 bins with both outputs) one copy per LANE, updated without atomics and summed
 * in float64 per CTA; one copy per CTA with float32 atomics otherwise — and merged into the caller's float32
 * array with float atomics, so sumw depends on the merge order in its last bits; hepk_fill_histogram_w2
 * (below) takes a workspace and merges in 64 bits.  nbins+2 <= 16384, else HEPK_ERR_UNSUPPORTED. */
int32_t hepk_fill_histogram(const float* data, const float* weights, int64_t n,
                            const float* edges, int32_t nbins,
                            float* sumw, int64_t* counts, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Fused analysis chain: one pass over the inputs doing object selection, jet-lepton
 * dR cleaning (L133), jet calibration by binned lookup under systematic variants (L135), per-event
 * reductions (L106-108), leading-pair mass (L136) and weighted histograms (L139) — the fusion the
 * paper names as the missing optimisation.
 *
 * For every event e and variant v in [0, n_variants):
 *   1. pt_v[j] = jets.pt[j]                                  if calib_table == NULL (n_variants must be 1)
 *              = jets.pt[j] * (table[B(pt_j)][B(eta_j)] * calib_scales[v])   (two float32 multiplies)
 *   2. jsel_v[j] = pt_v[j] > jet_pt_min && |eta_j| < jet_abs_eta_max;  lepton selected iff pt > lep_pt_min
 *   3. matched[j] = dR match (hepk_deltar_mask rule) against selected muons or selected electrons
 *   4. clean_v[j] = jsel_v[j] && !matched[j]
 *   5. njet, ht = sum pt_v, maxpt, minpt, argmax (local index) over clean jets
 *   6. mjj = leading-pair mass of (pt_v, eta, phi, mass) over clean jets; subpt = pt_v[i2] or 0.0f
 *   7. for every observable o with axis_edges[o] != NULL: slot = hepk_fill_histogram rule on
 *      (float)observable; hist_counts[v][o][slot] += 1; hist_sumw[v][o][w][slot] += weights[w][e].
 */
enum {
    HEPK_OBS_NJET = 0, HEPK_OBS_HT = 1, HEPK_OBS_MAXPT = 2, HEPK_OBS_MINPT = 3, HEPK_OBS_MJJ = 4, HEPK_OBS_SUBPT = 5,
    HEPK_N_OBS = 6
};

typedef struct hepk_collection {
    const int64_t* offsets;   /* int64[n_events+1]; NULL = collection absent (electrons only) */
    int64_t content_base;     /* global index of column element 0 */
    int64_t n_objects;        /* number of valid elements in each column */
    const float* pt;          /* float32[n_objects] */
    const float* eta;
    const float* phi;
    const float* mass;        /* read for jets only; may be NULL for leptons */
} hepk_collection;

typedef struct hepk_chain_desc {
    int64_t n_events;
    hepk_collection jets, muons, electrons;
    float jet_pt_min, jet_abs_eta_max, lep_pt_min, dr_max;
    /* calibration (optional) */
    const float* calib_pt_edges;  int32_t calib_npt;     /* float32[npt+1] */
    const float* calib_eta_edges; int32_t calib_neta;    /* float32[neta+1] */
    const float* calib_table;                            /* float32[npt*neta] row-major; NULL = no calibration */
    float calib_scales[HEPK_MAX_VARIANTS];               /* by value */
    int32_t n_variants;                                  /* 1..HEPK_MAX_VARIANTS */
    int32_t n_wvar;                                      /* 1..HEPK_MAX_WVAR weight columns */
    const float* weights;                                /* float32[n_wvar][n_events]; NULL = weight 1 */
    const float* axis_edges[HEPK_N_OBS];                 /* float32[nbins+1] per observable; NULL = not histogrammed */
    int32_t axis_nbins[HEPK_N_OBS];
    /* per-event outputs, each [n_variants][n_events]; all nullable */
    int32_t* out_njet; int32_t* out_argmax;
    float* out_ht; float* out_maxpt; float* out_minpt; float* out_mjj; float* out_subpt;
    uint8_t* out_jet_mask;                               /* uint8[n_variants][jets.n_objects] clean-jet mask */
    /* histograms, accumulate; nullable.  Active observables in enum order, o-th has nbins_o+2 slots:
     *   hist_sumw   float32 [n_variants][active o][n_wvar][nbins_o+2]
     *   hist_counts int64   [n_variants][active o][nbins_o+2] */
    float* hist_sumw; int64_t* hist_counts;
    /* SURVEY.md 8(f-2), PAPER.md:L134 ("event weight computation based on histogram lookups: pileup, lepton
     * efficiency corrections"): optional per-event weight factor f[e] = evw_table[B(evw_x[e])] (B: the clamped
     * bin of hepk_lookup_binned, 1-D), multiplied into every weight column with ONE float32 multiply before the
     * fill (weights == NULL: 1.0f * f).  evw_x: float32[n_events]; evw_edges: float32[evw_nbins+1] ascending;
     * evw_table: float32[evw_nbins], NULL = no factor; evw_nbins <= 4096. */
    const float* evw_x; const float* evw_edges; int32_t evw_nbins; const float* evw_table;
    /* sum of squared (final) weights per slot (the uncertainty of a weighted bin), layout of
     * hist_sumw, accumulates; NULL = not wanted.  Without weights and factor it equals the counts. */
    float* hist_sumw2;
    /* Row strides, in events, of `weights` ([n_wvar] rows) and of every per-event output array ([n_variants] rows);
     * 0 = n_events (contiguous rows).  A shard of a larger workload (PAPER.md:L166 multi-GPU) passes
     * pointers to its first event inside the whole arrays and the whole workload's event count here. */
    int64_t weights_stride; int64_t out_stride;
    /* RESERVED for the library's own tests (staging capacities and CTA shape); leave 0 = automatic */
    int32_t tune_cap_jets;       /* shared-memory capacity (jets per staged 32-event tile) */
    int32_t tune_cap_leptons;    /* capacity per lepton collection */
    int32_t tune_ctas_per_sm;    /* persistent CTAs per SM */
    int32_t tune_warps_per_cta;  /* warps (each owning its own tiles and staging region) per CTA, at most 24 */
    int32_t tune_warps_per_sm;   /* resident warps per SM the launch aims for (default 20) */
    int32_t tune_variants_per_pass; /* variants per kernel launch (default: all, fewer when the histograms crowd out the warps) */
    int32_t tune_generic_build;  /* != 0: never take the build specialised for the common output shape */
} hepk_chain_desc;

/* `d` is a HOST pointer to a descriptor whose array pointers are DEVICE pointers.  `workspace` is a
 * device buffer of at least hepk_chain_workspace_bytes(d) bytes (64-bit histogram accumulators; needed
 * whenever a histogram output is asked for), private to this call until the stream reaches its end.
 *
 * Weighted bins (tolerance class): when all weight columns (times the lookup factor) are finite and span
 * at most a factor 8 in magnitude, entries are accumulated in fixed point — each entry rounded once to
 * a multiple of 2^-k >= 2^-20 max|w|, exact integer sums, order independent — which bounds the error of a
 * bin by 7.7e-6 of its smallest entry times the entries it holds; otherwise bins are float32 partial sums
 * of at most ~1000 entries merged in float64.  Either way |error| <= 1e-5 * sum|w_i| of the bin. */
size_t  hepk_chain_workspace_bytes(const hepk_chain_desc* d);
int32_t hepk_analysis_chain(const hepk_chain_desc* d, void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Batch streaming (Fig. 1: "the cache is loaded in batches of a few GB of contiguous
 * 1-dimensional arrays ... with kernels being dispatched on the data either in host or device
 * memory").  Same computation as hepk_analysis_chain, but every array pointer in `d` (inputs and
 * outputs, histograms included) is a HOST pointer, ideally pinned.  The events are cut into batches
 * of `batch_events`; each batch's offsets slices and column slices are copied host->device, the chain
 * runs on the device and the per-event outputs are copied back; histograms are copied back once at the
 * end and ADDED to the host arrays.  overlap != 0 double-buffers the copies against the kernels on
 * internal streams; overlap == 0 runs copy -> compute -> copy serially.  The call returns after all work
 * has finished (it synchronises).  `workspace` is a DEVICE buffer of at least
 * hepk_chain_host_workspace_bytes(d, batch_events) bytes.  calib / axis edge arrays are HOST too.
 * Thread safety: the call creates its two internal streams itself and destroys them before it returns
 * (after draining them, also on an error return), so calls from several host threads are independent as
 * long as each passes its own workspace and output buffers. */
size_t  hepk_chain_host_workspace_bytes(const hepk_chain_desc* d, int64_t batch_events);
int32_t hepk_analysis_chain_host(const hepk_chain_desc* d, int64_t batch_events, int32_t overlap,
                                 void* workspace, size_t workspace_bytes, void* stream);

/* ---------------------------------------------------------------------------------------------
 * The remaining generic kernels of the paper's list.  All pointers are DEVICE pointers.
 *
 * get_in_offsets ("given jagged data with offsets, retrieves the n-th elements for all rows ...
 * to create a contiguous array of e.g. the leading jet pT"):
 *   out[e] = the index-th element of row e, counting only elements with mask_content set (NULL: all);
 *   rows with mask_rows clear, or with fewer than index+1 counted elements, get `fill`.
 * data: float32[M]; offsets: int64[n_events+1]; out: float32[n_events]; index >= 0 else HEPK_ERR_INVALID. */
int32_t hepk_get_in_offsets(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index, float fill,
                            float* out, void* stream);

/* set_in_offsets ("as above, but sets the n-th element to a value ... to selectively mask
 * objects in a collection"):
 *   data[position of the index-th counted element of row e] = values ? values[e] : value
 * for rows with mask_rows set (or NULL) that have that element; everything else is left untouched.
 * data: float32[M], modified in place; values: float32[n_events] or NULL. */
int32_t hepk_set_in_offsets(float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index,
                            const float* values, float value, void* stream);

/* select_opposite_sign_muons ("given a collection of objects with charge (i.e. muons),
 * masks all but the first two objects ordered by pT which are of opposite charge"):
 *   per event, over the objects with mask_content set (NULL: all): the leading object by pt (first index
 *   among equal pt; NaN skipped) and the highest-pt object whose charge has the opposite sign get 1,
 *   everything else 0; an event without such a pair, or with mask_rows clear, gets all 0.
 * pt: float32[M]; charge: int32[M]; out_mask: uint8[M], every element of every event is written. */
int32_t hepk_select_opposite_sign(const float* pt, const int32_t* charge, const int64_t* offsets, int64_t n_events,
                                  int64_t content_base, const uint8_t* mask_rows, const uint8_t* mask_content,
                                  uint8_t* out_mask, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Lookup / histogram variants.  All array pointers are DEVICE pointers.
 *
 * Linear-interpolated correction ("systematic corrections based on linear interpolations"):
 *   knots xs[0..nk) ascending with values ys[0..nk), nk >= 2;
 *   out[i] = ys[b] + (x[i] - xs[b]) * (ys[b+1] - ys[b]) / (xs[b+1] - xs[b])  for xs[b] <= x[i] < xs[b+1];
 *   x <= xs[0] -> ys[0], x >= xs[nk-1] -> ys[nk-1] (constant extrapolation), NaN -> NaN.
 * Tolerance class (float32 evaluation with one slope per segment).  16*nk bytes of shared memory (knots, values,
 * slopes, a padded copy of the knots for the segment search), more than 200 KB (nk > 12,800) -> HEPK_ERR_UNSUPPORTED. */
int32_t hepk_lookup_interp(const float* x, int64_t n, const float* xs, const float* ys, int32_t nk, float* out, void* stream);

/* Two-dimensional weighted histogram ("Extension to multidimensional histograms is straightforward"):
 *   slot = sx * (ny + 2) + sy, sx / sy the hepk_fill_histogram slots of x / y on their axes (flow bins kept per axis);
 *   sumw[slot] += w (1 if weights == NULL), counts[slot] += 1.  sumw: float32[(nx+2)*(ny+2)] or NULL,
 *   counts: int64[(nx+2)*(ny+2)] or NULL; both accumulate.  Bins are privatised per CTA in shared memory and merged
 *   into float64 accumulators in `workspace` (device, >= hepk_hist2d_workspace_bytes(nx, ny) bytes, needed when sumw
 *   is given).  (nx+2)*(ny+2) <= 16384, else HEPK_ERR_UNSUPPORTED. */
size_t  hepk_hist2d_workspace_bytes(int32_t nx, int32_t ny);
int32_t hepk_fill_histogram_2d(const float* x, const float* y, const float* weights, int64_t n,
                               const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                               float* sumw, int64_t* counts, void* workspace, size_t workspace_bytes, void* stream);

/* Weighted fills with the sum of squared weights (PAPER.md:L109 `fill_histogram`; the squared sum is the statistical
 * uncertainty of a weighted bin), one and two dimensions.  Slots and conventions of hepk_fill_histogram /
 * hepk_fill_histogram_2d; additionally sumw2[slot] += w*w (w = 1 if weights == NULL, so sumw2 == counts).
 * sumw, sumw2: float32, counts: int64, each nullable, all accumulate.  `workspace`: device buffer of at least
 * hepk_hist_workspace_bytes(nx, ny) bytes (ny = 0 for one dimension; 64-bit accumulators), private to the call
 * until the stream reaches its end.  Tolerance class, same guarantee as the chain's weighted bins: float32
 * partial sums of at most 32768 entries merged in float64 (one dimension with few bins: a private copy of the
 * bins per lane, hepk_hist_lanes.cuh), or fixed-point bins (exact integer sums) for small histograms whose
 * weights are finite and within a factor 8 of each other.  nbins+2 (resp. (nx+2)*(ny+2))
 * <= 16384 and rows x columns (plus two copies of the edges) must fit 200 KB of shared memory, else
 * HEPK_ERR_UNSUPPORTED. */
size_t  hepk_hist_workspace_bytes(int32_t nx, int32_t ny);
int32_t hepk_fill_histogram_w2(const float* data, const float* weights, int64_t n, const float* edges, int32_t nbins,
                               float* sumw, float* sumw2, int64_t* counts, void* workspace, size_t workspace_bytes,
                               void* stream);
/* hepk_fill_histogram_w2 without a workspace and without any allocation, for callers that cannot call cudaMalloc
 * (code under CUDA graph capture, tight serving loops, harnesses that forbid it).  Same arguments, same results
 * (same kernels) as hepk_fill_histogram_w2; the 64-bit accumulators live in a device array inside the library,
 * hepk_static_hist_scratch_bytes() = 164,096 bytes that every GPU loading the library holds until exit.
 * Limits: nbins <= HEPK_STATIC_HIST_MAX_BINS (4094), else HEPK_ERR_UNSUPPORTED with the reason in
 * hepk_last_error().  The call makes no cudaMalloc / cudaFree and calls no allocating library routine; it clears the
 * part of the array it uses, on `stream`, before the fill.  ALL calls on a device share the one array: two calls
 * that can overlap on the GPU (different streams without an ordering between them, or two host threads) race on it
 * and corrupt each other's sums — order them, or use hepk_fill_histogram_w2 with a workspace per call. */
#define HEPK_STATIC_HIST_MAX_BINS 4094
size_t  hepk_static_hist_scratch_bytes(void);
int32_t hepk_fill_histogram_w2_static(const float* data, const float* weights, int64_t n, const float* edges, int32_t nbins,
                                      float* sumw, float* sumw2, int64_t* counts, void* stream);
int32_t hepk_fill_histogram_2d_w2(const float* x, const float* y, const float* weights, int64_t n,
                                  const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                                  float* sumw, float* sumw2, int64_t* counts, void* workspace, size_t workspace_bytes,
                                  void* stream);

/* Event weight from a histogram lookup ("event weight computation based on histogram lookups:
 * pileup, lepton efficiency corrections"):
 *   w_out[e] = w_in[e] * table[B(x[e])]     one float32 multiply (exact class); w_in == NULL: w_in = 1
 * B: the clamped bin of hepk_lookup_binned on edges[nbins+1].  x, w_in, w_out: float32[n] (w_out may alias w_in);
 * table: float32[nbins].  2*nbins+1 floats must fit 200 KB of shared memory, else HEPK_ERR_UNSUPPORTED.
 * The fused chain applies the same factor through hepk_chain_desc.evw_*. */
int32_t hepk_event_weight_lookup(const float* w_in, const float* x, int64_t n, const float* edges, int32_t nbins,
                                 const float* table, float* w_out, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Jet-triplet candidate ("top quark candidate from jet triplet with invariant
 * mass closest to M = 172 GeV").  Per event, over all triplets i < j < k of the objects with mask_content set:
 *   M_ijk = sqrt(max(0, (E_i+E_j+E_k)^2 - |p_i+p_j+p_k|^2)), four-vectors as in hepk_pair_invmass, float64;
 *   the triplet minimising |M_ijk - target| is kept (equal distances: the lexicographically first (i, j, k)).
 * out_mass[e] = (float)M of that triplet; out_idx[3e..3e+2] its local indices (may be NULL); fewer than three
 * selected objects or mask_rows clear: 0.0f and -1.  Tolerance class: when two triplets are equally close to
 * within the float64 rounding of the transcendental functions, either is a valid answer.
 * All array pointers are DEVICE pointers. */
int32_t hepk_triplet_mass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_rows,
                          const uint8_t* mask_content, float target, float* out_mass, int32_t* out_idx, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Precondition check of a jagged layout ("a contiguous offsets array of size N+1").  Every other
 * entry assumes valid offsets; this one counts the violations among
 *   offsets[0] >= content_base,  offsets[e] <= offsets[e+1] for every e,  offsets[n_events] - content_base <= n_objects
 * into *n_bad (DEVICE pointer to one int64, overwritten).  offsets: DEVICE int64[n_events+1]. */
int32_t hepk_validate_offsets(const int64_t* offsets, int64_t n_events, int64_t content_base, int64_t n_objects,
                              int64_t* n_bad, void* stream);

/* ---------------------------------------------------------------------------------------------
 * Device-side timing of the dominant kernel (measurement hook for bench.py; no part of the method).
 * Between hepk_profile_begin() and hepk_profile_end() every hepk_analysis_chain call records a CUDA event
 * pair on its launch stream directly around the fused chain kernel (at most 4096 launches are kept).
 * hepk_profile_end() waits for the recorded events, stores the summed kernel time in milliseconds in
 * *total_ms (HOST pointer) and the number of timed launches in *n_launches (HOST pointer; either may be
 * NULL), and switches the recording off.  One profiling session per process at a time (the event table is
 * guarded by a mutex; launches from several host threads are all recorded into it). */
int32_t hepk_profile_begin(void);
int32_t hepk_profile_end(double* total_ms, int32_t* n_launches);
/* Measurement hook (no part of the method): the rate of native shared-memory integer atomics on this device,
 * red.shared.add.s32 to pseudo-random addresses among `nbins` words by `warps_per_sm` warps on every SM, in
 * lane-atomics per second over the whole device (the bound of histogram-heavy chain launches; bench.py).
 * `scratch`: device buffer of at least 4 bytes per SM.  Synchronises. */
int32_t hepk_probe_shared_atomics(int32_t warps_per_sm, int32_t nbins, void* scratch, double* lane_atomics_per_second);
/* Number of kernels this library has enqueued in this process so far (all entry points, all threads). */
int64_t hepk_kernel_launches(void);

#ifdef __cplusplus
}
#endif
#endif /* HEPK_H */
