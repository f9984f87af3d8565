/*
 * hepo.c — CPU ORACLE (see hepo.h).  TEST INFRASTRUCTURE ONLY; never on the product path.
 *
 * Plain C, one loop over events, one inner loop over particles, exactly the shape of the
 * paper's Listing 1.  No blocking, no fusion, no reordering.
 * Build: gcc -O2 -ffp-contract=off -fno-fast-math -shared -fPIC (oracle/build.py).
 *
 * "parity unpinned" items (Readings R3/R5/R9/R12/R14): the empty-event values
 * (0, -inf, +inf, -1), the clamp policy of hepo_lookup_binned, NaN routing, the electron cut
 * of the chain and the choice of config 4's 30 variables are conventions of this build; the
 * paper states none of them, so no test can pin them to the paper.
 */
#include "hepo.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* float32 constants of the dphi wrap (R6): PI_F = 0x40490FDB, TWO_PI_F = 0x40C90FDB. */
static const float PI_F = 3.14159274101257324f;
static const float TWO_PI_F = 6.28318548202514648f;

/* ------------------------------------------------------------------ c1: object selection */
int32_t hepo_select_mask(const float* pt, const float* eta, int64_t n, float pt_min, float abs_eta_max,
                         uint8_t* out_mask)
{
    if (n < 0 || (n > 0 && (!pt || !out_mask))) return -1;
    for (int64_t i = 0; i < n; ++i) {
        int pass = pt[i] > pt_min;                       /* strict: BASELINE.json "pt>30" */
        if (eta) pass = pass && (fabsf(eta[i]) < abs_eta_max);   /* strict: "|eta|<2.4" */
        out_mask[i] = (uint8_t)(pass ? 1 : 0);
    }
    return 0;
}

/* ------------------------------------------------------------------ c2: segmented reductions
 * Listing 1, PAPER.md:L66-87:
 *     for iev in prange(N):
 *         if not mask_rows[iev]: continue
 *         i0 = offsets[iev]; i1 = offsets[iev + 1]
 *         for ielem in range(i0, i1):
 *             if mask_content[ielem]: out[iev] += pt_data[ielem]
 */
static int seg_args_ok(const int64_t* offsets, int64_t n_events, const void* out)
{
    return n_events >= 0 && (n_events == 0 || (offsets && out));
}

int32_t hepo_segmented_reduce_sum(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out)
{
    if (!seg_args_ok(offsets, n_events, out)) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        double acc = 0.0;                                 /* tolerance class: float64 accumulator */
        if (!mask_rows || mask_rows[iev]) {
            for (int64_t g = offsets[iev]; g < offsets[iev + 1]; ++g) {
                int64_t i = g - content_base;
                if (!mask_content || mask_content[i]) acc += (double)data[i];
            }
        }
        out[iev] = (float)acc;
    }
    return 0;
}

int32_t hepo_segmented_reduce_count(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                    const uint8_t* mask_rows, const uint8_t* mask_content, int32_t* out)
{
    (void)data;                                           /* "count objects ... by summing masks" */
    if (!seg_args_ok(offsets, n_events, out)) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        int32_t c = 0;
        if (!mask_rows || mask_rows[iev]) {
            for (int64_t g = offsets[iev]; g < offsets[iev + 1]; ++g) {
                int64_t i = g - content_base;
                if (!mask_content || mask_content[i]) c += 1;
            }
        }
        out[iev] = c;
    }
    return 0;
}

int32_t hepo_segmented_reduce_max(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out)
{
    if (!seg_args_ok(offsets, n_events, out)) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        float best = -INFINITY;
        if (!mask_rows || mask_rows[iev]) {
            for (int64_t g = offsets[iev]; g < offsets[iev + 1]; ++g) {
                int64_t i = g - content_base;
                if (mask_content && !mask_content[i]) continue;
                if (data[i] > best) best = data[i];      /* NaN compares false: skipped */
            }
        }
        out[iev] = best;
    }
    return 0;
}

int32_t hepo_segmented_reduce_min(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, float* out)
{
    if (!seg_args_ok(offsets, n_events, out)) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        float best = INFINITY;
        if (!mask_rows || mask_rows[iev]) {
            for (int64_t g = offsets[iev]; g < offsets[iev + 1]; ++g) {
                int64_t i = g - content_base;
                if (mask_content && !mask_content[i]) continue;
                if (data[i] < best) best = data[i];
            }
        }
        out[iev] = best;
    }
    return 0;
}

int32_t hepo_segmented_reduce_argmax(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                     const uint8_t* mask_rows, const uint8_t* mask_content, int32_t* out)
{
    if (!seg_args_ok(offsets, n_events, out)) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        int32_t arg = -1;
        float best = 0.0f;
        if (!mask_rows || mask_rows[iev]) {
            for (int64_t g = offsets[iev]; g < offsets[iev + 1]; ++g) {
                int64_t i = g - content_base;
                if (mask_content && !mask_content[i]) continue;
                float v = data[i];
                if (v != v) continue;                    /* NaN skipped */
                if (arg < 0 || v > best) {               /* strict >: first index wins ties */
                    best = v;
                    arg = (int32_t)(g - offsets[iev]);   /* index local to the event */
                }
            }
        }
        out[iev] = arg;
    }
    return 0;
}

/* ------------------------------------------------------------------ c3: dR matching
 * "masks all objects in the first collection that are closer than a predefined value
 * in dR^2 = deta^2 + dphi^2 to an object in the second collection".  float32, one rounding per op. */
static float dr2_f32(float eta_a, float phi_a, float eta_b, float phi_b)
{
    float deta = eta_a - eta_b;
    float dphi = phi_a - phi_b;
    if (dphi > PI_F) dphi = dphi - TWO_PI_F;             /* single-step wrap, R6 */
    else if (dphi <= -PI_F) dphi = dphi + TWO_PI_F;
    float a = deta * deta;
    float b = dphi * dphi;
    return a + b;
}

int32_t hepo_deltar_mask(const float* eta1, const float* phi1, const int64_t* offsets1, int64_t base1, const uint8_t* sel1,
                         const float* eta2, const float* phi2, const int64_t* offsets2, int64_t base2, const uint8_t* sel2,
                         int64_t n_events, float dr_max, uint8_t* out_matched)
{
    if (n_events < 0) return -1;
    if (n_events > 0 && (!offsets1 || !offsets2)) return -1;
    const float thr = dr_max * dr_max;                    /* float32 product */
    for (int64_t iev = 0; iev < n_events; ++iev) {
        for (int64_t g1 = offsets1[iev]; g1 < offsets1[iev + 1]; ++g1) {
            int64_t j = g1 - base1;
            uint8_t matched = 0;
            if (!sel1 || sel1[j]) {
                for (int64_t g2 = offsets2[iev]; g2 < offsets2[iev + 1]; ++g2) {
                    int64_t m = g2 - base2;
                    if (sel2 && !sel2[m]) continue;
                    if (dr2_f32(eta1[j], phi1[j], eta2[m], phi2[m]) < thr) {   /* "closer than": strict */
                        matched = 1;
                        break;   /* "terminated when the matching criterion is satisfied" */
                    }
                }
            }
            out_matched[j] = matched;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ c4: leading-pair invariant mass
 * Massive four-vector from (pT, eta, phi, M), naive form in float64:
 *   px = pt cos(phi), py = pt sin(phi), pz = pt sinh(eta), E = sqrt(pt^2 cosh^2(eta) + m^2)
 *   M^2 = (E1+E2)^2 - (px1+px2)^2 - (py1+py2)^2 - (pz1+pz2)^2,  mass = sqrt(max(M^2, 0)). */
static float pair_mass_f64(float pt1, float eta1, float phi1, float m1,
                           float pt2, float eta2, float phi2, float m2)
{
    double px1 = (double)pt1 * cos((double)phi1), py1 = (double)pt1 * sin((double)phi1);
    double pz1 = (double)pt1 * sinh((double)eta1);
    double ch1 = cosh((double)eta1);
    double e1 = sqrt((double)pt1 * (double)pt1 * ch1 * ch1 + (double)m1 * (double)m1);
    double px2 = (double)pt2 * cos((double)phi2), py2 = (double)pt2 * sin((double)phi2);
    double pz2 = (double)pt2 * sinh((double)eta2);
    double ch2 = cosh((double)eta2);
    double e2 = sqrt((double)pt2 * (double)pt2 * ch2 * ch2 + (double)m2 * (double)m2);
    double e = e1 + e2, px = px1 + px2, py = py1 + py2, pz = pz1 + pz2;
    double m2sq = e * e - px * px - py * py - pz * pz;
    if (!(m2sq > 0.0)) m2sq = 0.0;                        /* clamp rounding negatives to 0 */
    return (float)sqrt(m2sq);
}

/* top-2 by value among selected entries of v[0..n), first-index tie rule (same rule as argmax, applied twice). */
static void top2(const float* v, const uint8_t* sel, int64_t n, int32_t* i1, int32_t* i2)
{
    int32_t a = -1, b = -1;
    for (int64_t k = 0; k < n; ++k) {
        if (sel && !sel[k]) continue;
        if (v[k] != v[k]) continue;
        if (a < 0 || v[k] > v[a]) a = (int32_t)k;
    }
    for (int64_t k = 0; k < n; ++k) {
        if (sel && !sel[k]) continue;
        if (v[k] != v[k]) continue;
        if ((int32_t)k == a) continue;
        if (b < 0 || v[k] > v[b]) b = (int32_t)k;
    }
    *i1 = a;
    *i2 = b;
}

int32_t hepo_pair_invmass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_content,
                          float* out_mass, int32_t* out_i1, int32_t* out_i2)
{
    if (n_events < 0 || (n_events > 0 && (!offsets || !out_mass))) return -1;
    for (int64_t iev = 0; iev < n_events; ++iev) {
        int64_t i0 = offsets[iev] - content_base, n = offsets[iev + 1] - offsets[iev];
        int32_t a, b;
        top2(pt + i0, mask_content ? mask_content + i0 : NULL, n, &a, &b);
        float m = 0.0f;                                   /* fewer than two selected: 0.0f (unpinned) */
        if (a >= 0 && b >= 0)
            m = pair_mass_f64(pt[i0 + a], eta[i0 + a], phi[i0 + a], mass[i0 + a],
                              pt[i0 + b], eta[i0 + b], phi[i0 + b], mass[i0 + b]);
        out_mass[iev] = m;
        if (out_i1) out_i1[iev] = a;
        if (out_i2) out_i2[iev] = b;
    }
    return 0;
}

/* ------------------------------------------------------------------ c5: binned lookup
 * B(v): the b with edges[b] <= v < edges[b+1] (right-open), clamped: v < edges[0] -> 0;
 * v >= edges[n] or NaN -> n-1 (clamp policy: parity unpinned). */
static int32_t find_bin_clamped(float v, const float* edges, int32_t n)
{
    if (v < edges[0]) return 0;
    if (!(v < edges[n])) return n - 1;
    int32_t lo = 0, hi = n;                               /* invariant: edges[lo] <= v < edges[hi] */
    while (hi - lo > 1) {
        int32_t mid = lo + (hi - lo) / 2;
        if (v >= edges[mid]) lo = mid; else hi = mid;
    }
    return lo;
}

int32_t hepo_lookup_binned(const float* x, const float* y, int64_t n,
                           const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                           const float* table, float* out)
{
    if (n < 0 || nx < 1 || !edges_x || !table || (n > 0 && (!x || !out))) return -1;
    if (y && (ny < 1 || !edges_y)) return -1;
    for (int64_t i = 0; i < n; ++i) {
        int32_t bx = find_bin_clamped(x[i], edges_x, nx);
        if (y) {
            int32_t by = find_bin_clamped(y[i], edges_y, ny);
            out[i] = table[(int64_t)bx * ny + by];
        } else {
            out[i] = table[bx];
        }
    }
    return 0;
}

/* ------------------------------------------------------------------ c6: histogram fill
 * Slot layout [underflow, bin 0 .. bin nbins-1, overflow]; NaN -> overflow. */
static int32_t hist_slot(float x, const float* edges, int32_t nbins)
{
    if (x < edges[0]) return 0;
    if (!(x < edges[nbins])) return nbins + 1;
    int32_t lo = 0, hi = nbins;
    while (hi - lo > 1) {
        int32_t mid = lo + (hi - lo) / 2;
        if (x >= edges[mid]) lo = mid; else hi = mid;
    }
    return 1 + lo;
}

int32_t hepo_fill_histogram(const float* data, const float* weights, int64_t n,
                            const float* edges, int32_t nbins, float* sumw, int64_t* counts)
{
    if (n < 0 || nbins < 1 || !edges || (n > 0 && !data)) return -1;
    double* acc = (double*)calloc((size_t)nbins + 2, sizeof(double));
    if (!acc) return -1;
    for (int64_t i = 0; i < n; ++i) {
        int32_t s = hist_slot(data[i], edges, nbins);
        acc[s] += weights ? (double)weights[i] : 1.0;
        if (counts) counts[s] += 1;
    }
    if (sumw)
        for (int32_t s = 0; s < nbins + 2; ++s) sumw[s] = (float)((double)sumw[s] + acc[s]);
    free(acc);
    return 0;
}

/* the same fill with the sum of squared weights per slot (the statistical
 * uncertainty of a weighted bin); w*w in float64 from the float32 weight, one rounding at the end.
 * weights == NULL: every weight is 1, so sumw2 == sumw == counts. */
int32_t hepo_fill_histogram_w2(const float* data, const float* weights, int64_t n,
                               const float* edges, int32_t nbins, float* sumw, float* sumw2, int64_t* counts)
{
    if (n < 0 || nbins < 1 || !edges || (n > 0 && !data)) return -1;
    double* acc = (double*)calloc(2 * ((size_t)nbins + 2), sizeof(double));
    if (!acc) return -1;
    double* acc2 = acc + nbins + 2;
    for (int64_t i = 0; i < n; ++i) {
        int32_t s = hist_slot(data[i], edges, nbins);
        double w = weights ? (double)weights[i] : 1.0;
        acc[s] += w;
        acc2[s] += w * w;
        if (counts) counts[s] += 1;
    }
    for (int32_t s = 0; s < nbins + 2; ++s) {
        if (sumw) sumw[s] = (float)((double)sumw[s] + acc[s]);
        if (sumw2) sumw2[s] = (float)((double)sumw2[s] + acc2[s]);
    }
    free(acc);
    return 0;
}

/* SURVEY.md 8(f-2), "event weight computation based on histogram lookups: pileup, lepton
 * efficiency corrections": w_out[e] = w_in[e] * table[B(x[e])], B the clamped bin of hepo_lookup_binned (1-D),
 * ONE float32 multiply (exact class).  w_in == NULL: w_in = 1. */
int32_t hepo_event_weight_lookup(const float* w_in, const float* x, int64_t n,
                                 const float* edges, int32_t nbins, const float* table, float* w_out)
{
    if (n < 0 || nbins < 1 || !edges || !table || (n > 0 && (!x || !w_out))) return -1;
    for (int64_t e = 0; e < n; ++e) {
        float f = table[find_bin_clamped(x[e], edges, nbins)];
        float w = w_in ? w_in[e] : 1.0f;
        w_out[e] = w * f;
    }
    return 0;
}

/* ------------------------------------------------------------------ c7: the fused chain, event by event
 * Steps follow the benchmark analysis list PAPER.md:L131-139 restricted to the hot path:
 * object selection (L132), jet-lepton dR matching (L133), jet corrections by histogram lookup
 * with systematic variants (L135), per-event reductions (L106-108), leading-pair mass (L136),
 * weighted histograms (L139). */
size_t hepo_chain_desc_size(void) { return sizeof(hepo_chain_desc); }

/* slot prefix of the active observables; returns the slots per variant */
static int64_t chain_hist_layout(const hepo_chain_desc* d, int64_t* obs_prefix)
{
    obs_prefix[0] = 0;
    for (int o = 0; o < HEPO_N_OBS; ++o)
        obs_prefix[o + 1] = obs_prefix[o] + (d->axis_edges[o] ? d->axis_nbins[o] + 2 : 0);
    return obs_prefix[HEPO_N_OBS];
}

/* Events [e_begin, e_end) of the chain.  acc / acc2: float64 accumulators of sumw / sumw2 (NULL: not wanted),
 * counts: int64 accumulators (NULL: not wanted), all in the layout of the descriptor's histogram arrays. */
static int32_t chain_event_range(const hepo_chain_desc* d, int64_t e_begin, int64_t e_end,
                                 double* acc, double* acc2, int64_t* counts)
{
    const int64_t N = d->n_events;
    const int32_t V = d->n_variants, W = d->n_wvar;
    const int has_el = d->electrons.offsets != NULL;
    const float thr = d->dr_max * d->dr_max;
    int64_t obs_prefix[HEPO_N_OBS + 1];
    const int64_t slots_per_variant = chain_hist_layout(d, obs_prefix);

    int64_t cap = 64;
    float* ptv = (float*)malloc((size_t)cap * sizeof(float));
    uint8_t* matched = (uint8_t*)malloc((size_t)cap);
    uint8_t* clean = (uint8_t*)malloc((size_t)cap);
    float* corr = (float*)malloc((size_t)cap * sizeof(float));
    if (!ptv || !matched || !clean || !corr) { free(ptv); free(matched); free(clean); free(corr); return -1; }

    for (int64_t iev = e_begin; iev < e_end; ++iev) {
        const int64_t j0 = d->jets.offsets[iev] - d->jets.content_base;
        const int64_t nj = d->jets.offsets[iev + 1] - d->jets.offsets[iev];
        if (nj > cap) {
            cap = nj * 2;
            ptv = (float*)realloc(ptv, (size_t)cap * sizeof(float));
            matched = (uint8_t*)realloc(matched, (size_t)cap);
            clean = (uint8_t*)realloc(clean, (size_t)cap);
            corr = (float*)realloc(corr, (size_t)cap * sizeof(float));
        }
        /* step 3: matched[j] vs selected muons OR selected electrons (variant independent) */
        for (int64_t k = 0; k < nj; ++k) {
            uint8_t mt = 0;
            for (int c = 0; c < 2 && !mt; ++c) {
                const hepo_collection* L = c == 0 ? &d->muons : &d->electrons;
                if (c == 1 && !has_el) break;
                for (int64_t g = L->offsets[iev]; g < L->offsets[iev + 1]; ++g) {
                    int64_t m = g - L->content_base;
                    if (!(L->pt[m] > d->lep_pt_min)) continue;   /* step 2: lepton selection, same cut for e and mu */
                    if (dr2_f32(d->jets.eta[j0 + k], d->jets.phi[j0 + k], L->eta[m], L->phi[m]) < thr) { mt = 1; break; }
                }
            }
            matched[k] = mt;
            /* calibration factor from the RAW pt and eta (step 1) */
            corr[k] = 1.0f;
            if (d->calib_table) {
                int32_t bx = find_bin_clamped(d->jets.pt[j0 + k], d->calib_pt_edges, d->calib_npt);
                int32_t by = find_bin_clamped(d->jets.eta[j0 + k], d->calib_eta_edges, d->calib_neta);
                corr[k] = d->calib_table[(int64_t)bx * d->calib_neta + by];
            }
        }
        /* event-weight factor from a 1-D lookup on a per-event column, variant independent */
        float evw = 1.0f;
        if (d->evw_table) evw = d->evw_table[find_bin_clamped(d->evw_x[iev], d->evw_edges, d->evw_nbins)];
        for (int32_t v = 0; v < V; ++v) {
            int32_t njet = 0, arg = -1;
            double ht = 0.0;
            float maxpt = -INFINITY, minpt = INFINITY;
            for (int64_t k = 0; k < nj; ++k) {
                float p = d->jets.pt[j0 + k];
                if (d->calib_table) {
                    float cv = corr[k] * d->calib_scales[v];   /* float32 multiply: table x scale */
                    p = p * cv;                                 /* float32 multiply: applied to pt only */
                }
                ptv[k] = p;
                int sel = (p > d->jet_pt_min) && (fabsf(d->jets.eta[j0 + k]) < d->jet_abs_eta_max);
                clean[k] = (uint8_t)(sel && !matched[k]);       /* step 4 */
                if (d->out_jet_mask) d->out_jet_mask[(int64_t)v * d->jets.n_objects + j0 + k] = clean[k];
                if (!clean[k]) continue;
                njet += 1;                                       /* step 5 */
                ht += (double)p;
                if (p > maxpt) maxpt = p;
                if (p < minpt) minpt = p;
                if (p == p && (arg < 0 || p > ptv[arg])) arg = (int32_t)k;
            }
            int32_t i1, i2;                                      /* step 6 */
            top2(ptv, clean, nj, &i1, &i2);
            float mjj = 0.0f, subpt = 0.0f;
            if (i1 >= 0 && i2 >= 0) {
                mjj = pair_mass_f64(ptv[i1], d->jets.eta[j0 + i1], d->jets.phi[j0 + i1], d->jets.mass[j0 + i1],
                                    ptv[i2], d->jets.eta[j0 + i2], d->jets.phi[j0 + i2], d->jets.mass[j0 + i2]);
                subpt = ptv[i2];
            }
            const int64_t o = (int64_t)v * N + iev;
            if (d->out_njet) d->out_njet[o] = njet;
            if (d->out_argmax) d->out_argmax[o] = arg;
            if (d->out_ht) d->out_ht[o] = (float)ht;
            if (d->out_maxpt) d->out_maxpt[o] = maxpt;
            if (d->out_minpt) d->out_minpt[o] = minpt;
            if (d->out_mjj) d->out_mjj[o] = mjj;
            if (d->out_subpt) d->out_subpt[o] = subpt;

            /* step 7: histograms */
            const float obs[HEPO_N_OBS] = { (float)njet, (float)ht, maxpt, minpt, mjj, subpt };
            for (int ob = 0; ob < HEPO_N_OBS; ++ob) {
                if (!d->axis_edges[ob]) continue;
                const int32_t nb = d->axis_nbins[ob];
                const int32_t s = hist_slot(obs[ob], d->axis_edges[ob], nb);
                if (counts) counts[(int64_t)v * slots_per_variant + obs_prefix[ob] + s] += 1;
                if (acc || acc2)
                    for (int32_t w = 0; w < W; ++w) {
                        float wf = d->weights ? d->weights[(int64_t)w * N + iev] : 1.0f;
                        if (d->evw_table) wf = wf * evw;        /* float32 multiply (hepo_event_weight_lookup) */
                        const double wt = (double)wf;
                        const int64_t slot = ((int64_t)v * slots_per_variant + obs_prefix[ob]) * W + (int64_t)w * (nb + 2) + s;
                        if (acc) acc[slot] += wt;
                        if (acc2) acc2[slot] += wt * wt;
                    }
            }
        }
    }
    free(ptv); free(matched); free(clean); free(corr);
    return 0;
}

static int chain_args_ok(const hepo_chain_desc* d)
{
    if (!d || d->n_events < 0 || d->n_variants < 1 || d->n_wvar < 1) return 0;
    if (d->n_events > 0 && (!d->jets.offsets || !d->muons.offsets)) return 0;
    if (!d->calib_table && d->n_variants != 1) return 0;
    if (d->evw_table && (!d->evw_x || !d->evw_edges || d->evw_nbins < 1)) return 0;
    return 1;
}

int32_t hepo_analysis_chain(const hepo_chain_desc* d)
{
    if (!chain_args_ok(d)) return -1;
    int64_t obs_prefix[HEPO_N_OBS + 1];
    const int64_t total = (int64_t)d->n_variants * d->n_wvar * chain_hist_layout(d, obs_prefix);
    double *acc = NULL, *acc2 = NULL;
    if (d->hist_sumw && total > 0) { acc = (double*)calloc((size_t)total, sizeof(double)); if (!acc) return -1; }
    if (d->hist_sumw2 && total > 0) { acc2 = (double*)calloc((size_t)total, sizeof(double)); if (!acc2) { free(acc); return -1; } }
    const int32_t rc = chain_event_range(d, 0, d->n_events, acc, acc2, d->hist_counts);
    if (rc == 0) {
        for (int64_t i = 0; acc && i < total; ++i) d->hist_sumw[i] = (float)((double)d->hist_sumw[i] + acc[i]);
        for (int64_t i = 0; acc2 && i < total; ++i) d->hist_sumw2[i] = (float)((double)d->hist_sumw2[i] + acc2[i]);
    }
    free(acc); free(acc2);
    return rc;
}

/* The same chain on all host cores (Listing 1's `prange` over events; Table I's thread columns):
 * contiguous event blocks, one per thread, each through chain_event_range with PRIVATE histogram accumulators
 * that are merged in thread order afterwards.  Per-event outputs are identical to the single-thread function's;
 * counts are identical; sumw / sumw2 differ only in the order of the float64 additions.  A timing baseline
 * (bench.py cpu_baseline); the single-thread function stays the checker. */
int32_t hepo_omp_max_threads(void)
{
#ifdef _OPENMP
    return (int32_t)omp_get_max_threads();
#else
    return 1;
#endif
}

int32_t hepo_analysis_chain_omp(const hepo_chain_desc* d, int32_t n_threads)
{
    if (!chain_args_ok(d)) return -1;
    if (n_threads < 1) n_threads = hepo_omp_max_threads();
    int64_t obs_prefix[HEPO_N_OBS + 1];
    const int64_t spv = chain_hist_layout(d, obs_prefix);
    const int64_t total = (int64_t)d->n_variants * d->n_wvar * spv;
    const int64_t ctotal = (int64_t)d->n_variants * spv;
    const int want1 = d->hist_sumw && total > 0, want2 = d->hist_sumw2 && total > 0, wantc = d->hist_counts && ctotal > 0;
    double* acc = want1 ? (double*)calloc((size_t)(total * n_threads), sizeof(double)) : NULL;
    double* acc2 = want2 ? (double*)calloc((size_t)(total * n_threads), sizeof(double)) : NULL;
    int64_t* cnt = wantc ? (int64_t*)calloc((size_t)(ctotal * n_threads), sizeof(int64_t)) : NULL;
    if ((want1 && !acc) || (want2 && !acc2) || (wantc && !cnt)) { free(acc); free(acc2); free(cnt); return -1; }
    int32_t rc = 0;
    const int64_t N = d->n_events;
#ifdef _OPENMP
#pragma omp parallel for num_threads(n_threads) schedule(static, 1)
#endif
    for (int32_t t = 0; t < n_threads; ++t) {
        const int64_t e0 = N * t / n_threads, e1 = N * (t + 1) / n_threads;
        const int32_t r = chain_event_range(d, e0, e1, acc ? acc + total * t : NULL, acc2 ? acc2 + total * t : NULL,
                                            cnt ? cnt + ctotal * t : NULL);
        if (r != 0) {
#ifdef _OPENMP
#pragma omp critical
#endif
            rc = r;
        }
    }
    if (rc == 0) {
        for (int64_t i = 0; acc && i < total; ++i) {
            double s = 0.0;
            for (int32_t t = 0; t < n_threads; ++t) s += acc[total * t + i];
            d->hist_sumw[i] = (float)((double)d->hist_sumw[i] + s);
        }
        for (int64_t i = 0; acc2 && i < total; ++i) {
            double s = 0.0;
            for (int32_t t = 0; t < n_threads; ++t) s += acc2[total * t + i];
            d->hist_sumw2[i] = (float)((double)d->hist_sumw2[i] + s);
        }
        for (int64_t i = 0; cnt && i < ctotal; ++i)
            for (int32_t t = 0; t < n_threads; ++t) d->hist_counts[i] += cnt[ctotal * t + i];
    }
    free(acc); free(acc2); free(cnt);
    return rc;
}

/* ---- SURVEY.md 8(f-1) ---------------------------------------------------------------------------------- */

/* position (column index) of the index-th counted element of row e, or -1 */
static int64_t nth_position(const int64_t* offsets, int64_t e, int64_t content_base, const uint8_t* mask_content, int32_t index)
{
    int32_t seen = 0;
    for (int64_t g = offsets[e]; g < offsets[e + 1]; ++g) {
        const int64_t i = g - content_base;
        if (mask_content && !mask_content[i]) continue;
        if (seen == index) return i;
        ++seen;
    }
    return -1;
}

int32_t hepo_get_in_offsets(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index, float fill, float* out)
{
    if (!seg_args_ok(offsets, n_events, out) || index < 0) return -1;
    for (int64_t e = 0; e < n_events; ++e) {
        out[e] = fill;
        if (mask_rows && !mask_rows[e]) continue;
        const int64_t i = nth_position(offsets, e, content_base, mask_content, index);
        if (i >= 0) out[e] = data[i];
    }
    return 0;
}

int32_t hepo_set_in_offsets(float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                            const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index,
                            const float* values, float value)
{
    if (!seg_args_ok(offsets, n_events, data) || index < 0) return -1;
    for (int64_t e = 0; e < n_events; ++e) {
        if (mask_rows && !mask_rows[e]) continue;
        const int64_t i = nth_position(offsets, e, content_base, mask_content, index);
        if (i >= 0) data[i] = values ? values[e] : value;
    }
    return 0;
}

int32_t hepo_select_opposite_sign(const float* pt, const int32_t* charge, const int64_t* offsets, int64_t n_events,
                                  int64_t content_base, const uint8_t* mask_rows, const uint8_t* mask_content,
                                  uint8_t* out_mask)
{
    if (!seg_args_ok(offsets, n_events, out_mask) || !charge) return -1;
    for (int64_t e = 0; e < n_events; ++e) {
        const int64_t g0 = offsets[e], g1 = offsets[e + 1];
        for (int64_t g = g0; g < g1; ++g) out_mask[g - content_base] = 0;
        if (mask_rows && !mask_rows[e]) continue;
        /* leading object: strict > keeps the first index among equal pt */
        int64_t lead = -1;
        for (int64_t g = g0; g < g1; ++g) {
            const int64_t i = g - content_base;
            if (mask_content && !mask_content[i]) continue;
            if (pt[i] != pt[i]) continue;
            if (lead < 0 || pt[i] > pt[lead]) lead = i;
        }
        if (lead < 0) continue;
        /* highest-pt object of the opposite sign */
        int64_t part = -1;
        for (int64_t g = g0; g < g1; ++g) {
            const int64_t i = g - content_base;
            if (mask_content && !mask_content[i]) continue;
            if (pt[i] != pt[i]) continue;
            if ((int64_t)charge[i] * (int64_t)charge[lead] >= 0) continue;
            if (part < 0 || pt[i] > pt[part]) part = i;
        }
        if (part < 0) continue;
        out_mask[lead] = 1;
        out_mask[part] = 1;
    }
    return 0;
}

/* ---- SURVEY.md 8(f-2) ---------------------------------------------------------------------------------- */

int32_t hepo_lookup_interp(const float* x, int64_t n, const float* xs, const float* ys, int32_t nk, float* out)
{
    if (n < 0 || nk < 2 || !xs || !ys || (n > 0 && (!x || !out))) return -1;
    for (int64_t i = 0; i < n; ++i) {
        const float v = x[i];
        if (v != v) { out[i] = v; continue; }
        if (v <= xs[0]) { out[i] = ys[0]; continue; }
        if (v >= xs[nk - 1]) { out[i] = ys[nk - 1]; continue; }
        int32_t lo = 0, hi = nk - 1;               /* xs[lo] <= v < xs[hi] */
        while (hi - lo > 1) {
            const int32_t mid = (lo + hi) / 2;
            if (v >= xs[mid]) lo = mid; else hi = mid;
        }
        const double x0 = xs[lo], x1 = xs[lo + 1], y0 = ys[lo], y1 = ys[lo + 1];
        out[i] = (float)(y0 + ((double)v - x0) * (y1 - y0) / (x1 - x0));
    }
    return 0;
}

int32_t hepo_fill_histogram_2d(const float* x, const float* y, const float* weights, int64_t n,
                               const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                               float* sumw, int64_t* counts)
{
    if (n < 0 || nx < 1 || ny < 1 || !edges_x || !edges_y || (n > 0 && (!x || !y))) return -1;
    const size_t slots = ((size_t)nx + 2) * ((size_t)ny + 2);
    double* acc = (double*)calloc(slots, sizeof(double));
    if (!acc) return -1;
    for (int64_t i = 0; i < n; ++i) {
        const size_t s = (size_t)hist_slot(x[i], edges_x, nx) * ((size_t)ny + 2) + (size_t)hist_slot(y[i], edges_y, ny);
        acc[s] += weights ? (double)weights[i] : 1.0;
        if (counts) counts[s] += 1;
    }
    if (sumw)
        for (size_t s = 0; s < slots; ++s) sumw[s] = (float)((double)sumw[s] + acc[s]);
    free(acc);
    return 0;
}

/* the same with the sum of squared weights per slot (see hepo_fill_histogram_w2) */
int32_t hepo_fill_histogram_2d_w2(const float* x, const float* y, const float* weights, int64_t n,
                                  const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                                  float* sumw, float* sumw2, int64_t* counts)
{
    if (n < 0 || nx < 1 || ny < 1 || !edges_x || !edges_y || (n > 0 && (!x || !y))) return -1;
    const size_t slots = ((size_t)nx + 2) * ((size_t)ny + 2);
    double* acc = (double*)calloc(2 * slots, sizeof(double));
    if (!acc) return -1;
    double* acc2 = acc + slots;
    for (int64_t i = 0; i < n; ++i) {
        const size_t s = (size_t)hist_slot(x[i], edges_x, nx) * ((size_t)ny + 2) + (size_t)hist_slot(y[i], edges_y, ny);
        const double w = weights ? (double)weights[i] : 1.0;
        acc[s] += w;
        acc2[s] += w * w;
        if (counts) counts[s] += 1;
    }
    for (size_t s = 0; s < slots; ++s) {
        if (sumw) sumw[s] = (float)((double)sumw[s] + acc[s]);
        if (sumw2) sumw2[s] = (float)((double)sumw2[s] + acc2[s]);
    }
    free(acc);
    return 0;
}

/* ---- SURVEY.md 8(f-3) ---------------------------------------------------------------------------------- */

int32_t hepo_triplet_mass(const float* pt, const float* eta, const float* phi, const float* mass,
                          const int64_t* offsets, int64_t n_events, int64_t content_base,
                          const uint8_t* mask_rows, const uint8_t* mask_content, float target,
                          float* out_mass, int32_t* out_idx)
{
    if (!seg_args_ok(offsets, n_events, out_mass)) return -1;
    for (int64_t e = 0; e < n_events; ++e) {
        out_mass[e] = 0.0f;
        if (out_idx) { out_idx[3 * e] = out_idx[3 * e + 1] = out_idx[3 * e + 2] = -1; }
        if (mask_rows && !mask_rows[e]) continue;
        const int64_t g0 = offsets[e], g1 = offsets[e + 1];
        double best = 0.0, best_m = 0.0;
        int have = 0;
        for (int64_t a = g0; a < g1; ++a) {
            if (mask_content && !mask_content[a - content_base]) continue;
            for (int64_t b = a + 1; b < g1; ++b) {
                if (mask_content && !mask_content[b - content_base]) continue;
                for (int64_t c = b + 1; c < g1; ++c) {
                    if (mask_content && !mask_content[c - content_base]) continue;
                    const int64_t id[3] = {a - content_base, b - content_base, c - content_base};
                    double E = 0, px = 0, py = 0, pz = 0;
                    for (int t = 0; t < 3; ++t) {
                        const double p = pt[id[t]], m = mass[id[t]];
                        const double ch = cosh((double)eta[id[t]]);
                        px += p * cos((double)phi[id[t]]);
                        py += p * sin((double)phi[id[t]]);
                        pz += p * sinh((double)eta[id[t]]);
                        E += sqrt(p * p * ch * ch + m * m);
                    }
                    double m2 = E * E - px * px - py * py - pz * pz;
                    if (!(m2 > 0.0)) m2 = 0.0;
                    const double M = sqrt(m2);
                    const double d = fabs(M - (double)target);
                    if (!have || d < best) {            /* strict <: the first triplet in (i, j, k) order wins ties */
                        have = 1; best = d; best_m = M;
                        if (out_idx) {
                            out_idx[3 * e] = (int32_t)(a - g0);
                            out_idx[3 * e + 1] = (int32_t)(b - g0);
                            out_idx[3 * e + 2] = (int32_t)(c - g0);
                        }
                    }
                }
            }
        }
        if (have) out_mass[e] = (float)best_m;
    }
    return 0;
}

int32_t hepo_validate_offsets(const int64_t* offsets, int64_t n_events, int64_t content_base, int64_t n_objects, int64_t* n_bad)
{
    if (!offsets || n_events < 0 || !n_bad) return -1;
    int64_t bad = 0;
    if (offsets[0] < content_base) ++bad;
    for (int64_t e = 0; e < n_events; ++e)
        if (offsets[e] > offsets[e + 1]) ++bad;
    if (offsets[n_events] - content_base > n_objects) ++bad;
    *n_bad = bad;
    return 0;
}
