// hepk_chain.cu — the fused analysis chain (include/hepk.h, hepk_analysis_chain).
//
// One persistent kernel.  Each CTA walks tiles of TILE events; per tile it
//   1. turns the three int64 offsets slices into tile-local int32 offsets in shared memory,
//   2. stages the tile's contiguous column slices (jets: pt, eta, phi, mass; leptons: pt, eta, phi)
//      into shared memory with TMA 1-D bulk copies (cp.async.bulk + mbarrier), and meanwhile expands
//      the offsets into a per-jet event id,
//   3. phase 1, one thread per JET (flat, every lane busy): selection, dR cleaning against the event's
//      leptons, calibration lookup; the verdict is folded into the staged pt (NaN = not clean),
//   4. phase 2, one thread per EVENT: count / sum / min / top-2 over the event's jets from shared
//      memory, leading-pair mass, coalesced per-event outputs, shared-memory histograms,
// and merges its privatised histograms into float64 accumulators (workspace) every few tiles.
// A tile that does not fit the staging buffers is processed in pieces; a single event that does not fit
// goes through a plain per-event loop on global memory.
#include <string.h>

#include "hepk_common.cuh"

namespace hepk {

struct ChainParams {
    long long n_events;
    const long long* joff; long long jbase; long long jn;
    const float *jpt, *jeta, *jphi, *jmass;
    const long long* moff; long long mbase; long long mn;
    const float *mpt, *meta, *mphi;
    const long long* eoff; long long ebase; long long en;     // eoff == nullptr: no electrons
    const float *ept, *eeta, *ephi;
    float jet_pt_min, jet_abs_eta_max, lep_pt_min, dr2_max;
    const float* cal_pt_edges; const float* cal_eta_edges; const float* cal_table;
    int cal_npt, cal_neta;
    float scales[HEPK_MAX_VARIANTS];
    int V, W;
    const float* weights;
    const float* axis_edges[HEPK_N_OBS];
    int axis_nbins[HEPK_N_OBS];
    int obs_prefix[HEPK_N_OBS + 1];      // slot prefix of the active observables; [HEPK_N_OBS] = slots per variant
    int edge_prefix[HEPK_N_OBS + 1];     // float prefix of the staged edges
    int* out_njet; int* out_argmax;
    float *out_ht, *out_maxpt, *out_minpt, *out_mjj, *out_subpt;
    unsigned char* out_jet_mask;
    double* hist_acc;                    // workspace: [V][active o][W][nbins_o+2] float64, or nullptr
    unsigned long long* hist_counts;     // [V][active o][nbins_o+2], or nullptr
    int cap_j, cap_l;
    long long n_tiles;
    int flush_tiles;
};

namespace dev {

struct ChainSmem {
    uint64_t* bar;
    int *loc_j, *loc_m, *loc_e;
    float *jpt, *jeta, *jphi, *jmass, *corr;
    unsigned short* evid;
    float *mpt, *meta, *mphi, *ept, *eeta, *ephi;
    float *edges, *axis_lo, *axis_inv;
    float *cal_pt_edges, *cal_eta_edges, *cal_table;
    float* h_sumw;
    unsigned int* h_cnt;
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// One layout function used by the host (size) and the device (pointers).
template <int TILE>
__host__ __device__ inline size_t chain_smem_layout(const ChainParams& P, bool calib, unsigned char* base, ChainSmem* s)
{
    size_t o = 0;
    auto take = [&](size_t bytes, size_t al) { o = align_up(o, al); size_t r = o; o += bytes; return r; };
    size_t r;
    r = take(8, 8); if (s) s->bar = (uint64_t*)(base + r);
    r = take((TILE + 1) * 4, 4); if (s) s->loc_j = (int*)(base + r);
    r = take((TILE + 1) * 4, 4); if (s) s->loc_m = (int*)(base + r);
    r = take((TILE + 1) * 4, 4); if (s) s->loc_e = (int*)(base + r);
    const size_t cj = (size_t)P.cap_j * 4, cl = (size_t)P.cap_l * 4;
    r = take(cj, 16); if (s) s->jpt = (float*)(base + r);
    r = take(cj, 16); if (s) s->jeta = (float*)(base + r);
    r = take(cj, 16); if (s) s->jphi = (float*)(base + r);
    r = take(cj, 16); if (s) s->jmass = (float*)(base + r);
    r = take(calib ? cj : 0, 16); if (s) s->corr = (float*)(base + r);
    r = take((size_t)P.cap_j * 2, 4); if (s) s->evid = (unsigned short*)(base + r);
    r = take(cl, 16); if (s) s->mpt = (float*)(base + r);
    r = take(cl, 16); if (s) s->meta = (float*)(base + r);
    r = take(cl, 16); if (s) s->mphi = (float*)(base + r);
    r = take(cl, 16); if (s) s->ept = (float*)(base + r);
    r = take(cl, 16); if (s) s->eeta = (float*)(base + r);
    r = take(cl, 16); if (s) s->ephi = (float*)(base + r);
    r = take((size_t)P.edge_prefix[HEPK_N_OBS] * 4, 4); if (s) s->edges = (float*)(base + r);
    r = take(HEPK_N_OBS * 4, 4); if (s) s->axis_lo = (float*)(base + r);
    r = take(HEPK_N_OBS * 4, 4); if (s) s->axis_inv = (float*)(base + r);
    r = take(calib ? (size_t)(P.cal_npt + 1) * 4 : 0, 4); if (s) s->cal_pt_edges = (float*)(base + r);
    r = take(calib ? (size_t)(P.cal_neta + 1) * 4 : 0, 4); if (s) s->cal_eta_edges = (float*)(base + r);
    r = take(calib ? (size_t)P.cal_npt * P.cal_neta * 4 : 0, 4); if (s) s->cal_table = (float*)(base + r);
    const size_t spv = (size_t)P.obs_prefix[HEPK_N_OBS];
    r = take(P.hist_acc ? spv * P.V * P.W * 4 : 0, 4); if (s) s->h_sumw = (float*)(base + r);
    r = take(P.hist_counts ? spv * P.V * 4 : 0, 4); if (s) s->h_cnt = (unsigned int*)(base + r);
    return align_up(o, 16);
}

// Per event and variant: leading-pair mass, outputs, histograms.  Shared by the tile path and the
// per-event fallback.  `k1`/`k2` leading jets' (eta, phi, mass) are passed in by value.
__device__ __forceinline__ void finish_event(const ChainParams& P, const ChainSmem& S, long long ev, int v,
                                             int cnt, float sum, float mn, const Top2& top,
                                             float eta1, float phi1, float m1, float eta2, float phi2, float m2)
{
    float mjj = 0.0f, subpt = 0.0f;
    if (top.i2 >= 0) {
        subpt = top.b2;
        mjj = pair_mass_f32(top.b1, eta1, phi1, m1, top.b2, eta2, phi2, m2);
        if (P.axis_edges[HEPK_OBS_MJJ] && (P.hist_acc || P.hist_counts)) {
            // the bin of mjj is decided by the float64-defined value: refine when the fast value is near an edge
            const float* ed = S.edges + P.edge_prefix[HEPK_OBS_MJJ];
            const int nb = P.axis_nbins[HEPK_OBS_MJJ];
            const int slot = hist_slot(mjj, ed, nb, S.axis_lo[HEPK_OBS_MJJ], S.axis_inv[HEPK_OBS_MJJ]);
            const float band = fmaf(mjj, HEPK_MASS_GUARD_REL, HEPK_MASS_GUARD_ABS);
            const bool near_lo = slot >= 1 && mjj - ed[slot - 1] <= band;
            const bool near_hi = slot <= nb && ed[slot] - mjj <= band;
            if (near_lo || near_hi) mjj = pair_mass_f64(top.b1, eta1, phi1, m1, top.b2, eta2, phi2, m2);
        }
    }
    const long long o = (long long)v * P.n_events + ev;
    if (P.out_njet) P.out_njet[o] = cnt;
    if (P.out_argmax) P.out_argmax[o] = top.i1;
    if (P.out_ht) P.out_ht[o] = sum;
    if (P.out_maxpt) P.out_maxpt[o] = top.b1;
    if (P.out_minpt) P.out_minpt[o] = mn;
    if (P.out_mjj) P.out_mjj[o] = mjj;
    if (P.out_subpt) P.out_subpt[o] = subpt;

    if (!P.hist_acc && !P.hist_counts) return;
    const float obs[HEPK_N_OBS] = {(float)cnt, sum, top.b1, mn, mjj, subpt};
    const int spv = P.obs_prefix[HEPK_N_OBS];
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        const int slot = hist_slot(obs[ob], S.edges + P.edge_prefix[ob], nb, S.axis_lo[ob], S.axis_inv[ob]);
        if (P.hist_counts) atomicAdd(&S.h_cnt[v * spv + P.obs_prefix[ob] + slot], 1u);
        if (P.hist_acc) {
            float* h = S.h_sumw + (size_t)(v * spv + P.obs_prefix[ob]) * P.W + slot;
            for (int w = 0; w < P.W; ++w) {
                const float wt = P.weights ? __ldg(P.weights + (long long)w * P.n_events + ev) : 1.0f;
                atomicAdd(h + w * (nb + 2), wt);
            }
        }
    }
}

// dR match of one jet against one lepton collection of event `ev`, straight from global memory.
__device__ inline bool match_global(const ChainParams& P, float eta, float phi, const long long* off, long long base,
                                    const float* lpt, const float* leta, const float* lphi, long long ev)
{
    for (long long g = off[ev]; g < off[ev + 1]; ++g) {
        const long long m = g - base;
        if (!(lpt[m] > P.lep_pt_min)) continue;
        if (dr2_exact(eta, phi, leta[m], lphi[m]) < P.dr2_max) return true;
    }
    return false;
}

// Fallback for an event too large for the staging buffers: the paper's own loop shape (Listing 1),
// one thread, everything from global memory.  Slow; only pathological inputs get here.
template <bool CALIB>
__device__ __noinline__ void chain_event_global(const ChainParams& P, const ChainSmem& S, long long ev)
{
    const long long g0 = P.joff[ev], g1 = P.joff[ev + 1];
    for (int v = 0; v < P.V; ++v) {
        int cnt = 0;
        double sum = 0.0;
        float mn = CUDART_INF_F;
        Top2 top;
        top.init();
        for (long long g = g0; g < g1; ++g) {
            const long long j = g - P.jbase;
            const float eta = P.jeta[j], phi = P.jphi[j];
            float p = P.jpt[j];
            if (CALIB) {
                const int bx = find_bin_clamped(p, S.cal_pt_edges, P.cal_npt);
                const int by = find_bin_clamped(eta, S.cal_eta_edges, P.cal_neta);
                p = __fmul_rn(p, __fmul_rn(S.cal_table[bx * P.cal_neta + by], P.scales[v]));
            }
            bool clean = (p > P.jet_pt_min) && (fabsf(eta) < P.jet_abs_eta_max);
            if (clean) {
                bool matched = match_global(P, eta, phi, P.moff, P.mbase, P.mpt, P.meta, P.mphi, ev);
                if (!matched && P.eoff) matched = match_global(P, eta, phi, P.eoff, P.ebase, P.ept, P.eeta, P.ephi, ev);
                clean = !matched;
            }
            if (P.out_jet_mask) P.out_jet_mask[(long long)v * P.jn + j] = clean ? 1 : 0;
            if (clean) {
                cnt++;
                sum += (double)p;
                mn = fminf(mn, p);
                top.push(p, (int)(g - g0));
            }
        }
        float e1 = 0, p1 = 0, m1 = 0, e2 = 0, p2 = 0, m2 = 0;
        if (top.i2 >= 0) {
            const long long a = g0 - P.jbase + top.i1, b = g0 - P.jbase + top.i2;
            e1 = P.jeta[a]; p1 = P.jphi[a]; m1 = P.jmass[a];
            e2 = P.jeta[b]; p2 = P.jphi[b]; m2 = P.jmass[b];
        }
        finish_event(P, S, ev, v, cnt, (float)sum, mn, top, e1, p1, m1, e2, p2, m2);
    }
}

template <int TILE>
__device__ __forceinline__ void flush_hist(const ChainParams& P, const ChainSmem& S, int tid)
{
    const int spv = P.obs_prefix[HEPK_N_OBS];
    if (P.hist_acc) {
        const int n = spv * P.V * P.W;
        for (int i = tid; i < n; i += TILE) {
            const float x = S.h_sumw[i];
            if (x != 0.0f) { atomicAdd(P.hist_acc + i, (double)x); S.h_sumw[i] = 0.0f; }
        }
    }
    if (P.hist_counts) {
        const int n = spv * P.V;
        for (int i = tid; i < n; i += TILE) {
            const unsigned int c = S.h_cnt[i];
            if (c) { atomicAdd(P.hist_counts + i, (unsigned long long)c); S.h_cnt[i] = 0u; }
        }
    }
}

template <int TILE, bool CALIB>
__global__ void __launch_bounds__(TILE) chain_kernel(const __grid_constant__ ChainParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ChainSmem S;
    chain_smem_layout<TILE>(P, CALIB, smem_raw, &S);
    const int tid = threadIdx.x;
    const bool has_el = P.eoff != nullptr;

    // ---- one-time setup: barrier, axis edges, calibration tables, zeroed histograms
    if (tid == 0) { mbar_init(S.bar, 1); fence_mbar_init(); }
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        for (int i = tid; i <= nb; i += TILE) S.edges[P.edge_prefix[ob] + i] = P.axis_edges[ob][i];
        if (tid == 0) {
            const float lo = P.axis_edges[ob][0], hi = P.axis_edges[ob][nb];
            S.axis_lo[ob] = lo;
            S.axis_inv[ob] = (float)nb / (hi - lo);
        }
    }
    if (CALIB) {
        for (int i = tid; i <= P.cal_npt; i += TILE) S.cal_pt_edges[i] = P.cal_pt_edges[i];
        for (int i = tid; i <= P.cal_neta; i += TILE) S.cal_eta_edges[i] = P.cal_eta_edges[i];
        for (int i = tid; i < P.cal_npt * P.cal_neta; i += TILE) S.cal_table[i] = P.cal_table[i];
    }
    {
        const int spv = P.obs_prefix[HEPK_N_OBS];
        if (P.hist_acc) for (int i = tid; i < spv * P.V * P.W; i += TILE) S.h_sumw[i] = 0.0f;
        if (P.hist_counts) for (int i = tid; i < spv * P.V; i += TILE) S.h_cnt[i] = 0u;
    }
    __syncthreads();

    uint32_t parity = 0;
    int tiles_since_flush = 0;
    const int cap_j = P.cap_j - 8, cap_l = P.cap_l - 8;     // room for the alignment shift and padding

    for (long long tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x) {
        const long long e0 = tile * TILE;
        const int ne = (int)((P.n_events - e0) < TILE ? (P.n_events - e0) : TILE);
        // ---- 1. tile-local offsets
        const long long jb = P.joff[e0], mb = P.moff[e0], eb = has_el ? P.eoff[e0] : 0;
        for (int i = tid; i <= ne; i += TILE) {
            S.loc_j[i] = (int)(P.joff[e0 + i] - jb);
            S.loc_m[i] = (int)(P.moff[e0 + i] - mb);
            S.loc_e[i] = has_el ? (int)(P.eoff[e0 + i] - eb) : 0;
        }
        __syncthreads();

        int ev0 = 0;
        while (ev0 < ne) {
            // ---- how many events from ev0 fit the staging buffers
            const int bj = S.loc_j[ev0], bm = S.loc_m[ev0], be = S.loc_e[ev0];
            int n_fit;
            if (S.loc_j[ne] - bj <= cap_j && S.loc_m[ne] - bm <= cap_l && S.loc_e[ne] - be <= cap_l) {
                n_fit = ne - ev0;
            } else {
                const bool f = tid >= ev0 && tid < ne && S.loc_j[tid + 1] - bj <= cap_j &&
                               S.loc_m[tid + 1] - bm <= cap_l && S.loc_e[tid + 1] - be <= cap_l;
                n_fit = __syncthreads_count(f);
            }
            if (n_fit == 0) {   // a single event larger than the buffers
                if (tid == 0) chain_event_global<CALIB>(P, S, e0 + ev0);
                ev0 += 1;
                __syncthreads();
                continue;
            }
            const int ev1 = ev0 + n_fit;
            const int nj = S.loc_j[ev1] - bj, nm = S.loc_m[ev1] - bm, nel = S.loc_e[ev1] - be;

            // ---- 2. stage the column slices with bulk copies
            long long a0;
            int sh_pt, sh_eta, sh_phi, sh_mass, sh_mpt, sh_meta, sh_mphi, sh_ept = 0, sh_eeta = 0, sh_ephi = 0;
            const long long lj0 = jb + bj - P.jbase, lm0 = mb + bm - P.mbase, le0 = eb + be - P.ebase;
            if (tid == 0) fence_proxy_async_smem();
            uint32_t bytes = 0;
            bytes += stage_column(S.jpt, P.jpt, lj0, lj0 + nj, P.jn, S.bar, tid, 0, &a0);   sh_pt = (int)(lj0 - a0);
            bytes += stage_column(S.jeta, P.jeta, lj0, lj0 + nj, P.jn, S.bar, tid, 0, &a0); sh_eta = (int)(lj0 - a0);
            bytes += stage_column(S.jphi, P.jphi, lj0, lj0 + nj, P.jn, S.bar, tid, 0, &a0); sh_phi = (int)(lj0 - a0);
            bytes += stage_column(S.jmass, P.jmass, lj0, lj0 + nj, P.jn, S.bar, tid, 0, &a0); sh_mass = (int)(lj0 - a0);
            bytes += stage_column(S.mpt, P.mpt, lm0, lm0 + nm, P.mn, S.bar, tid, 0, &a0);   sh_mpt = (int)(lm0 - a0);
            bytes += stage_column(S.meta, P.meta, lm0, lm0 + nm, P.mn, S.bar, tid, 0, &a0); sh_meta = (int)(lm0 - a0);
            bytes += stage_column(S.mphi, P.mphi, lm0, lm0 + nm, P.mn, S.bar, tid, 0, &a0); sh_mphi = (int)(lm0 - a0);
            if (has_el) {
                bytes += stage_column(S.ept, P.ept, le0, le0 + nel, P.en, S.bar, tid, 0, &a0);   sh_ept = (int)(le0 - a0);
                bytes += stage_column(S.eeta, P.eeta, le0, le0 + nel, P.en, S.bar, tid, 0, &a0); sh_eeta = (int)(le0 - a0);
                bytes += stage_column(S.ephi, P.ephi, le0, le0 + nel, P.en, S.bar, tid, 0, &a0); sh_ephi = (int)(le0 - a0);
            }
            if (tid == 0) mbar_arrive_expect_tx(S.bar, bytes);

            // ---- meanwhile: expand offsets into a per-jet event id (needs only the offsets)
            if (tid < n_fit) {
                const int k0 = S.loc_j[ev0 + tid] - bj, k1 = S.loc_j[ev0 + tid + 1] - bj;
                for (int k = k0; k < k1; ++k) S.evid[k] = (unsigned short)tid;
            }
            mbar_wait(S.bar, parity);
            parity ^= 1u;
            __syncthreads();

            // ---- lepton selection folded into the staged eta (NaN never matches)
            for (int m = tid; m < nm; m += TILE)
                if (!(S.mpt[m + sh_mpt] > P.lep_pt_min)) S.meta[m + sh_meta] = CUDART_NAN_F;
            for (int m = tid; m < nel; m += TILE)
                if (!(S.ept[m + sh_ept] > P.lep_pt_min)) S.eeta[m + sh_eeta] = CUDART_NAN_F;
            __syncthreads();

            // ---- 3. phase 1: one thread per jet
            for (int j = tid; j < nj; j += TILE) {
                const float pt = S.jpt[j + sh_pt], eta = S.jeta[j + sh_eta], phi = S.jphi[j + sh_phi];
                const int a = ev0 + (int)S.evid[j];
                bool matched = false;
                {
                    const int m0 = S.loc_m[a] - bm, m1 = S.loc_m[a + 1] - bm;
                    for (int m = m0; m < m1; ++m)
                        matched |= dr2_exact(eta, phi, S.meta[m + sh_meta], S.mphi[m + sh_mphi]) < P.dr2_max;
                    const int q0 = S.loc_e[a] - be, q1 = S.loc_e[a + 1] - be;
                    for (int m = q0; m < q1; ++m)
                        matched |= dr2_exact(eta, phi, S.eeta[m + sh_eeta], S.ephi[m + sh_ephi]) < P.dr2_max;
                }
                const bool base = (fabsf(eta) < P.jet_abs_eta_max) && !matched;
                if (!CALIB) {
                    const bool clean = base && (pt > P.jet_pt_min);
                    if (P.out_jet_mask) P.out_jet_mask[lj0 + j] = clean ? 1 : 0;
                    if (!clean) S.jpt[j + sh_pt] = CUDART_NAN_F;
                } else {
                    const int bx = find_bin_clamped(pt, S.cal_pt_edges, P.cal_npt);
                    const int by = find_bin_clamped(eta, S.cal_eta_edges, P.cal_neta);
                    const float c = S.cal_table[bx * P.cal_neta + by];
                    S.corr[j] = base ? c : CUDART_NAN_F;
                    if (P.out_jet_mask)
                        for (int v = 0; v < P.V; ++v)
                            P.out_jet_mask[(long long)v * P.jn + lj0 + j] =
                                (base && (__fmul_rn(pt, __fmul_rn(c, P.scales[v])) > P.jet_pt_min)) ? 1 : 0;
                }
            }
            __syncthreads();

            // ---- 4. phase 2: one thread per event
            if (tid < n_fit) {
                const int k0 = S.loc_j[ev0 + tid] - bj, k1 = S.loc_j[ev0 + tid + 1] - bj;
                for (int v = 0; v < P.V; ++v) {
                    const float sv = P.scales[v];
                    int cnt = 0;
                    double sum = 0.0;      // float64: exact for these inputs, so HT and its bin do not depend on the order (R15)
                    float mn = CUDART_INF_F;
                    Top2 top;
                    top.init();
                    for (int k = k0; k < k1; ++k) {
                        float p = S.jpt[k + sh_pt];
                        if (CALIB) p = __fmul_rn(p, __fmul_rn(S.corr[k], sv));
                        if (p > P.jet_pt_min) {
                            cnt++;
                            sum += (double)p;
                            mn = fminf(mn, p);
                            top.push(p, k - k0);
                        }
                    }
                    float e1 = 0, p1 = 0, m1 = 0, e2 = 0, p2 = 0, m2 = 0;
                    if (top.i2 >= 0) {
                        const int a = k0 + top.i1, b = k0 + top.i2;
                        e1 = S.jeta[a + sh_eta]; p1 = S.jphi[a + sh_phi]; m1 = S.jmass[a + sh_mass];
                        e2 = S.jeta[b + sh_eta]; p2 = S.jphi[b + sh_phi]; m2 = S.jmass[b + sh_mass];
                    }
                    finish_event(P, S, e0 + ev0 + tid, v, cnt, (float)sum, mn, top, e1, p1, m1, e2, p2, m2);
                }
            }
            fence_proxy_async_smem();   // this thread's generic writes to the staging buffers precede the next bulk copies
            __syncthreads();
            ev0 = ev1;
        }
        if (++tiles_since_flush >= P.flush_tiles) {
            flush_hist<TILE>(P, S, tid);
            tiles_since_flush = 0;
            __syncthreads();
        }
    }
    __syncthreads();
    flush_hist<TILE>(P, S, tid);
}

// sumw[i] = float32(float64(sumw[i]) + acc[i])
__global__ void chain_finalize_hist(float* __restrict__ sumw, const double* __restrict__ acc, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) sumw[i] = (float)((double)sumw[i] + acc[i]);
}

}  // namespace dev

// ------------------------------------------------------------------------------------------ host side
static int32_t chain_validate(const hepk_chain_desc* d)
{
    HEPK_REQUIRE(d != nullptr, "descriptor is NULL");
    HEPK_REQUIRE(d->n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(d->n_variants >= 1 && d->n_variants <= HEPK_MAX_VARIANTS, "n_variants out of range");
    HEPK_REQUIRE(d->n_wvar >= 1 && d->n_wvar <= HEPK_MAX_WVAR, "n_wvar out of range");
    HEPK_REQUIRE(d->calib_table || d->n_variants == 1, "n_variants > 1 needs a calibration table");
    if (d->calib_table) {
        HEPK_REQUIRE(d->calib_pt_edges && d->calib_eta_edges, "calibration edges are NULL");
        HEPK_REQUIRE(d->calib_npt >= 1 && d->calib_neta >= 1, "calibration table has no bins");
    }
    if (d->n_events > 0) {
        HEPK_REQUIRE(d->jets.offsets && d->muons.offsets, "jets/muons offsets are NULL");
        HEPK_REQUIRE(d->jets.n_objects >= 0 && d->muons.n_objects >= 0, "n_objects < 0");
        HEPK_REQUIRE(d->jets.n_objects == 0 || (d->jets.pt && d->jets.eta && d->jets.phi && d->jets.mass), "jet column is NULL");
        HEPK_REQUIRE(d->muons.n_objects == 0 || (d->muons.pt && d->muons.eta && d->muons.phi), "muon column is NULL");
        if (d->electrons.offsets)
            HEPK_REQUIRE(d->electrons.n_objects == 0 || (d->electrons.pt && d->electrons.eta && d->electrons.phi),
                         "electron column is NULL");
    }
    for (int o = 0; o < HEPK_N_OBS; ++o)
        if (d->axis_edges[o]) HEPK_REQUIRE(d->axis_nbins[o] >= 1, "histogram axis has no bins");
    return HEPK_OK;
}

static long long hist_slots_per_variant(const hepk_chain_desc* d)
{
    long long s = 0;
    for (int o = 0; o < HEPK_N_OBS; ++o)
        if (d->axis_edges[o]) s += d->axis_nbins[o] + 2;
    return s;
}

static int round_up4(long long x) { return (int)((x + 3) / 4 * 4); }

template <int TILE>
static int32_t chain_launch(const hepk_chain_desc* d, void* workspace, cudaStream_t st)
{
    ChainParams P;
    memset(&P, 0, sizeof(P));
    P.n_events = d->n_events;
    P.joff = (const long long*)d->jets.offsets; P.jbase = d->jets.content_base; P.jn = d->jets.n_objects;
    P.jpt = d->jets.pt; P.jeta = d->jets.eta; P.jphi = d->jets.phi; P.jmass = d->jets.mass;
    P.moff = (const long long*)d->muons.offsets; P.mbase = d->muons.content_base; P.mn = d->muons.n_objects;
    P.mpt = d->muons.pt; P.meta = d->muons.eta; P.mphi = d->muons.phi;
    P.eoff = (const long long*)d->electrons.offsets; P.ebase = d->electrons.content_base; P.en = d->electrons.n_objects;
    P.ept = d->electrons.pt; P.eeta = d->electrons.eta; P.ephi = d->electrons.phi;
    P.jet_pt_min = d->jet_pt_min; P.jet_abs_eta_max = d->jet_abs_eta_max; P.lep_pt_min = d->lep_pt_min;
    P.dr2_max = d->dr_max * d->dr_max;      // float32 product (exact class)
    const bool calib = d->calib_table != nullptr;
    P.cal_pt_edges = d->calib_pt_edges; P.cal_eta_edges = d->calib_eta_edges; P.cal_table = d->calib_table;
    P.cal_npt = d->calib_npt; P.cal_neta = d->calib_neta;
    for (int v = 0; v < HEPK_MAX_VARIANTS; ++v) P.scales[v] = calib ? d->calib_scales[v] : 1.0f;
    P.V = d->n_variants; P.W = d->n_wvar;
    P.weights = d->weights;
    int sp = 0, ep = 0;
    for (int o = 0; o < HEPK_N_OBS; ++o) {
        P.axis_edges[o] = d->axis_edges[o];
        P.axis_nbins[o] = d->axis_nbins[o];
        P.obs_prefix[o] = sp; P.edge_prefix[o] = ep;
        if (d->axis_edges[o]) { sp += d->axis_nbins[o] + 2; ep += d->axis_nbins[o] + 1; }
    }
    P.obs_prefix[HEPK_N_OBS] = sp; P.edge_prefix[HEPK_N_OBS] = ep;
    P.out_njet = d->out_njet; P.out_argmax = d->out_argmax; P.out_ht = d->out_ht; P.out_maxpt = d->out_maxpt;
    P.out_minpt = d->out_minpt; P.out_mjj = d->out_mjj; P.out_subpt = d->out_subpt; P.out_jet_mask = d->out_jet_mask;
    const long long n_sumw = (long long)sp * P.V * P.W;
    const bool want_sumw = d->hist_sumw && sp > 0, want_cnt = d->hist_counts && sp > 0;
    P.hist_acc = want_sumw ? (double*)workspace : nullptr;
    P.hist_counts = want_cnt ? (unsigned long long*)d->hist_counts : nullptr;
    P.n_tiles = (d->n_events + TILE - 1) / TILE;
    P.flush_tiles = 4096 / TILE > 0 ? 4096 / TILE : 1;

    // staging capacities from the mean multiplicities (a tile that overflows is processed in pieces)
    const double nev = (double)(d->n_events > 0 ? d->n_events : 1);
    auto cap_for = [&](double mean, int floor_) {
        const double t = TILE * mean;
        long long c = (long long)(t * 1.12 + 6.0 * sqrt(2.0 * t + 1.0)) + 24;
        return c < floor_ ? floor_ : (int)c;
    };
    double mean_l = (double)d->muons.n_objects / nev;
    if (d->electrons.offsets && (double)d->electrons.n_objects / nev > mean_l) mean_l = (double)d->electrons.n_objects / nev;
    P.cap_j = round_up4(d->tune_cap_jets > 0 ? d->tune_cap_jets : cap_for((double)d->jets.n_objects / nev, 256));
    P.cap_l = round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons : cap_for(mean_l, 128));
    if (P.cap_j > 65536 - 8) P.cap_j = 65536 - 8;        // event ids are 16-bit, jet indices must stay small
    if (P.cap_j < 16) P.cap_j = 16;
    if (P.cap_l < 16) P.cap_l = 16;

    const int smem_max = max_smem_optin();
    size_t smem = dev::chain_smem_layout<TILE>(P, calib, nullptr, nullptr);
    while (smem > (size_t)smem_max && P.cap_j > 64) {   // shrink the jet buffers before giving up
        P.cap_j = round_up4(P.cap_j / 2);
        smem = dev::chain_smem_layout<TILE>(P, calib, nullptr, nullptr);
    }
    if (smem > (size_t)smem_max) {
        set_error("hepk_analysis_chain: histograms need %zu bytes of shared memory (max %d)", smem, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    auto kern = calib ? dev::chain_kernel<TILE, true> : dev::chain_kernel<TILE, false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    HEPK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, TILE, smem));
    if (occ < 1) occ = 1;
    if (d->tune_ctas_per_sm > 0 && d->tune_ctas_per_sm < occ) occ = d->tune_ctas_per_sm;
    long long grid = (long long)sm_count() * occ;
    if (grid > P.n_tiles) grid = P.n_tiles;
    if (grid < 1) grid = 1;

    if (want_sumw) HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, (size_t)n_sumw * sizeof(double), st));
    profile_mark(st, 0);
    kern<<<(unsigned)grid, TILE, smem, st>>>(P);
    profile_mark(st, 1);
    HEPK_CUDA_TRY(cudaGetLastError());
    if (want_sumw) {
        dev::chain_finalize_hist<<<(unsigned)((n_sumw + 255) / 256), 256, 0, st>>>(d->hist_sumw, (const double*)workspace, (int)n_sumw);
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    return HEPK_OK;
}

}  // namespace hepk

extern "C" size_t hepk_chain_workspace_bytes(const hepk_chain_desc* d)
{
    if (!d || d->n_variants < 1 || d->n_wvar < 1) return 0;
    const long long n = hepk::hist_slots_per_variant(d) * d->n_variants * d->n_wvar;
    return (size_t)(n > 0 ? n : 1) * sizeof(double);
}

extern "C" int32_t hepk_analysis_chain(const hepk_chain_desc* d, void* workspace, size_t workspace_bytes, void* stream)
{
    using namespace hepk;
    const int32_t rc = chain_validate(d);
    if (rc != HEPK_OK) return rc;
    if (d->n_events == 0) return HEPK_OK;
    if (d->hist_sumw && hist_slots_per_variant(d) > 0) {
        HEPK_REQUIRE(workspace != nullptr, "workspace is NULL");
        HEPK_REQUIRE(workspace_bytes >= hepk_chain_workspace_bytes(d), "workspace too small");
    }
    return chain_launch<128>(d, workspace, (cudaStream_t)stream);
}
