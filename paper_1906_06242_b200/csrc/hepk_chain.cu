// hepk_chain.cu — the fused analysis chain (include/hepk.h, hepk_analysis_chain).
//
// One persistent kernel; the path is bound by instruction issue before it is bound by HBM (DESIGN.md
// "chain kernel"), so the layout below is chosen to execute as few instructions per event as possible
// with every lane busy.  Each CTA walks tiles of T events (T threads); per tile
//   0. the tile's jet-column slices (pt, eta, phi, mass: 63 % of the bytes) are moved into shared memory by
//      TMA 1-D bulk copies (cp.async.bulk + mbarrier) issued by warp 0 — no thread instructions per byte;
//   1. prep, one thread per EVENT, while the bulk copies are in flight: the event's six offsets (coalesced
//      LDG), its selected leptons compacted into one combined (eta, phi) list in shared memory, and a packed
//      (list start, list length) word written for each of its jets;
//   2. phase 1, one thread per JET (flat: every lane busy): dR test against the event's combined lepton list,
//      eta cut, (calibration lookup), verdict folded into the staged pt (-inf / NaN = not clean);
//   3. phase 2, one thread per EVENT: count / float64 sum / min / top-2 over the event's jets from shared
//      memory, leading-pair mass, coalesced per-event outputs, shared-memory histograms.
// Privatised histograms are merged into float64 global accumulators every few thousand events.
// A tile whose jets or leptons do not fit the shared-memory buffers (a giant event, a dense run) is processed
// by the paper's own loop shape (Listing 1): one thread per event, straight from global memory.
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
    int cap_j, cap_l;                    // staged jets per tile / combined selected leptons per tile
    int jk[4];                           // (misalignment of the jet column in floats - jbase) mod 4: pt, eta, phi, mass
    long long n_tiles;
    int flush_tiles;
};

namespace dev {

struct ChainSmem {
    uint64_t* bar;
    long long* bnd;                      // [2][6]: joff[e0], joff[e1], moff[e0], moff[e1], eoff[e0], eoff[e1] of this / the next tile
    float *jpt, *jeta, *jphi, *jmass, *corr;
    unsigned int* info;                  // per staged jet: combined-lepton list start | length << 16
    float2* lep;                         // combined (eta, phi) of the tile's selected leptons, event by event
    float *edges, *axis_lo, *axis_inv;
    float *cal_pt_edges, *cal_eta_edges, *cal_table;
    float* h_sumw;
    unsigned int* h_cnt;
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// One layout function used by the host (size) and the device (pointers).
__host__ __device__ inline size_t chain_smem_layout(const ChainParams& P, bool calib, unsigned char* base, ChainSmem* s)
{
    size_t o = 0;
    auto take = [&](size_t bytes, size_t al) { o = align_up(o, al); size_t r = o; o += bytes; return r; };
    size_t r;
    r = take(8, 8); if (s) s->bar = (uint64_t*)(base + r);
    r = take(12 * 8, 8); if (s) s->bnd = (long long*)(base + r);
    const size_t cj = (size_t)P.cap_j * 4;
    r = take(cj, 16); if (s) s->jpt = (float*)(base + r);
    r = take(cj, 16); if (s) s->jeta = (float*)(base + r);
    r = take(cj, 16); if (s) s->jphi = (float*)(base + r);
    r = take(cj, 16); if (s) s->jmass = (float*)(base + r);
    r = take(calib ? cj : 0, 16); if (s) s->corr = (float*)(base + r);
    r = take(cj, 4); if (s) s->info = (unsigned int*)(base + r);
    r = take((size_t)P.cap_l * 8, 8); if (s) s->lep = (float2*)(base + r);
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

// One observable of one event and variant into the privatised histograms.
template <int OB>
__device__ __forceinline__ void fill_obs(const ChainParams& P, const ChainSmem& S, long long ev, int v, float x)
{
    if (!P.axis_edges[OB]) return;
    const int nb = P.axis_nbins[OB];
    const int slot = hist_slot(x, S.edges + P.edge_prefix[OB], nb, S.axis_lo[OB], S.axis_inv[OB]);
    const int spv = P.obs_prefix[HEPK_N_OBS];
    if (P.hist_counts) atomicAdd(&S.h_cnt[v * spv + P.obs_prefix[OB] + slot], 1u);
    if (P.hist_acc) {
        float* h = S.h_sumw + (size_t)(v * spv + P.obs_prefix[OB]) * P.W + slot;
        for (int w = 0; w < P.W; ++w) {
            const float wt = P.weights ? __ldg(P.weights + (long long)w * P.n_events + ev) : 1.0f;
            atomicAdd(h + w * (nb + 2), wt);
        }
    }
}

// Per event and variant: leading-pair mass, outputs, histograms.  Shared by the tile path and the per-event
// path.  The leading jets' (eta, phi, mass) are passed in by value; i2 < 0 means fewer than two clean jets.
__device__ __forceinline__ void finish_event(const ChainParams& P, const ChainSmem& S, long long ev, int v,
                                             int cnt, float sum, float mn, float b1, float b2, int i1, int i2,
                                             float eta1, float phi1, float m1, float eta2, float phi2, float m2)
{
    float mjj = 0.0f, subpt = 0.0f;
    const bool hists = P.hist_acc || P.hist_counts;
    if (i2 >= 0) {
        subpt = b2;
        mjj = pair_mass_fast(b1, eta1, phi1, m1, b2, eta2, phi2, m2);
        if (hists && P.axis_edges[HEPK_OBS_MJJ]) {
            // the bin of mjj is decided by the float64-defined value: refine when the fast value is near an edge
            const float* ed = S.edges + P.edge_prefix[HEPK_OBS_MJJ];
            const int nb = P.axis_nbins[HEPK_OBS_MJJ];
            const int slot = hist_slot(mjj, ed, nb, S.axis_lo[HEPK_OBS_MJJ], S.axis_inv[HEPK_OBS_MJJ]);
            const float band = fmaf(mjj, HEPK_MASS_GUARD_REL, HEPK_MASS_GUARD_ABS);
            const bool near_lo = slot >= 1 && mjj - ed[slot - 1] <= band;
            const bool near_hi = slot <= nb && ed[slot] - mjj <= band;
            if (near_lo || near_hi) mjj = pair_mass_f64(b1, eta1, phi1, m1, b2, eta2, phi2, m2);
        }
    }
    const long long o = (long long)v * P.n_events + ev;
    if (P.out_njet) P.out_njet[o] = cnt;
    if (P.out_argmax) P.out_argmax[o] = i1;
    if (P.out_ht) P.out_ht[o] = sum;
    if (P.out_maxpt) P.out_maxpt[o] = b1;
    if (P.out_minpt) P.out_minpt[o] = mn;
    if (P.out_mjj) P.out_mjj[o] = mjj;
    if (P.out_subpt) P.out_subpt[o] = subpt;
    if (!hists) return;
    fill_obs<HEPK_OBS_NJET>(P, S, ev, v, (float)cnt);
    fill_obs<HEPK_OBS_HT>(P, S, ev, v, sum);
    fill_obs<HEPK_OBS_MAXPT>(P, S, ev, v, b1);
    fill_obs<HEPK_OBS_MINPT>(P, S, ev, v, mn);
    fill_obs<HEPK_OBS_MJJ>(P, S, ev, v, mjj);
    fill_obs<HEPK_OBS_SUBPT>(P, S, ev, v, subpt);
}

// Running per-event state of phase 2.  `p` is the jet's pt if it is clean in this variant, else -inf.
struct EventAcc {
    int cnt, i1, i2;
    double sum;      // float64: exact for float32 terms of like magnitude, so HT and its bin do not depend on the order (R15)
    float mn, b1, b2;
    __device__ __forceinline__ void init() { cnt = 0; i1 = i2 = -1; sum = 0.0; mn = CUDART_INF_F; b1 = b2 = -CUDART_INF_F; }
    __device__ __forceinline__ void push(float p, bool ok, int k)
    {
        cnt += ok ? 1 : 0;
        if (ok) sum += (double)p;
        mn = fminf(mn, ok ? p : CUDART_INF_F);
        // top-2 with the first-index tie rule: strict > keeps the smallest index among equal values, for both places
        const bool gt1 = p > b1, gt2 = p > b2;
        i2 = gt1 ? i1 : (gt2 ? k : i2);
        i1 = gt1 ? k : i1;
        b2 = fmaxf(b2, fminf(b1, p));
        b1 = fmaxf(b1, p);
    }
};

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

// Path for the events of a tile that does not fit the shared-memory buffers: the paper's own loop shape
// (Listing 1), one thread per event, everything from global memory.  Slow; only unusual tiles get here.
template <bool CALIB>
__device__ __noinline__ void chain_event_global(const ChainParams& P, const ChainSmem& S, long long ev)
{
    const long long g0 = P.joff[ev], g1 = P.joff[ev + 1];
    for (int v = 0; v < P.V; ++v) {
        EventAcc a;
        a.init();
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
            a.push(clean ? p : -CUDART_INF_F, clean, (int)(g - g0));
        }
        float e1 = 0, p1 = 0, m1 = 0, e2 = 0, p2 = 0, m2 = 0;
        if (a.i2 >= 0) {
            const long long x = g0 - P.jbase + a.i1, y = g0 - P.jbase + a.i2;
            e1 = P.jeta[x]; p1 = P.jphi[x]; m1 = P.jmass[x];
            e2 = P.jeta[y]; p2 = P.jphi[y]; m2 = P.jmass[y];
        }
        finish_event(P, S, ev, v, a.cnt, (float)a.sum, a.mn, a.b1, a.b2, a.i1, a.i2, e1, p1, m1, e2, p2, m2);
    }
}

template <int T>
__device__ __forceinline__ void flush_hist(const ChainParams& P, const ChainSmem& S, int tid)
{
    const int spv = P.obs_prefix[HEPK_N_OBS];
    if (P.hist_acc) {
        const int n = spv * P.V * P.W;
        for (int i = tid; i < n; i += T) {
            const float x = S.h_sumw[i];
            if (x != 0.0f) { atomicAdd(P.hist_acc + i, (double)x); S.h_sumw[i] = 0.0f; }
        }
    }
    if (P.hist_counts) {
        const int n = spv * P.V;
        for (int i = tid; i < n; i += T) {
            const unsigned int c = S.h_cnt[i];
            if (c) { atomicAdd(P.hist_counts + i, (unsigned long long)c); S.h_cnt[i] = 0u; }
        }
    }
}

// The six boundary offsets of tile `tile` (first and one-past-last event of each collection).
template <int T, bool HAS_EL>
__device__ __forceinline__ void load_bounds(const ChainParams& P, long long tile, long long* b)
{
    const long long e0 = tile * T;
    const long long e1 = e0 + T < P.n_events ? e0 + T : P.n_events;
    b[0] = __ldg(P.joff + e0); b[1] = __ldg(P.joff + e1);
    b[2] = __ldg(P.moff + e0); b[3] = __ldg(P.moff + e1);
    if (HAS_EL) { b[4] = __ldg(P.eoff + e0); b[5] = __ldg(P.eoff + e1); }
    else { b[4] = 0; b[5] = 0; }
}

template <int T, bool CALIB, bool HAS_EL>
__global__ void __launch_bounds__(T) chain_kernel(const __grid_constant__ ChainParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    ChainSmem S;
    chain_smem_layout(P, CALIB, smem_raw, &S);
    const int tid = threadIdx.x;
    const int warp = tid >> 5, lane = tid & 31;

    // ---- one-time setup: barrier, axis edges, calibration tables, zeroed histograms, first tile's bounds
    if (tid == 0) {
        mbar_init(S.bar, 1);
        fence_mbar_init();
        long long b[6];
        load_bounds<T, HAS_EL>(P, blockIdx.x, b);
#pragma unroll
        for (int i = 0; i < 6; ++i) S.bnd[i] = b[i];
    }
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        for (int i = tid; i <= nb; i += T) S.edges[P.edge_prefix[ob] + i] = P.axis_edges[ob][i];
        if (tid == 0) {
            const float lo = P.axis_edges[ob][0], hi = P.axis_edges[ob][nb];
            S.axis_lo[ob] = lo;
            S.axis_inv[ob] = (float)nb / (hi - lo);
        }
    }
    if (CALIB) {
        for (int i = tid; i <= P.cal_npt; i += T) S.cal_pt_edges[i] = P.cal_pt_edges[i];
        for (int i = tid; i <= P.cal_neta; i += T) S.cal_eta_edges[i] = P.cal_eta_edges[i];
        for (int i = tid; i < P.cal_npt * P.cal_neta; i += T) S.cal_table[i] = P.cal_table[i];
    }
    {
        const int spv = P.obs_prefix[HEPK_N_OBS];
        if (P.hist_acc) for (int i = tid; i < spv * P.V * P.W; i += T) S.h_sumw[i] = 0.0f;
        if (P.hist_counts) for (int i = tid; i < spv * P.V; i += T) S.h_cnt[i] = 0u;
    }
    __syncthreads();

    uint32_t parity = 0;
    int tiles_since_flush = 0, it = 0;
    const int V = CALIB ? P.V : 1;

    for (long long tile = blockIdx.x; tile < P.n_tiles; tile += gridDim.x, ++it) {
        const long long* B = S.bnd + (it & 1) * 6;
        const long long e0 = tile * T;
        const int ne = (int)((P.n_events - e0) < T ? (P.n_events - e0) : T);
        const long long jb = B[0], je = B[1], mb = B[2], me = B[3], qb = B[4], qe = B[5];
        const bool fit = (je - jb) <= (long long)(P.cap_j - 8) && (me - mb) + (qe - qb) <= (long long)P.cap_l;

        // bounds of this CTA's next tile: loaded now, stored at the end of this one (latency hidden)
        const long long tile_next = tile + gridDim.x;
        long long nb[6];
        if (tid == 0 && tile_next < P.n_tiles) load_bounds<T, HAS_EL>(P, tile_next, nb);

        if (fit) {
            const int njt = (int)(je - jb);
            const long long lj0 = jb - P.jbase;
            // ---- 0. warp 0 starts the bulk copies of the four jet columns
            if (warp == 0) {
                long long a0;
                uint32_t bytes = 0;
                bytes += stage_column(S.jpt, P.jpt, lj0, lj0 + njt, P.jn, S.bar, lane, 0, &a0);
                bytes += stage_column(S.jeta, P.jeta, lj0, lj0 + njt, P.jn, S.bar, lane, 0, &a0);
                bytes += stage_column(S.jphi, P.jphi, lj0, lj0 + njt, P.jn, S.bar, lane, 0, &a0);
                bytes += stage_column(S.jmass, P.jmass, lj0, lj0 + njt, P.jn, S.bar, lane, 0, &a0);
                __syncwarp();                       // the lanes' scalar head/tail stores precede lane 0's release
                if (lane == 0) mbar_arrive_expect_tx(S.bar, bytes);
            }
            // ---- 1. prep, one thread per event (overlaps the copies)
            int kj0 = 0, nj = 0;
            if (tid < ne) {
                const long long ev = e0 + tid;
                const long long j0 = __ldg(P.joff + ev), j1 = __ldg(P.joff + ev + 1);
                const long long m0 = __ldg(P.moff + ev), m1 = __ldg(P.moff + ev + 1);
                long long q0 = 0, q1 = 0;
                if (HAS_EL) { q0 = __ldg(P.eoff + ev); q1 = __ldg(P.eoff + ev + 1); }
                kj0 = (int)(j0 - jb);
                nj = (int)(j1 - j0);
                const int l0 = (int)(m0 - mb) + (int)(q0 - qb);
                int c = 0;
                {
                    const int nm = (int)(m1 - m0);
                    const float* lp = P.mpt + (m0 - P.mbase);
                    const float* le = P.meta + (m0 - P.mbase);
                    const float* lf = P.mphi + (m0 - P.mbase);
                    for (int i = 0; i < nm; ++i) {
                        const float pt = lp[i], eta = le[i], phi = lf[i];
                        if (pt > P.lep_pt_min) S.lep[l0 + c++] = make_float2(eta, phi);
                    }
                }
                if (HAS_EL) {
                    const int nq = (int)(q1 - q0);
                    const float* lp = P.ept + (q0 - P.ebase);
                    const float* le = P.eeta + (q0 - P.ebase);
                    const float* lf = P.ephi + (q0 - P.ebase);
                    for (int i = 0; i < nq; ++i) {
                        const float pt = lp[i], eta = le[i], phi = lf[i];
                        if (pt > P.lep_pt_min) S.lep[l0 + c++] = make_float2(eta, phi);
                    }
                }
                const unsigned int info = (unsigned int)l0 | ((unsigned int)c << 16);
                unsigned int* ip = S.info + kj0;
                for (int k = 0; k < nj; ++k) ip[k] = info;
            }
            mbar_wait(S.bar, parity);
            parity ^= 1u;
            __syncthreads();

            // ---- 2. phase 1: one thread per jet
            const int sh_pt = ((int)jb + P.jk[0]) & 3, sh_eta = ((int)jb + P.jk[1]) & 3;
            const int sh_phi = ((int)jb + P.jk[2]) & 3, sh_mass = ((int)jb + P.jk[3]) & 3;
            {
                float* ppt = S.jpt + sh_pt;
                const float* peta = S.jeta + sh_eta;
                const float* pphi = S.jphi + sh_phi;
                for (int j = tid; j < njt; j += T) {
                    const unsigned int info = S.info[j];
                    const float eta = peta[j], phi = pphi[j];
                    const float2* L = S.lep + (info & 0xffffu);
                    const int n = (int)(info >> 16);
                    bool matched = false;
                    for (int t = 0; t < n; ++t) {
                        const float2 l = L[t];
                        matched |= dr2_exact(eta, phi, l.x, l.y) < P.dr2_max;
                    }
                    const float pt = ppt[j];
                    const bool base = (fabsf(eta) < P.jet_abs_eta_max) && !matched;
                    if (!CALIB) {
                        const bool clean = base && (pt > P.jet_pt_min);
                        if (P.out_jet_mask) P.out_jet_mask[lj0 + j] = clean ? 1 : 0;
                        ppt[j] = clean ? pt : -CUDART_INF_F;
                    } else {
                        const int bx = find_bin_clamped(pt, S.cal_pt_edges, P.cal_npt);
                        const int by = find_bin_clamped(eta, S.cal_eta_edges, P.cal_neta);
                        const float c = S.cal_table[bx * P.cal_neta + by];
                        S.corr[j] = c;
                        if (!base) ppt[j] = CUDART_NAN_F;
                        if (P.out_jet_mask)
                            for (int v = 0; v < V; ++v)
                                P.out_jet_mask[(long long)v * P.jn + lj0 + j] =
                                    (base && (__fmul_rn(pt, __fmul_rn(c, P.scales[v])) > P.jet_pt_min)) ? 1 : 0;
                    }
                }
            }
            __syncthreads();

            // ---- 3. phase 2: one thread per event
            if (tid < ne) {
                const float* pp = S.jpt + sh_pt + kj0;
                const float* cc = S.corr + kj0;
                for (int v = 0; v < V; ++v) {
                    const float sv = P.scales[v];
                    EventAcc a;
                    a.init();
#pragma unroll 2
                    for (int k = 0; k < nj; ++k) {
                        float p = pp[k];
                        bool ok;
                        if (CALIB) {
                            p = __fmul_rn(p, __fmul_rn(cc[k], sv));     // NaN when the jet failed eta / dR
                            ok = p > P.jet_pt_min;
                            p = ok ? p : -CUDART_INF_F;
                        } else {
                            ok = p > P.jet_pt_min;                      // -inf when not clean
                        }
                        a.push(p, ok, k);
                    }
                    float e1 = 0, p1 = 0, m1 = 0, e2 = 0, p2 = 0, m2 = 0;
                    if (a.i2 >= 0) {
                        const int x = kj0 + a.i1, y = kj0 + a.i2;
                        e1 = S.jeta[x + sh_eta]; p1 = S.jphi[x + sh_phi]; m1 = S.jmass[x + sh_mass];
                        e2 = S.jeta[y + sh_eta]; p2 = S.jphi[y + sh_phi]; m2 = S.jmass[y + sh_mass];
                    }
                    finish_event(P, S, e0 + tid, v, a.cnt, (float)a.sum, a.mn, a.b1, a.b2, a.i1, a.i2, e1, p1, m1, e2, p2, m2);
                }
            }
        } else {
            if (tid < ne) chain_event_global<CALIB>(P, S, e0 + tid);
        }

        if (tid == 0 && tile_next < P.n_tiles) {
            long long* Bn = S.bnd + ((it + 1) & 1) * 6;
#pragma unroll
            for (int i = 0; i < 6; ++i) Bn[i] = nb[i];
        }
        fence_proxy_async_smem();   // this thread's generic accesses to the staging buffers precede the next bulk copies
        __syncthreads();
        if (++tiles_since_flush >= P.flush_tiles) {
            flush_hist<T>(P, S, tid);
            tiles_since_flush = 0;
            __syncthreads();
        }
    }
    __syncthreads();
    flush_hist<T>(P, S, tid);
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

template <int T>
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
    const bool has_el = d->electrons.offsets != nullptr;
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
    P.n_tiles = (d->n_events + T - 1) / T;
    P.flush_tiles = 4096 / T > 0 ? 4096 / T : 1;
    const float* jc[4] = {d->jets.pt, d->jets.eta, d->jets.phi, d->jets.mass};
    for (int c = 0; c < 4; ++c) {
        const long long mis = (long long)((reinterpret_cast<uintptr_t>(jc[c]) / sizeof(float)) % 4);
        P.jk[c] = (int)((((mis - d->jets.content_base) % 4) + 4) % 4);
    }

    // staging capacities from the mean multiplicities: mean + ~5 sigma of a Poisson-like tile total
    // (a tile that does not fit takes the per-event path)
    const double nev = (double)(d->n_events > 0 ? d->n_events : 1);
    auto cap_for = [&](double mean, int floor_) {
        const double t = T * mean;
        long long c = (long long)(t + 5.0 * sqrt(2.0 * t + 1.0)) + 16;
        return c < floor_ ? floor_ : (int)c;
    };
    double mean_l = (double)d->muons.n_objects / nev;
    if (has_el) mean_l += (double)d->electrons.n_objects / nev;
    P.cap_j = round_up4(d->tune_cap_jets > 0 ? d->tune_cap_jets : cap_for((double)d->jets.n_objects / nev, 256));
    P.cap_l = round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons : cap_for(mean_l, 128));
    if (P.cap_j < 16) P.cap_j = 16;
    if (P.cap_l < 4) P.cap_l = 4;
    if (P.cap_l > 65532) P.cap_l = 65532;      // list start and length are packed in 16 bits each

    const int smem_max = max_smem_optin();
    size_t smem = dev::chain_smem_layout(P, calib, nullptr, nullptr);
    while (smem > (size_t)smem_max && P.cap_j > 64) {   // shrink the jet buffers before giving up
        P.cap_j = round_up4(P.cap_j / 2);
        smem = dev::chain_smem_layout(P, calib, nullptr, nullptr);
    }
    while (smem > (size_t)smem_max && P.cap_l > 64) {
        P.cap_l = round_up4(P.cap_l / 2);
        smem = dev::chain_smem_layout(P, calib, nullptr, nullptr);
    }
    if (smem > (size_t)smem_max) {
        set_error("hepk_analysis_chain: histograms need %zu bytes of shared memory (max %d)", smem, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    void (*kern)(ChainParams);
    if (calib) kern = has_el ? dev::chain_kernel<T, true, true> : dev::chain_kernel<T, true, false>;
    else kern = has_el ? dev::chain_kernel<T, false, true> : dev::chain_kernel<T, false, false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    HEPK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, T, smem));
    if (occ < 1) occ = 1;
    if (d->tune_ctas_per_sm > 0 && d->tune_ctas_per_sm < occ) occ = d->tune_ctas_per_sm;
    long long grid = (long long)sm_count() * occ;
    if (grid > P.n_tiles) grid = P.n_tiles;
    if (grid < 1) grid = 1;

    if (want_sumw) HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, (size_t)n_sumw * sizeof(double), st));
    profile_mark(st, 0);
    kern<<<(unsigned)grid, T, smem, st>>>(P);
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
    switch (d->tune_tile_events) {
        case 32: return chain_launch<32>(d, workspace, (cudaStream_t)stream);
        case 64: return chain_launch<64>(d, workspace, (cudaStream_t)stream);
        case 256: return chain_launch<256>(d, workspace, (cudaStream_t)stream);
        default: return chain_launch<128>(d, workspace, (cudaStream_t)stream);
    }
}
