// hepk_chain.cu — the fused analysis chain (include/hepk.h, hepk_analysis_chain).
//
// The path is bound by instruction issue before it is bound by HBM, so the layout is
// chosen to execute few instructions per event, keep lanes busy and never stall a whole CTA:
//
//   * WARP-AUTONOMOUS tiles.  A tile is 32 consecutive events and belongs to ONE warp, which owns a private
//     staging region of shared memory and a private mbarrier.  There is no CTA-wide barrier in the steady state;
//     warps drift apart and hide each other's latencies.
//   * TMA staging of everything.  For a tile the warp's lanes 0..12 each issue one 1-D bulk copy
//     (cp.async.bulk + mbarrier complete_tx): the four jet columns, three muon and three electron columns, and
//     the three offsets slices.  No thread instruction is spent per byte and every byte is read from HBM once.
//     The bounds (offsets[e0], offsets[e1]) a copy needs are loaded one tile ahead.
//   * phase 0, one lane per EVENT: offsets from shared memory, selected leptons compacted into one combined
//     (eta, phi) list, a 16-bit (list start, length) word written for each of the event's jets;
//   * phase 1, one lane per JET (flat, all lanes busy): dR against the event's lepton list, eta cut,
//     (calibration lookup), verdict folded into the staged pt;
//   * phase 2, one lane per EVENT: count / float64 sum / min / top-2 over the event's jets, the leading pair's
//     (eta, phi, mass) into registers — after which the staging region is released and the next tile's copies are
//     issued — then the pair mass, coalesced per-event outputs and the CTA's shared-memory histograms.
// Privatised histograms are merged into float64 global accumulators every few thousand events.
// A tile that does not fit its staging region (giant events, misaligned or out-of-range slices) takes the
// paper's own loop shape (Listing 1): one lane per event, straight from global memory.
#include <string.h>

#include "hepk_common.cuh"

namespace hepk {

constexpr int TILE_EVENTS = 32;     // events per warp tile
constexpr int NCOL = 13;            // staged columns: 0-3 jets pt,eta,phi,mass; 4-6 muons; 7-9 electrons; 10-12 offsets j,m,e
constexpr int MAX_LIST = 2047;      // combined lepton list start fits 11 bits
constexpr int MAX_LEP_EVENT = 31;   // selected leptons of one event fit 5 bits

struct ChainParams {
    long long n_events;
    long long n_tiles;
    // staged columns (see NCOL)
    const char* col_ptr[NCOL];      // element 0 of the column
    long long col_base[NCOL];       // content_base of the collection (0 for offsets)
    long long col_n[NCOL];          // valid elements
    int col_mis[NCOL];              // (address / element size) mod (16 / element size)
    int col_dst[NCOL];              // byte offset of the staging buffer inside a warp's region
    int col_cap[NCOL];              // slice capacity in elements (the buffer has 8 more)
    int col_coll[NCOL];             // collection 0 jets, 1 muons, 2 electrons
    int n_col;                      // 13, or 0 when the staged path is disabled
    int sh_add[10];                 // (col_mis - content_base) mod 4 per float column: shift = (lo32(offsets[e0]) + sh_add) & 3
    const long long* off[3];        // offsets arrays: jets, muons, electrons (electrons nullptr if absent)
    long long jn;
    const float *jpt, *jeta, *jphi, *jmass; long long jbase;
    const float *mpt, *meta, *mphi; long long mbase;
    const float *ept, *eeta, *ephi; long long ebase;
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
    int info_off, lep_off, corr_off;     // byte offsets inside a warp's region
    int region_bytes, shared_bytes;      // per-warp region; CTA-shared part in front of the regions
    int flush_tiles;                     // warp 0 of a CTA flushes the histograms every this many of its tiles
};

namespace dev {

// CTA-shared part of shared memory (in front of the warps' staging regions).
struct ChainShared {
    float *edges, *axis_lo, *axis_inv;
    float *cal_pt_edges, *cal_eta_edges, *cal_table;
    float* h_sumw;
    unsigned int* h_cnt;
};

__host__ __device__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// One layout function used by the host (size) and the device (pointers).
__host__ __device__ inline size_t chain_shared_layout(const ChainParams& P, bool calib, unsigned char* base, ChainShared* s)
{
    size_t o = 0;
    auto take = [&](size_t bytes, size_t al) { o = align_up(o, al); size_t r = o; o += bytes; return r; };
    size_t r;
    r = take((size_t)P.edge_prefix[HEPK_N_OBS] * 4, 4); if (s) s->edges = (float*)(base + r);
    r = take(HEPK_N_OBS * 4, 4); if (s) s->axis_lo = (float*)(base + r);
    r = take(HEPK_N_OBS * 4, 4); if (s) s->axis_inv = (float*)(base + r);
    r = take(calib ? (size_t)(P.cal_npt + 1) * 4 : 0, 4); if (s) s->cal_pt_edges = (float*)(base + r);
    r = take(calib ? (size_t)(P.cal_neta + 1) * 4 : 0, 4); if (s) s->cal_eta_edges = (float*)(base + r);
    r = take(calib ? (size_t)P.cal_npt * P.cal_neta * 4 : 0, 4); if (s) s->cal_table = (float*)(base + r);
    const size_t spv = (size_t)P.obs_prefix[HEPK_N_OBS];
    r = take(P.hist_acc ? spv * P.V * P.W * 4 : 0, 4); if (s) s->h_sumw = (float*)(base + r);
    r = take(P.hist_counts ? spv * P.V * 4 : 0, 4); if (s) s->h_cnt = (unsigned int*)(base + r);
    return align_up(o, 128);
}

// Histogram slot of one observable (uniform branch on whether the observable is histogrammed).
template <int OB>
__device__ __forceinline__ int obs_slot(const ChainParams& P, const ChainShared& S, float x)
{
    if (!P.axis_edges[OB]) return -1;
    return P.obs_prefix[OB] + hist_slot(x, S.edges + P.edge_prefix[OB], P.axis_nbins[OB], S.axis_lo[OB], S.axis_inv[OB]);
}

// dR^2 < thr, exact class.  Same value as dr2_exact: with a = |dphi| and t = a - 2PI_F, the wrapped magnitude
// is min(a, |t|): a > PI_F  =>  |t| <= PI_F < a (rn is monotone), a < PI_F  =>  |t| >= PI_F > a, and at
// a == PI_F both are PI_F.  Three instructions for the wrap instead of four (|.| is a free operand modifier).
__device__ __forceinline__ float dr2_min(float eta_a, float phi_a, float eta_b, float phi_b)
{
    const float deta = __fsub_rn(eta_a, eta_b);
    const float d = __fsub_rn(phi_a, phi_b);
    const float t = __fsub_rn(fabsf(d), HEPK_TWO_PI_F);
    const float w = fminf(fabsf(d), fabsf(t));
    return __fadd_rn(__fmul_rn(deta, deta), __fmul_rn(w, w));
}

// Per event and variant: leading-pair mass, outputs, histograms.  Shared by the staged path and the per-event
// path.  The leading jets' (eta, phi, mass) are passed in by value; i2 < 0 means fewer than two clean jets.
__device__ __forceinline__ void finish_event(const ChainParams& P, const ChainShared& S, long long ev, int v,
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
    int slot[HEPK_N_OBS];
    slot[HEPK_OBS_NJET] = obs_slot<HEPK_OBS_NJET>(P, S, (float)cnt);
    slot[HEPK_OBS_HT] = obs_slot<HEPK_OBS_HT>(P, S, sum);
    slot[HEPK_OBS_MAXPT] = obs_slot<HEPK_OBS_MAXPT>(P, S, b1);
    slot[HEPK_OBS_MINPT] = obs_slot<HEPK_OBS_MINPT>(P, S, mn);
    slot[HEPK_OBS_MJJ] = obs_slot<HEPK_OBS_MJJ>(P, S, mjj);
    slot[HEPK_OBS_SUBPT] = obs_slot<HEPK_OBS_SUBPT>(P, S, subpt);
    const int spv = P.obs_prefix[HEPK_N_OBS];
    if (P.hist_counts) {
        unsigned int* hc = S.h_cnt + v * spv;
#pragma unroll
        for (int ob = 0; ob < HEPK_N_OBS; ++ob)
            if (slot[ob] >= 0) atomicAdd(hc + slot[ob], 1u);
    }
    if (P.hist_acc) {
        // sumw layout [v][o][w][nbins_o + 2]: slot index inside observable o's block moves with w
        for (int w = 0; w < P.W; ++w) {
            const float wt = P.weights ? __ldg(P.weights + (long long)w * P.n_events + ev) : 1.0f;
            float* h = S.h_sumw + (size_t)v * spv * P.W;
#pragma unroll
            for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
                if (slot[ob] < 0) continue;
                const int pre = P.obs_prefix[ob];
                atomicAdd(h + (size_t)pre * P.W + (size_t)w * (P.axis_nbins[ob] + 2) + (slot[ob] - pre), wt);
            }
        }
    }
}

// Running per-event state of phase 2.
struct EventAcc {
    int cnt, i1, i2;
    double sum;      // float64: exact for float32 terms of like magnitude, so HT and its bin do not depend on the order (R15)
    float mn, b1, b2;
    __device__ __forceinline__ void init() { cnt = 0; i1 = i2 = -1; sum = 0.0; mn = CUDART_INF_F; b1 = b2 = -CUDART_INF_F; }
    // `p` must be -inf when !ok
    __device__ __forceinline__ void push(float p, bool ok, int k)
    {
        cnt += ok ? 1 : 0;
        if (ok) sum += (double)p;
        mn = fminf(mn, ok ? p : CUDART_INF_F);
        // top-2 with the first-index tie rule: strict > keeps the smallest index among equal values, for both places
        const bool gt1 = p > b1, gt2 = p > b2;
        i2 = gt1 ? i1 : (gt2 ? k : i2);
        i1 = gt1 ? k : i1;
        b2 = gt1 ? b1 : (gt2 ? p : b2);
        b1 = gt1 ? p : b1;
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

// Path for the events of a tile that does not fit the staging region: the paper's own loop shape
// (Listing 1), one lane per event, everything from global memory.  Slow; only unusual tiles get here.
template <bool CALIB>
__device__ __noinline__ void chain_event_global(const ChainParams& P, const ChainShared& S, long long ev)
{
    const long long g0 = P.off[0][ev], g1 = P.off[0][ev + 1];
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
                bool matched = match_global(P, eta, phi, P.off[1], P.mbase, P.mpt, P.meta, P.mphi, ev);
                if (!matched && P.off[2]) matched = match_global(P, eta, phi, P.off[2], P.ebase, P.ept, P.eeta, P.ephi, ev);
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

// Move the privatised histograms of the CTA into the global accumulators.  Safe against concurrent fills by
// other warps: every bin is taken with an atomic exchange.
__device__ __forceinline__ void flush_hist(const ChainParams& P, const ChainShared& S, int t, int nt)
{
    const int spv = P.obs_prefix[HEPK_N_OBS];
    if (P.hist_acc) {
        const int n = spv * P.V * P.W;
        for (int i = t; i < n; i += nt) {
            if (S.h_sumw[i] == 0.0f) continue;
            const float x = atomicExch(S.h_sumw + i, 0.0f);
            if (x != 0.0f) atomicAdd(P.hist_acc + i, (double)x);
        }
    }
    if (P.hist_counts) {
        const int n = spv * P.V;
        for (int i = t; i < n; i += nt) {
            if (S.h_cnt[i] == 0u) continue;
            const unsigned int c = atomicExch(S.h_cnt + i, 0u);
            if (c) atomicAdd(P.hist_counts + i, (unsigned long long)c);
        }
    }
}

// What a lane needs to stage "its" column (lanes 0..NCOL-1), loaded once into registers.
struct LaneCol {
    const char* ptr;            // nullptr: nothing to stage (other lanes, absent electrons)
    const long long* off;       // the collection's offsets array
    long long base, n;
    int mis, cap;
    uint32_t dst;               // shared-memory address of the staging buffer
};

// offsets[e0] and offsets[e1] of the lane's collection for tile `tile` (loaded one tile ahead of their use)
__device__ __forceinline__ void load_bounds(const ChainParams& P, const LaneCol& c, long long tile, long long& lo, long long& hi)
{
    lo = hi = 0;
    if (c.ptr) {
        const long long e0 = tile * TILE_EVENTS;
        const long long e1 = e0 + TILE_EVENTS < P.n_events ? e0 + TILE_EVENTS : P.n_events;
        lo = __ldg(c.off + e0);
        hi = __ldg(c.off + e1);
    }
}

// Start the bulk copies of tile `tile` into the warp's staging region; all 32 lanes call it, converged.
// Returns false (nothing issued) when some slice does not fit: capacity, 16-byte alignment at the array ends.
// Element l of a column lands at buffer index l - a0, a0 = l0 - ((l0 + mis) mod A), so the copy is 16-byte
// aligned on both sides; the consumer recomputes the same shift.
__device__ __forceinline__ bool issue_tile(const ChainParams& P, const LaneCol& c, long long tile, int lane,
                                           long long lo, long long hi, uint64_t* bar)
{
    const long long e0 = tile * TILE_EVENTS;
    const long long rest = P.n_events - e0;
    const int ne = rest < TILE_EVENTS ? (int)rest : TILE_EVENTS;
    const bool is_off = lane >= 10;
    const int A = is_off ? 2 : 4, esh = is_off ? 3 : 2;
    const long long l0 = is_off ? e0 : lo - c.base;
    const long long l1 = is_off ? e0 + ne + 1 : hi - c.base;
    const long long n = l1 - l0;
    const int sh = ((int)l0 + c.mis) & (A - 1);
    const long long a0 = l0 - sh;
    const long long len = (n + sh + A - 1) & ~(long long)(A - 1);
    const bool active = c.ptr != nullptr && n != 0;
    const bool ok = !active || (n > 0 && n <= c.cap && a0 >= 0 && a0 + len <= c.n);
    if (!__all_sync(0xffffffffu, ok)) return false;
    const uint32_t bytes = active ? ((uint32_t)len << esh) : 0u;
    const uint32_t total = __reduce_add_sync(0xffffffffu, bytes);
    if (lane == 0) mbar_arrive_expect_tx(bar, total);
    __syncwarp();
    if (active) bulk_g2s_addr(c.dst, c.ptr + (a0 << esh), bytes, bar);
    return true;
}

template <bool CALIB, bool HAS_EL>
__global__ void __launch_bounds__(512, 1) chain_kernel(const __grid_constant__ ChainParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ChainShared S;
    chain_shared_layout(P, CALIB, smem_raw, &S);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = tid >> 5, lane = tid & 31, nwarp = nthr >> 5;
    unsigned char* R = smem_raw + P.shared_bytes + (size_t)warp * P.region_bytes;   // this warp's staging region
    uint64_t* bar = (uint64_t*)R;

    // ---- one-time setup: barrier, axis edges, calibration tables, zeroed histograms
    if (lane == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        for (int i = tid; i <= nb; i += nthr) S.edges[P.edge_prefix[ob] + i] = P.axis_edges[ob][i];
        if (tid == 0) {
            const float lo = P.axis_edges[ob][0], hi = P.axis_edges[ob][nb];
            S.axis_lo[ob] = lo;
            S.axis_inv[ob] = (float)nb / (hi - lo);
        }
    }
    if (CALIB) {
        for (int i = tid; i <= P.cal_npt; i += nthr) S.cal_pt_edges[i] = P.cal_pt_edges[i];
        for (int i = tid; i <= P.cal_neta; i += nthr) S.cal_eta_edges[i] = P.cal_eta_edges[i];
        for (int i = tid; i < P.cal_npt * P.cal_neta; i += nthr) S.cal_table[i] = P.cal_table[i];
    }
    {
        const int spv = P.obs_prefix[HEPK_N_OBS];
        if (P.hist_acc) for (int i = tid; i < spv * P.V * P.W; i += nthr) S.h_sumw[i] = 0.0f;
        if (P.hist_counts) for (int i = tid; i < spv * P.V; i += nthr) S.h_cnt[i] = 0u;
    }
    LaneCol col;
    col.ptr = nullptr; col.off = nullptr; col.base = 0; col.n = 0; col.mis = 0; col.cap = 0; col.dst = 0;
    if (lane < P.n_col) {
        const int k = P.col_coll[lane];
        col.off = P.off[k];
        col.ptr = col.off ? P.col_ptr[lane] : nullptr;
        col.base = P.col_base[lane]; col.n = P.col_n[lane];
        col.mis = P.col_mis[lane]; col.cap = P.col_cap[lane];
        col.dst = smem_u32(R + P.col_dst[lane]);
    }
    __syncthreads();

    // staging buffers of this warp
    const int* const so_j = (const int*)(R + P.col_dst[10]) + 2 * P.col_mis[10];   // low words of the offsets slices
    const int* const so_m = (const int*)(R + P.col_dst[11]) + 2 * P.col_mis[11];
    const int* const so_e = (const int*)(R + P.col_dst[12]) + 2 * P.col_mis[12];
    unsigned short* const sinfo = (unsigned short*)(R + P.info_off);
    float2* const slep = (float2*)(R + P.lep_off);
    float* const scorr = (float*)(R + P.corr_off);
    const int V = CALIB ? P.V : 1;

    const long long GW = (long long)gridDim.x * nwarp;
    long long tile = (long long)warp * gridDim.x + blockIdx.x;
    uint32_t parity = 0;
    int since_flush = 0;
    bool fit = false;
    if (tile < P.n_tiles) {
        long long lo, hi;
        load_bounds(P, col, tile, lo, hi);
        fit = issue_tile(P, col, tile, lane, lo, hi, bar);
    }

    for (; tile < P.n_tiles; tile += GW) {
        const long long e0 = tile * TILE_EVENTS;
        const long long rest = P.n_events - e0;
        const int ne = rest < TILE_EVENTS ? (int)rest : TILE_EVENTS;
        const long long tile_next = tile + GW;
        const bool has_next = tile_next < P.n_tiles;
        long long nlo = 0, nhi = 0;
        if (has_next) load_bounds(P, col, tile_next, nlo, nhi);
        bool staged = fit;
        bool released = false;
        fit = false;

        if (staged) {
            mbar_wait(bar, parity);
            parity ^= 1u;
            // ---- phase 0: one lane per event
            const int jb = so_j[0], mb = so_m[0], qb = HAS_EL ? so_e[0] : 0;
            const int njt = so_j[2 * ne] - jb;
            const float* spt = (const float*)(R + P.col_dst[0]) + ((jb + P.sh_add[0]) & 3);
            const float* seta = (const float*)(R + P.col_dst[1]) + ((jb + P.sh_add[1]) & 3);
            const float* sphi = (const float*)(R + P.col_dst[2]) + ((jb + P.sh_add[2]) & 3);
            const float* smass = (const float*)(R + P.col_dst[3]) + ((jb + P.sh_add[3]) & 3);
            int kj0 = 0, nj = 0, c = 0;
            if (lane < ne) {
                kj0 = so_j[2 * lane] - jb;
                nj = so_j[2 * lane + 2] - so_j[2 * lane];
                const int m0 = so_m[2 * lane] - mb, nm = so_m[2 * lane + 2] - so_m[2 * lane];
                int q0 = 0, nq = 0;
                if (HAS_EL) { q0 = so_e[2 * lane] - qb; nq = so_e[2 * lane + 2] - so_e[2 * lane]; }
                const int l0 = m0 + q0;
                {
                    const float* lp = (const float*)(R + P.col_dst[4]) + ((mb + P.sh_add[4]) & 3) + m0;
                    const float* le = (const float*)(R + P.col_dst[5]) + ((mb + P.sh_add[5]) & 3) + m0;
                    const float* lf = (const float*)(R + P.col_dst[6]) + ((mb + P.sh_add[6]) & 3) + m0;
                    for (int i = 0; i < nm; ++i)
                        if (lp[i] > P.lep_pt_min) {
                            if (c < MAX_LEP_EVENT) slep[l0 + c] = make_float2(le[i], lf[i]);
                            ++c;
                        }
                }
                if (HAS_EL) {
                    const float* lp = (const float*)(R + P.col_dst[7]) + ((qb + P.sh_add[7]) & 3) + q0;
                    const float* le = (const float*)(R + P.col_dst[8]) + ((qb + P.sh_add[8]) & 3) + q0;
                    const float* lf = (const float*)(R + P.col_dst[9]) + ((qb + P.sh_add[9]) & 3) + q0;
                    for (int i = 0; i < nq; ++i)
                        if (lp[i] > P.lep_pt_min) {
                            if (c < MAX_LEP_EVENT) slep[l0 + c] = make_float2(le[i], lf[i]);
                            ++c;
                        }
                }
                const unsigned short info = (unsigned short)(l0 | (c << 11));
                unsigned short* ip = sinfo + kj0;
                for (int k = 0; k < nj; ++k) ip[k] = info;
            }
            // an event with more selected leptons than the packed word can count: the whole tile goes the slow way
            staged = !__any_sync(0xffffffffu, c > MAX_LEP_EVENT);
            __syncwarp();

            if (staged) {
                // ---- phase 1: one lane per jet
                const long long lj0 = ((const long long*)(R + P.col_dst[10]) + P.col_mis[10])[0] - P.jbase;
                float* wpt = const_cast<float*>(spt);
                for (int j = lane; j < njt; j += 32) {
                    const unsigned int info = sinfo[j];
                    const float eta = seta[j], phi = sphi[j];
                    const float2* L = slep + (info & 2047u);
                    const int n = (int)(info >> 11);
                    bool matched = false;
                    for (int t = 0; t < n; ++t) {
                        const float2 l = L[t];
                        matched |= dr2_min(eta, phi, l.x, l.y) < P.dr2_max;
                    }
                    const float pt = spt[j];
                    const bool base = (fabsf(eta) < P.jet_abs_eta_max) && !matched;
                    if (!CALIB) {
                        const bool clean = base && (pt > P.jet_pt_min);
                        if (P.out_jet_mask) P.out_jet_mask[lj0 + j] = clean ? 1 : 0;
                        wpt[j] = clean ? pt : -CUDART_INF_F;
                    } else {
                        const int bx = find_bin_clamped(pt, S.cal_pt_edges, P.cal_npt);
                        const int by = find_bin_clamped(eta, S.cal_eta_edges, P.cal_neta);
                        const float cf = S.cal_table[bx * P.cal_neta + by];
                        scorr[j] = cf;
                        if (!base) wpt[j] = CUDART_NAN_F;
                        if (P.out_jet_mask)
                            for (int v = 0; v < V; ++v)
                                P.out_jet_mask[(long long)v * P.jn + lj0 + j] =
                                    (base && (__fmul_rn(pt, __fmul_rn(cf, P.scales[v])) > P.jet_pt_min)) ? 1 : 0;
                    }
                }
                __syncwarp();

                // ---- phase 2: one lane per event (lanes past the last event run with nj = 0)
                const float* pp = spt + kj0;
                const float* cc = scorr + kj0;
                for (int v = 0; v < V; ++v) {
                    const float sv = P.scales[v];
                    EventAcc a;
                    a.init();
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
                        e1 = seta[x]; p1 = sphi[x]; m1 = smass[x];
                        e2 = seta[y]; p2 = sphi[y]; m2 = smass[y];
                    }
                    if (v == V - 1) {
                        // the staging region is dead from here: start the next tile's copies under the finishing math
                        fence_proxy_async_smem();
                        __syncwarp();
                        if (has_next) fit = issue_tile(P, col, tile_next, lane, nlo, nhi, bar);
                        released = true;
                    }
                    if (lane < ne)
                        finish_event(P, S, e0 + lane, v, a.cnt, (float)a.sum, a.mn, a.b1, a.b2, a.i1, a.i2, e1, p1, m1, e2, p2, m2);
                }
            }
        }
        if (!released) {
            fence_proxy_async_smem();
            __syncwarp();
            if (has_next) fit = issue_tile(P, col, tile_next, lane, nlo, nhi, bar);
        }
        if (!staged && lane < ne) chain_event_global<CALIB>(P, S, e0 + lane);
        __syncwarp();

        if (warp == 0 && ++since_flush >= P.flush_tiles) {
            flush_hist(P, S, lane, 32);
            since_flush = 0;
        }
    }
    __syncthreads();
    flush_hist(P, S, tid, nthr);
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

// Fill the staged-column table and the per-warp region layout for the given capacities; returns the region size.
static int chain_region_layout(ChainParams& P, const hepk_chain_desc* d, bool calib, int cap_j, int cap_m, int cap_e)
{
    const hepk_collection* coll[3] = {&d->jets, &d->muons, &d->electrons};
    const float* fcol[10] = {d->jets.pt, d->jets.eta, d->jets.phi, d->jets.mass, d->muons.pt, d->muons.eta, d->muons.phi,
                             d->electrons.pt, d->electrons.eta, d->electrons.phi};
    const int fcoll[10] = {0, 0, 0, 0, 1, 1, 1, 2, 2, 2};
    const int caps[3] = {cap_j, cap_m, cap_e};
    size_t o = 16;      // the mbarrier sits at the start of the region
    auto take = [&](size_t bytes) { o = dev::align_up(o, 16); size_t r = o; o += bytes; return (int)r; };
    for (int c = 0; c < 10; ++c) {
        const int k = fcoll[c];
        P.col_ptr[c] = (const char*)fcol[c];
        P.col_base[c] = coll[k]->content_base;
        P.col_n[c] = coll[k]->n_objects;
        P.col_mis[c] = (int)((reinterpret_cast<uintptr_t>(fcol[c]) / 4) % 4);
        P.col_cap[c] = caps[k];
        P.col_coll[c] = k;
        P.col_dst[c] = take((size_t)(caps[k] + 8) * 4);
        const long long b = coll[k]->content_base % 4;
        P.sh_add[c] = (int)(((P.col_mis[c] - b) % 4 + 4) % 4);
    }
    for (int k = 0; k < 3; ++k) {
        const int c = 10 + k;
        P.col_ptr[c] = (const char*)coll[k]->offsets;
        P.col_base[c] = 0;
        P.col_n[c] = d->n_events + 1;
        P.col_mis[c] = (int)((reinterpret_cast<uintptr_t>(coll[k]->offsets) / 8) % 2);
        P.col_cap[c] = TILE_EVENTS + 1;
        P.col_coll[c] = k;
        P.col_dst[c] = take((size_t)(TILE_EVENTS + 1 + 3) * 8);
    }
    P.info_off = take((size_t)cap_j * 2);
    P.lep_off = take((size_t)(cap_m + cap_e) * 8);
    P.corr_off = take(calib ? (size_t)cap_j * 4 : 0);
    return (int)dev::align_up(o, 128);
}

static int32_t chain_launch(const hepk_chain_desc* d, void* workspace, cudaStream_t st)
{
    ChainParams P;
    memset(&P, 0, sizeof(P));
    P.n_events = d->n_events;
    P.n_tiles = (d->n_events + TILE_EVENTS - 1) / TILE_EVENTS;
    P.off[0] = (const long long*)d->jets.offsets;
    P.off[1] = (const long long*)d->muons.offsets;
    P.off[2] = (const long long*)d->electrons.offsets;
    P.jn = d->jets.n_objects;
    P.jpt = d->jets.pt; P.jeta = d->jets.eta; P.jphi = d->jets.phi; P.jmass = d->jets.mass; P.jbase = d->jets.content_base;
    P.mpt = d->muons.pt; P.meta = d->muons.eta; P.mphi = d->muons.phi; P.mbase = d->muons.content_base;
    P.ept = d->electrons.pt; P.eeta = d->electrons.eta; P.ephi = d->electrons.phi; P.ebase = d->electrons.content_base;
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

    // staging capacities per 32-event tile from the mean multiplicities: mean + ~5 sigma of a Poisson-like
    // tile total (a tile that does not fit takes the per-event path)
    const double nev = (double)(d->n_events > 0 ? d->n_events : 1);
    auto cap_for = [&](double mean, int floor_) {
        const double t = TILE_EVENTS * mean;
        long long c = (long long)(t + 5.0 * sqrt(2.0 * t + 1.0)) + 16;
        return c < floor_ ? floor_ : (int)c;
    };
    int cap_j = round_up4(d->tune_cap_jets > 0 ? d->tune_cap_jets : cap_for((double)d->jets.n_objects / nev, 64));
    int cap_m = round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons : cap_for((double)d->muons.n_objects / nev, 32));
    int cap_e = has_el ? round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons
                                                              : cap_for((double)d->electrons.n_objects / nev, 32)) : 0;
    if (cap_j < 16) cap_j = 16;
    if (cap_m < 4) cap_m = 4;
    if (has_el && cap_e < 4) cap_e = 4;
    if (cap_m > MAX_LIST / 2 - 4) cap_m = MAX_LIST / 2 - 4;      // the list start is packed in 11 bits
    if (cap_e > MAX_LIST / 2 - 4) cap_e = MAX_LIST / 2 - 4;

    const int smem_max = max_smem_optin();
    const int shared_bytes = (int)dev::chain_shared_layout(P, calib, nullptr, nullptr);
    if (shared_bytes + 1024 > smem_max) {
        set_error("hepk_analysis_chain: histograms need %d bytes of shared memory (max %d)", shared_bytes, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    int region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
    while (shared_bytes + region > smem_max && cap_j > 64) {      // shrink the jet buffers before giving up
        cap_j = round_up4(cap_j / 2);
        region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
    }
    while (shared_bytes + region > smem_max && (cap_m > 16 || cap_e > 16)) {
        if (cap_m > 16) cap_m = round_up4(cap_m / 2);
        if (cap_e > 16) cap_e = round_up4(cap_e / 2);
        region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
    }
    if (shared_bytes + region > smem_max) {
        set_error("hepk_analysis_chain: %d + %d bytes of shared memory needed (max %d)", shared_bytes, region, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    P.shared_bytes = shared_bytes;
    P.region_bytes = region;
    P.n_col = NCOL;

    // CTA shape: as many warps per SM as shared memory allows (up to 16), in as few CTAs as possible so that
    // the privatised histograms are shared by many warps
    const int sm_total = smem_max + 1024;              // per SM; each CTA also pays 1 KB of system shared memory
    int best_ctas = 1, best_wpc = 1, best_total = 0;
    const int max_warps_sm = 16;
    for (int ctas = 1; ctas <= 4; ++ctas) {
        if (d->tune_ctas_per_sm > 0 && ctas != d->tune_ctas_per_sm && !(ctas == 1 && d->tune_ctas_per_sm > 4)) continue;
        int budget = sm_total / ctas - 1024;
        if (budget > smem_max) budget = smem_max;
        int wpc = (budget - shared_bytes) / region;
        if (wpc > 16) wpc = 16;
        if (wpc * ctas > max_warps_sm) wpc = max_warps_sm / ctas;
        if (d->tune_warps_per_cta > 0 && wpc > d->tune_warps_per_cta) wpc = d->tune_warps_per_cta;
        if (wpc < 1) continue;
        if (wpc * ctas > best_total) { best_total = wpc * ctas; best_ctas = ctas; best_wpc = wpc; }
    }
    const int wpc = best_wpc;
    const size_t smem = (size_t)shared_bytes + (size_t)wpc * region;
    P.flush_tiles = 4096 / (TILE_EVENTS * wpc) > 0 ? 4096 / (TILE_EVENTS * wpc) : 1;

    void (*kern)(ChainParams);
    if (calib) kern = has_el ? dev::chain_kernel<true, true> : dev::chain_kernel<true, false>;
    else kern = has_el ? dev::chain_kernel<false, true> : dev::chain_kernel<false, false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    HEPK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, wpc * 32, smem));
    if (occ < 1) occ = 1;
    if (occ > best_ctas) occ = best_ctas;
    long long grid = (long long)sm_count() * occ;
    const long long need = (P.n_tiles + wpc - 1) / wpc;
    if (grid > need) grid = need;
    if (grid < 1) grid = 1;

    if (want_sumw) HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, (size_t)n_sumw * sizeof(double), st));
    profile_mark(st, 0);
    kern<<<(unsigned)grid, wpc * 32, smem, st>>>(P);
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
    return chain_launch(d, workspace, (cudaStream_t)stream);
}
