// hepk_chain.cu — the fused analysis chain (include/hepk.h, hepk_analysis_chain).
//
// The path is bound by instruction issue before it is bound by HBM: at 60 % of the
// HBM peak an SM may spend ~40 warp instructions per event.  The layout is chosen to execute few instructions
// per event, keep lanes busy and never stall a whole CTA:
//
//   * WARP-AUTONOMOUS tiles.  A tile is 32 consecutive events and belongs to ONE warp, which owns a private
//     staging region of shared memory and a private mbarrier.  There is no CTA-wide barrier in the steady state;
//     warps drift apart and hide each other's latencies.
//   * TMA staging of the content columns.  Lanes 0..9 of the warp each issue one 1-D bulk copy
//     (cp.async.bulk + mbarrier complete_tx): four jet columns, three muon and three electron columns.  No thread
//     instruction is spent per byte and every byte is read from HBM once.  The offsets of the tile's events are
//     read one tile ahead with coalesced loads and live in registers (one event per lane).
//   * phase 0, one lane per EVENT: selected leptons compacted into one combined (eta, phi) list; the event's
//     jets are appended to one of eight buckets keyed by the number of selected leptons, which yields a
//     permutation of the tile's jets in which neighbouring jets have the same dR trip count;
//   * phase 1, one lane per JET in that order (flat, all lanes busy, uniform trip counts): dR against the
//     event's lepton list, eta cut, (calibration lookup), verdict folded into the staged pt;
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
constexpr int NCOL = 10;            // staged columns: 0-3 jets pt,eta,phi,mass; 4-6 muons pt,eta,phi; 7-9 electrons
constexpr int MAX_JETS_TILE = 512;  // byte offset of a jet inside a tile column (4 * index) fits 11 bits
constexpr int MAX_LIST = 1023;      // byte offset of an event's lepton list (8 * start) fits 13 bits
constexpr int MAX_LEP_EVENT = 30;   // byte length of an event's lepton list, padded to pairs (16 * pairs), fits 8 bits
constexpr int LIST_PAD = 36;        // list entries beyond the leptons of a tile: every event's list starts at an even entry
constexpr int TAIL_CUT = 16;        // jets of an event beyond this many are handled by the whole warp, not by the event's lane
constexpr int N_BUCKETS = 8;        // jets are ordered by min(selected leptons of their event, 7)

struct ChainParams {
    long long n_events;
    long long n_tiles;
    long long w_stride, out_stride;   // row strides (in events) of the weights and of the per-event outputs
    // staged columns (see NCOL)
    const char* col_ptr[NCOL];      // element 0 of the column
    long long col_base[NCOL];       // content_base of the collection
    long long col_n[NCOL];          // valid elements
    int col_mis[NCOL];              // (address / 4) mod 4
    int col_dst[NCOL];              // byte offset of the staging buffer inside a warp's region
    int col_cap[NCOL];              // slice capacity in elements (the buffer has 8 more)
    int col_coll[NCOL];             // collection 0 jets, 1 muons, 2 electrons
    int n_col;                      // NCOL, or 0 when the staged path is disabled
    int sh_add[NCOL];               // (col_mis - content_base) mod 4: shift = (lo32(offsets[e0]) + sh_add) & 3
    int col_stride[3];              // bytes between the staging buffers of consecutive columns of a collection
    int col_n32[3];                 // valid elements per collection (the staged path requires them to fit an int)
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
    // Histograms.  Privatised bins (shared memory) and their global accumulators (workspace) share one INTERNAL
    // layout: word (v, o, slot, col) at ((v * spv + obs_prefix[o] + slot) * WS + col), columns: W x sumw, then
    // 2W x sumw2 (if asked for), then the event count (if asked for); WS >= the number of columns.  All columns of a
    // slot are neighbours, so one event's updates of a slot are immediate offsets from one address.  sumw2 takes two
    // columns per weight (value and rounding remainder, see add_weights).
    int WS, ncol, col_w2, col_cnt;       // col_w2 / col_cnt: first sumw2 column / count column, -1 = absent
    long long* hist_acc;                 // workspace: n_words accumulators (int64 fixed point, or float64 bits), or nullptr
    unsigned int* hist_hdr;              // workspace header (HDR_* words), or nullptr
    float *hist_sumw, *hist_sumw2;       // the caller's arrays (chain_finalize_hist)
    long long* hist_counts;
    const float *evw_x, *evw_edges, *evw_table;   // per-event weight factor from a lookup (evw_table nullptr: none)
    int evw_nbins;
    int order_off, lep_off, corr_off, bucket_off;   // byte offsets inside a warp's region
    int region_bytes, shared_bytes;      // per-warp region; CTA-shared part in front of the regions
    unsigned int* tile_counter;          // zeroed per launch: the last eighth of the tiles is handed out through it (nullptr: static)
};

// Workspace header words (uint32), written by chain_weight_range_kernel, read by the chain kernel and the finalize step.
enum { HDR_WMAX = 0, HDR_BAD = 1, HDR_TILE = 2, HDR_WMIN = 3, HDR_TMAX = 4, HDR_TMIN = 5, HDR_WORDS = 16 };
constexpr int SCAN_SLICES = 32;          // the bins are checked for overflow in this many slices, one per finished tile
constexpr int FLUSH_AT = 1 << 29;        // a fixed-point bin is moved to its global accumulator when |bin| reaches this

namespace dev {

// CTA-shared part of shared memory (in front of the warps' staging regions).
struct ChainShared {
    float *edges, *axis_lo, *axis_inv;   // axis_inv == 0: the axis is not uniform enough for the arithmetic bin guess
    float *cal_pt_edges, *cal_eta_edges, *cal_table;
    float* cal_axis;                     // per calibration axis (pt, eta): [mode (0 search, 1 linear, 2 log2), lo, inv, unused]
    unsigned int* h_bins;                // internal layout; sumw / sumw2 columns: int32 fixed point when wscale[0] != 0, else float
    float* wscale;                       // [0] 2^k (0: float bins), [1] 2^k2 for squared weights
    float *evw_edges, *evw_table;
    unsigned int* scan;                  // ticket of the overflow scan
    unsigned int* next;                  // tiles of the CTA's own range handed out so far
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
    r = take(calib ? 32 : 0, 16); if (s) s->cal_axis = (float*)(base + r);
    const size_t spv = (size_t)P.obs_prefix[HEPK_N_OBS];
    r = take(P.evw_table ? (size_t)(P.evw_nbins + 1) * 4 : 0, 4); if (s) s->evw_edges = (float*)(base + r);
    r = take(P.evw_table ? (size_t)P.evw_nbins * 4 : 0, 4); if (s) s->evw_table = (float*)(base + r);
    r = take(P.hist_acc ? spv * P.V * P.WS * 4 : 0, 16); if (s) s->h_bins = (unsigned int*)(base + r);
    r = take(8, 4); if (s) s->wscale = (float*)(base + r);
    r = take(4, 4); if (s) s->scan = (unsigned int*)(base + r);
    r = take(4, 4); if (s) s->next = (unsigned int*)(base + r);
    return align_up(o, 128);
}

// [profile phase: shared-memory / atomic helpers]
// ---- shared-memory atomics in the shared state space (no generic-address dispatch) ----------------------
__device__ __forceinline__ unsigned int atom_add_shared_u32(uint32_t addr, unsigned int v)
{
    unsigned int r;
    asm volatile("atom.shared.add.u32 %0, [%1], %2;" : "=r"(r) : "r"(addr), "r"(v) : "memory");
    return r;
}
// global atomic add whose result is not needed at once (the compiler's own atomicAdd aggregates over the warp and
// shuffles the result out immediately, which exposes the whole round trip)
__device__ __forceinline__ unsigned int atom_add_global_u32(unsigned int* p, unsigned int v)
{
    unsigned int r;
    asm volatile("atom.global.add.u32 %0, [%1], %2;" : "=r"(r) : "l"(p), "r"(v) : "memory");
    return r;
}
__device__ __forceinline__ void red_add_shared_u32(uint32_t addr, unsigned int v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void red_add_shared_s32(uint32_t addr, int v)
{
    asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(addr), "r"(v) : "memory");
}
__device__ __forceinline__ void red_add_shared_f32(uint32_t addr, float v)
{
    asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(addr), "f"(v) : "memory");
}
// ---- shared-memory loads / stores by 32-bit shared address (keeps address arithmetic to one add) ----------
__device__ __forceinline__ float lds_f32(uint32_t a)
{
    float r;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ unsigned int lds_u32(uint32_t a)
{
    unsigned int r;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ float2 lds_v2(uint32_t a)
{
    float2 r;
    asm volatile("ld.shared.v2.f32 {%0, %1}, [%2];" : "=f"(r.x), "=f"(r.y) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ float4 lds_v4(uint32_t a)
{
    float4 r;
    asm volatile("ld.shared.v4.f32 {%0, %1, %2, %3}, [%4];" : "=f"(r.x), "=f"(r.y), "=f"(r.z), "=f"(r.w) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ int4 lds_v4i(uint32_t a)
{
    int4 r;
    asm volatile("ld.shared.v4.s32 {%0, %1, %2, %3}, [%4];" : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ void sts_f32(uint32_t a, float v) { asm volatile("st.shared.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory"); }
__device__ __forceinline__ void sts_u32(uint32_t a, unsigned int v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_v2(uint32_t a, float x, float y)
{
    asm volatile("st.shared.v2.f32 [%0], {%1, %2};" ::"r"(a), "f"(x), "f"(y) : "memory");
}
// [profile phase: histogram slot]
// Histogram slot (0 underflow, 1+b, nbins+1 overflow/NaN).  inv != 0 means the kernel has verified at start-up
// that |(edges[i] - lo) * inv - i| <= 0.5 for every edge; the same monotone float32 expression applied to x then
// lands within one bin of the right one, and a single +-1 step against the edges makes the result exact.
__device__ __forceinline__ int slot_lean(float x, uint32_t edges_a, int nb, float lo, float inv)
{
    if (inv == 0.0f) {       // irregular axis: binary search on the edges
        if (x < lds_f32(edges_a)) return 0;
        if (!(x < lds_f32(edges_a + 4u * (unsigned)nb))) return nb + 1;
        int a = 0, b = nb;
        while (b - a > 1) {
            const int mid = (a + b) >> 1;
            if (x >= lds_f32(edges_a + 4u * (unsigned)mid)) a = mid; else b = mid;
        }
        return 1 + a;
    }
    int g = (int)((x - lo) * inv);                 // NaN -> 0, +-inf saturate
    g = max(0, min(g, nb - 1));
    const float2 ab = make_float2(lds_f32(edges_a + 4u * (unsigned)g), lds_f32(edges_a + 4u * (unsigned)g + 4u));
    int s = g + 1;
    s += (x >= ab.y) ? 1 : 0;
    s -= (x < ab.x) ? 1 : 0;
    return (x != x) ? nb + 1 : s;
}

// [profile phase: calibration bin]
// B(v) of the lookup tables (clamped bin, include/hepk.h hepk_lookup_binned) without a search: for an axis the
// kernel has verified at start-up to be uniform in v (mode 1) or in log2 v (mode 2) to within 0.45 bins, the
// arithmetic guess lands within one bin of the right one (the log2 approximation is good to 1e-5 bins), and one
// +-1 step against the edges makes it exact.  mode 0: binary search.
__device__ __forceinline__ int find_bin_fast(float v, uint32_t edges_a, int n, uint32_t axis_a)
{
    const float mode = lds_f32(axis_a);
    if (mode == 0.0f) {
        if (v < lds_f32(edges_a)) return 0;
        if (!(v < lds_f32(edges_a + 4u * (unsigned)n))) return n - 1;
        int lo = 0, hi = n;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (v >= lds_f32(edges_a + 4u * (unsigned)mid)) lo = mid; else hi = mid;
        }
        return lo;
    }
    float lg;
    asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(v));      // a guess: denormals flush to -inf and clamp to bin 0, where they belong
    const float pos = mode == 1.0f ? v : lg;
    int g = (int)((pos - lds_f32(axis_a + 4u)) * lds_f32(axis_a + 8u));       // NaN -> 0, +-inf saturate
    g = max(0, min(g, n - 1));
    const float a = lds_f32(edges_a + 4u * (unsigned)g), b = lds_f32(edges_a + 4u * (unsigned)g + 4u);
    g += (v >= b) ? 1 : 0;
    g -= (v < a) ? 1 : 0;
    g = max(0, min(g, n - 1));
    return (v != v) ? n - 1 : g;
}

// [profile phase: dR^2]
// dR^2, exact class.  Same value as dr2_exact: with a = |dphi| and t = a - 2PI_F, the wrapped magnitude is
// min(a, |t|): a > PI_F  =>  |t| <= PI_F < a (rn is monotone), a < PI_F  =>  |t| >= PI_F > a, and at a == PI_F
// both are PI_F.  Three instructions for the wrap instead of four (|.| is a free operand modifier).
__device__ __forceinline__ float dr2_min(float eta_a, float phi_a, float eta_b, float phi_b)
{
    const float deta = __fsub_rn(eta_a, eta_b);
    const float d = __fsub_rn(phi_a, phi_b);
    const float t = __fsub_rn(fabsf(d), HEPK_TWO_PI_F);
    const float w = fminf(fabsf(d), fabsf(t));
    return __fadd_rn(__fmul_rn(deta, deta), __fmul_rn(w, w));
}

// The same value from packed float32x2 operations (FADD2 rounds each half like FADD): `jet` and `lep` are (eta, phi)
// pairs, so one packed subtraction yields (deta, dphi).
__device__ __forceinline__ float dr2_packed(float2 jet, float2 lep)
{
    float r;
    asm("{\n\t"
        ".reg .b64 j, l, d;\n\t"
        ".reg .f32 dx, dy, ay, t, at, w, qx, qy;\n\t"
        "mov.b64 j, {%1, %2};\n\t"
        "mov.b64 l, {%3, %4};\n\t"
        "sub.rn.f32x2 d, j, l;\n\t"
        "mov.b64 {dx, dy}, d;\n\t"
        "abs.f32 ay, dy;\n\t"
        "add.rn.f32 t, ay, 0fC0C90FDB;\n\t"      // |dphi| - 2PI_F
        "abs.f32 at, t;\n\t"
        "min.f32 w, ay, at;\n\t"
        "mul.rn.f32 qx, dx, dx;\n\t"             // (a packed multiply of a pair by itself costs two register moves)
        "mul.rn.f32 qy, w, w;\n\t"
        "add.rn.f32 %0, qx, qy;\n\t"
        "}"
        : "=f"(r)
        : "f"(jet.x), "f"(jet.y), "f"(lep.x), "f"(lep.y));
    return r;
}

// [profile phase: feature word]
// What the launch asked for, as one register of flags (tested with one instruction instead of a pointer compare).
enum : unsigned {
    F_NJET = 1u << 0, F_ARGMAX = 1u << 1, F_HT = 1u << 2, F_MAXPT = 1u << 3, F_MINPT = 1u << 4, F_MJJ = 1u << 5,
    F_SUBPT = 1u << 6, F_OBS0 = 1u << 8 /* .. << 13 */, F_COUNTS = 1u << 16, F_SUMW = 1u << 17, F_WEIGHTS = 1u << 18, F_MULTIW = 1u << 19 /* more than one weight column */,
    F_SUMW2 = 1u << 20, F_EVW = 1u << 21
};
__device__ __forceinline__ unsigned chain_features(const ChainParams& P)
{
    unsigned f = 0;
    if (P.out_njet) f |= F_NJET;
    if (P.out_argmax) f |= F_ARGMAX;
    if (P.out_ht) f |= F_HT;
    if (P.out_maxpt) f |= F_MAXPT;
    if (P.out_minpt) f |= F_MINPT;
    if (P.out_mjj) f |= F_MJJ;
    if (P.out_subpt) f |= F_SUBPT;
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob)
        if (P.axis_edges[ob]) f |= F_OBS0 << ob;
    if (P.col_cnt >= 0) f |= F_COUNTS;
    if (P.hist_acc && P.hist_sumw) f |= F_SUMW;
    if (P.col_w2 >= 0) f |= F_SUMW2;
    if (P.weights) f |= F_WEIGHTS;
    if (P.W > 1) f |= F_MULTIW;
    if (P.evw_table) f |= F_EVW;
    return f;
}

// [profile phase: histogram fill]
// Slot of one observable: bumps its count and returns the shared-memory address of its bin in weight column 0
// (0 when the observable is not histogrammed).  sumw layout [v][o][w][nbins_o + 2].
// Shared-memory address of the slot row (all columns of one slot) of observable OB for value x; 0: not histogrammed.
template <int OB>
__device__ __forceinline__ uint32_t obs_row(const ChainParams& P, const ChainShared& S, unsigned feat, int v, float x)
{
    if (!(feat & (F_OBS0 << OB))) return 0u;
    const int nb = P.axis_nbins[OB];
    const int slot = slot_lean(x, smem_u32(S.edges) + 4u * (unsigned)P.edge_prefix[OB], nb, lds_f32(smem_u32(S.axis_lo) + 4u * OB),
                               lds_f32(smem_u32(S.axis_inv) + 4u * OB));
    return smem_u32(S.h_bins) + 4u * (unsigned)((v * P.obs_prefix[HEPK_N_OBS] + P.obs_prefix[OB] + slot) * P.WS);
}

// One value into column `col` of the slot rows of the active observables.  Fixed point (FIXED): q is the weight
// rounded once to a multiple of 2^-k, added with the native integer shared-memory atomic; else the float weight
// (a compare-and-swap loop in hardware).
template <bool FIXED>
__device__ __forceinline__ void add_column(unsigned feat, const uint32_t (&row)[HEPK_N_OBS], int col, int q, float wt)
{
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!(feat & (F_OBS0 << ob))) continue;
        const uint32_t a = row[ob] + 4u * (unsigned)col;
        if (FIXED) red_add_shared_s32(a, q);
        else red_add_shared_f32(a, wt);
    }
}

// All weight columns of one event into its slot rows.
template <bool FIXED, int NW>
__device__ __forceinline__ void add_weights(const ChainParams& P, unsigned feat, const uint32_t (&row)[HEPK_N_OBS],
                                            const float (&wt)[NW], long long ev, float evf, float sc, float sc2)
{
    const bool w2 = (feat & F_SUMW2) != 0, w1 = (feat & F_SUMW) != 0;
    auto one = [&](int w, float x) {
        if (w1) add_column<FIXED>(feat, row, w, FIXED ? __float2int_rn(x * sc) : 0, x);
        if (w2) {
            // squared weights span the square of the weights' range: two fixed-point columns per weight, the second
            // holding the rounding remainder of the first at 2^20 times its scale (both exact integers below 2^19)
            const float x2 = x * x, y = x2 * sc2;
            const int qh = FIXED ? __float2int_rn(y) : 0;
            add_column<FIXED>(feat, row, P.col_w2 + 2 * w, qh, x2);
            if (FIXED) add_column<true>(feat, row, P.col_w2 + 2 * w + 1, __float2int_rn((y - (float)qh) * 1048576.0f), 0.0f);
        }
    };
    one(0, wt[0]);
    if ((feat & (F_WEIGHTS | F_MULTIW)) != (F_WEIGHTS | F_MULTIW)) return;
    if (NW > 1) {
        // the event's weights were loaded once per tile and serve every variant and observable
#pragma unroll
        for (int w = 1; w < NW; ++w)
            if (w < P.W) one(w, wt[w]);
    } else {
        // eight loads in flight, then their fills (one memory latency per eight columns, not per column)
        for (int w0 = 1; w0 < P.W; w0 += 8) {
            float x[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) x[k] = w0 + k < P.W ? __ldg(P.weights + (long long)(w0 + k) * P.w_stride + ev) : 0.0f;
#pragma unroll
            for (int k = 0; k < 8; ++k)
                if (w0 + k < P.W) one(w0 + k, (feat & F_EVW) ? __fmul_rn(x[k], evf) : x[k]);
        }
    }
}

// [profile phase: finish_event: outputs, slots, fills]
// Per event and variant: leading-pair mass, outputs, histograms.  Shared by the staged path and the per-event
// path.  The leading jets' (eta, phi, mass) are passed in by value; i2 < 0 means fewer than two clean jets.
template <int NW>
__device__ __forceinline__ void finish_event(const ChainParams& P, const ChainShared& S, unsigned feat, long long ev, int v,
                                             const float (&wt)[NW], float evf,
                                             int cnt, float sum, float mn, float b1, float b2, int i1, int i2,
                                             float eta1, float phi1, float m1, float eta2, float phi2, float m2)
{
    float mjj = 0.0f, subpt = 0.0f;
    const bool hists = (feat & (F_COUNTS | F_SUMW)) != 0;
    if (i2 >= 0) {
        subpt = b2;
        mjj = pair_mass_lean(b1, eta1, phi1, m1, b2, eta2, phi2, m2);
        if (hists && (feat & (F_OBS0 << HEPK_OBS_MJJ))) {
            // the bin of mjj is decided by the float64-defined value: refine when the fast value is near an edge
            const uint32_t ed = smem_u32(S.edges) + 4u * (unsigned)P.edge_prefix[HEPK_OBS_MJJ];
            const int nb = P.axis_nbins[HEPK_OBS_MJJ];
            const int s = slot_lean(mjj, ed, nb, lds_f32(smem_u32(S.axis_lo) + 4u * HEPK_OBS_MJJ),
                                    lds_f32(smem_u32(S.axis_inv) + 4u * HEPK_OBS_MJJ));
            const float band = fmaf(mjj, HEPK_MASS_GUARD_REL, HEPK_MASS_GUARD_ABS);
            const bool near_lo = s >= 1 && mjj - lds_f32(ed + 4u * (unsigned)(s - 1)) <= band;
            const bool near_hi = s <= nb && lds_f32(ed + 4u * (unsigned)s) - mjj <= band;
            if (near_lo || near_hi) mjj = pair_mass_f64(b1, eta1, phi1, m1, b2, eta2, phi2, m2);
        }
    }
    const long long o = (long long)v * P.out_stride + ev;
    if (feat & F_NJET) P.out_njet[o] = cnt;
    if (feat & F_ARGMAX) P.out_argmax[o] = i1;
    if (feat & F_HT) P.out_ht[o] = sum;
    if (feat & F_MAXPT) P.out_maxpt[o] = b1;
    if (feat & F_MINPT) P.out_minpt[o] = mn;
    if (feat & F_MJJ) P.out_mjj[o] = mjj;
    if (feat & F_SUBPT) P.out_subpt[o] = subpt;
    if (!hists) return;
    uint32_t row[HEPK_N_OBS];
    row[HEPK_OBS_NJET] = obs_row<HEPK_OBS_NJET>(P, S, feat, v, (float)cnt);
    row[HEPK_OBS_HT] = obs_row<HEPK_OBS_HT>(P, S, feat, v, sum);
    row[HEPK_OBS_MAXPT] = obs_row<HEPK_OBS_MAXPT>(P, S, feat, v, b1);
    row[HEPK_OBS_MINPT] = obs_row<HEPK_OBS_MINPT>(P, S, feat, v, mn);
    row[HEPK_OBS_MJJ] = obs_row<HEPK_OBS_MJJ>(P, S, feat, v, mjj);
    row[HEPK_OBS_SUBPT] = obs_row<HEPK_OBS_SUBPT>(P, S, feat, v, subpt);
    if (feat & F_COUNTS) {
#pragma unroll
        for (int ob = 0; ob < HEPK_N_OBS; ++ob)
            if (feat & (F_OBS0 << ob)) red_add_shared_u32(row[ob] + 4u * (unsigned)P.col_cnt, 1u);
    }
    if (!(feat & (F_SUMW | F_SUMW2))) return;
    const float2 sc = lds_v2(smem_u32(S.wscale));
    if (sc.x != 0.0f) add_weights<true, NW>(P, feat, row, wt, ev, evf, sc.x, sc.y);
    else add_weights<false, NW>(P, feat, row, wt, ev, evf, 0.0f, 0.0f);
}

// [profile phase: per-event reduction state (push)]
// Order-preserving map float -> unsigned (and back): a < b  <=>  ord_key(a) < ord_key(b); no finite value maps to 0.
__device__ __forceinline__ unsigned int ord_key(float f)
{
    const unsigned int b = __float_as_uint(f);
    return b ^ ((unsigned int)((int)b >> 31) | 0x80000000u);
}
__device__ __forceinline__ float ord_value(unsigned int u)
{
    return __uint_as_float(u ^ ((u & 0x80000000u) ? 0x80000000u : 0xffffffffu));
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
    // top-2 part of push for a value that counts
    __device__ __forceinline__ void push_top(float p, int k)
    {
        const bool gt1 = p > b1, gt2 = p > b2;
        i2 = gt1 ? i1 : (gt2 ? k : i2);
        i1 = gt1 ? k : i1;
        b2 = gt1 ? b1 : (gt2 ? p : b2);
        b1 = gt1 ? p : b1;
    }
    // The same update for a jet that counts iff p > pt_min (p may be anything, NaN included, otherwise), written
    // with predicated instructions: 3 compares, 1 convert and 9 predicated operations.
    __device__ __forceinline__ void push_lean_nomin(float p, float pt_min, int k)
    {
        asm("{\n\t"
            ".reg .pred ok, g1, g2;\n\t"
            ".reg .f64 pd;\n\t"
            ".reg .f32 pz;\n\t"
            "setp.gt.f32 ok, %7, %8;\n\t"
            "setp.gt.and.f32 g1, %7, %4, ok;\n\t"
            "setp.gt.and.f32 g2, %7, %5, ok;\n\t"
            "selp.f32 pz, %7, 0f00000000, ok;\n\t"
            "cvt.f64.f32 pd, pz;\n\t"
            "@ok add.s32 %0, %0, 1;\n\t"
            "add.f64 %1, %1, pd;\n\t"
            "@g2 mov.b32 %6, %9;\n\t"
            "@g1 mov.b32 %6, %3;\n\t"
            "@g1 mov.b32 %3, %9;\n\t"
            "@g2 mov.f32 %5, %7;\n\t"
            "@g1 mov.f32 %5, %4;\n\t"
            "@g1 mov.f32 %4, %7;\n\t"
            "}"
            : "+&r"(cnt), "+&d"(sum), "+&f"(mn), "+&r"(i1), "+&f"(b1), "+&f"(b2), "+&r"(i2)
            : "f"(p), "f"(pt_min), "r"(k));
    }
    template <bool NEED_MIN>
    __device__ __forceinline__ void push_lean(float p, float pt_min, int k)
    {
        if (!NEED_MIN) { push_lean_nomin(p, pt_min, k); return; }
        asm("{\n\t"
            ".reg .pred ok, g1, g2;\n\t"
            ".reg .f64 pd;\n\t"
            ".reg .f32 pz;\n\t"
            "setp.gt.f32 ok, %7, %8;\n\t"
            "setp.gt.and.f32 g1, %7, %4, ok;\n\t"
            "setp.gt.and.f32 g2, %7, %5, ok;\n\t"
            "selp.f32 pz, %7, 0f00000000, ok;\n\t"
            "cvt.f64.f32 pd, pz;\n\t"
            "@ok add.s32 %0, %0, 1;\n\t"
            "add.f64 %1, %1, pd;\n\t"
            "@ok min.f32 %2, %2, %7;\n\t"
            "@g2 mov.b32 %6, %9;\n\t"
            "@g1 mov.b32 %6, %3;\n\t"
            "@g1 mov.b32 %3, %9;\n\t"
            "@g2 mov.f32 %5, %7;\n\t"
            "@g1 mov.f32 %5, %4;\n\t"
            "@g1 mov.f32 %4, %7;\n\t"
            "}"
            : "+&r"(cnt), "+&d"(sum), "+&f"(mn), "+&r"(i1), "+&f"(b1), "+&f"(b2), "+&r"(i2)
            : "f"(p), "f"(pt_min), "r"(k));
    }
};

// [profile phase: histogram scales]
// Fixed-point scales of the weighted bins (R18) from the weight range in the workspace header: entries are
// rint(w * 2^k) with |w| * 2^k < 2^19 (2^k2 likewise for w^2).  A bin is checked at least every ~1024 events of the
// CTA plus the tiles in flight and moved out at 2^29, so it stays below 2^31.  The rounding error per entry is
// <= 2^-20 max|w|, so the scheme is taken only when the weights span at most a factor 8 (error <= 7.7e-6 of the
// smallest entry); otherwise sc = sc2 = 0: float bins.
__device__ __forceinline__ void hist_scales(const ChainParams& P, float& sc, float& sc2)
{
    sc = sc2 = 0.0f;
    if (!P.hist_hdr || P.hist_hdr[HDR_BAD] != 0u) return;
    const float tmax = P.evw_table ? __uint_as_float(P.hist_hdr[HDR_TMAX]) : 1.0f;
    const float tmin = P.evw_table ? __uint_as_float(~P.hist_hdr[HDR_TMIN]) : 1.0f;      // (never updated: NaN, and the scheme is off)
    const float wm = __uint_as_float(P.hist_hdr[HDR_WMAX]) * tmax;
    const float wn = __uint_as_float(~P.hist_hdr[HDR_WMIN]) * tmin;
    if (!(wm > 0.0f && wm < CUDART_INF_F && wn > 0.0f && wm <= 8.0f * wn)) return;
    if (!(wm * wm < CUDART_INF_F && wn * wn > 0.0f)) return;
    int e, e2;
    frexpf(wm, &e);                                    // wm < 2^e
    frexpf(wm * wm, &e2);
    const int k = 19 - e, k2 = 19 - e2;
    if (k <= -100 || k >= 100 || k2 <= -100 || k2 >= 100) return;
    sc = ldexpf(1.0f, k);
    sc2 = ldexpf(1.0f, k2);
}

// [profile phase: event-weight factor]
// Per-event weight factor table[B(x)] (hepk_lookup_binned's clamped bin, 1-D) from the staged lookup.
__device__ __forceinline__ float evw_factor(const ChainParams& P, const ChainShared& S, long long ev)
{
    const float x = __ldg(P.evw_x + ev);
    const int n = P.evw_nbins;
    const uint32_t ed = smem_u32(S.evw_edges);
    int b;
    if (x < lds_f32(ed)) b = 0;
    else if (!(x < lds_f32(ed + 4u * (unsigned)n))) b = n - 1;
    else {
        int lo = 0, hi = n;
        while (hi - lo > 1) {
            const int mid = (lo + hi) >> 1;
            if (x >= lds_f32(ed + 4u * (unsigned)mid)) lo = mid; else hi = mid;
        }
        b = lo;
    }
    return lds_f32(smem_u32(S.evw_table) + 4u * (unsigned)b);
}

// [profile phase: per-event fallback path]
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
__device__ __noinline__ void chain_event_global(const ChainParams& P, unsigned char* smem_base, long long ev)
{
    ChainShared S;          // rebuilt here: passing the caller's by reference would force it into local memory
    chain_shared_layout(P, CALIB, smem_base, &S);
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
        const float evf = P.evw_table ? evw_factor(P, S, ev) : 1.0f;
        const float w0 = P.weights ? __ldg(P.weights + ev) : 1.0f;
        const float wt[1] = {P.evw_table ? __fmul_rn(w0, evf) : w0};
        finish_event<1>(P, S, chain_features(P), ev, v, wt, evf, a.cnt, (float)a.sum, a.mn, a.b1, a.b2, a.i1, a.i2, e1, p1, m1, e2, p2, m2);
    }
}

// [profile phase: histogram flush]
// Move privatised bins [i0, i1) of the CTA into the global accumulators (thread t of nt).  Safe against concurrent
// fills by other warps: a bin is taken with an atomic exchange.  Fixed-point and count columns are exact integers,
// so they only move when `all` is set or the bin is about to leave the int32 range (|bin| >= FLUSH_AT); float bins
// move whenever they are non-zero (their rounding error grows with their content).
__device__ __forceinline__ void flush_bins(const ChainParams& P, const ChainShared& S, int i0, int i1, int t, int nt, bool all)
{
    const bool fixed = S.wscale[0] != 0.0f;
    int* bins = (int*)S.h_bins;
    const int WS = P.WS, ccol = P.col_cnt;
    for (int i = i0 + t; i < i1; i += nt) {
        const int x = bins[i];
        if (x == 0) continue;                         // +0.0f and integer 0 share the bit pattern
        const bool is_int = fixed || (i % WS) == ccol;
        if (is_int) {
            if (!all && (unsigned)(x + FLUSH_AT) < 2u * (unsigned)FLUSH_AT) continue;      // |x| < FLUSH_AT
            const int y = atomicExch(bins + i, 0);
            if (y) atomicAdd((unsigned long long*)P.hist_acc + i, (unsigned long long)(long long)y);
        } else {
            const float y = atomicExch((float*)bins + i, 0.0f);
            if (y != 0.0f) atomicAdd((double*)P.hist_acc + i, (double)y);
        }
    }
}

// [profile phase: offsets load]
// Low words of offsets[e] and offsets[e+1] of the lane's event (lane = event of the tile), three collections.
struct EventOffsets { int j0, j1, m0, m1, q0, q1; };

template <bool HAS_EL>
__device__ __forceinline__ void load_event_offsets(const ChainParams& P, long long tile, int lane, EventOffsets& o)
{
    const long long e = tile * TILE_EVENTS + lane;
    long long i0 = e, i1 = e + 1;
    if ((tile + 1) * TILE_EVENTS > P.n_events) {        // only the last tile can be ragged (uniform branch)
        i0 = e < P.n_events ? e : P.n_events;
        i1 = e + 1 < P.n_events ? e + 1 : P.n_events;
    }
    o.j0 = (int)__ldg(P.off[0] + i0); o.j1 = (int)__ldg(P.off[0] + i1);
    o.m0 = (int)__ldg(P.off[1] + i0); o.m1 = (int)__ldg(P.off[1] + i1);
    if (HAS_EL) { o.q0 = (int)__ldg(P.off[2] + i0); o.q1 = (int)__ldg(P.off[2] + i1); }
    else { o.q0 = 0; o.q1 = 0; }
}

// one lane of the (converged) warp
__device__ __forceinline__ bool elect_one()
{
    unsigned int pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0u;
}

// [profile phase: TMA issue]
// Start the bulk copies of a tile whose slices start at global element lo[k] and hold cnt[k] elements (k: jets, muons,
// electrons) into the warp's staging region; all 32 lanes call it, converged, with the same arguments in every lane.
// Returns false (nothing issued) when a slice does not fit: capacity, 16-byte alignment at the array ends.
// Element l of a column lands at buffer index l - a0, a0 = l0 - ((l0 + mis) mod 4), so every copy is 16-byte aligned
// on both sides; the consumer recomputes the same shift.  One lane issues all copies: its operands are then uniform
// by construction (a bulk copy takes uniform registers; copies issued from several lanes are serialised with a
// register hand-over per operand and lane).
template <bool HAS_EL>
__device__ __forceinline__ bool issue_tile(const ChainParams& P, uint32_t region_a, int lane, const int (&lo)[3],
                                           const int (&cnt)[3])
{
    int a0[3];
    int len[3], tail[3] = {0, 0, 0};
    int bad = 0, edge = 0;
#pragma unroll
    for (int k = 0; k < (HAS_EL ? 3 : 2); ++k) {
        const int c0 = k == 0 ? 0 : (k == 1 ? 4 : 7);
        // low words only: the staged path requires n_objects < 2^31, so offsets[e0] - content_base fits an int
        const int l0 = (int)((unsigned)lo[k] - (unsigned)P.col_base[c0]);
        const int sh = (l0 + P.col_mis[c0]) & 3;
        a0[k] = l0 - sh;
        const int ln = (cnt[k] + sh + 3) & ~3;
        // fits: 0 <= cnt <= capacity, 0 <= a0 and the slice ends inside the array (an empty slice always fits).  Sign
        // bits, no branches.  At the very end of an array the aligned window may reach past it: the bulk copy then
        // stops at the last full 16 bytes and the (at most three) elements beyond are moved by ordinary loads.
        const int e0k = cnt[k] != 0 ? a0[k] : 0;
        a0[k] = e0k;
        len[k] = cnt[k] != 0 ? ln : 0;
        edge |= P.col_n32[k] - e0k - len[k];           // negative: the aligned window reaches past the array
        bad |= cnt[k] | (P.col_cap[c0] - cnt[k]) | e0k | (P.col_n32[k] - l0 - cnt[k]);
    }
    if (bad < 0) return false;
    if (edge < 0) {          // (uniform, rare: the last tile of a launch)
#pragma unroll
        for (int k = 0; k < (HAS_EL ? 3 : 2); ++k) {
            const int c0 = k == 0 ? 0 : (k == 1 ? 4 : 7);
            if (a0[k] + len[k] > P.col_n32[k]) {
                const int l0 = (int)((unsigned)lo[k] - (unsigned)P.col_base[c0]);
                const int lb = (P.col_n32[k] - a0[k]) & ~3;
                tail[k] = l0 + cnt[k] - a0[k] - lb;    // elements of the slice past the bulk copy (0..3)
                len[k] = lb;
            }
        }
#pragma unroll
        for (int c = 0; c < (HAS_EL ? NCOL : 7); ++c) {
            const int k = c < 4 ? 0 : (c < 7 ? 1 : 2);
            if (lane < tail[k])
                sts_f32(region_a + (uint32_t)P.col_dst[c] + 4u * (unsigned)(len[k] + lane),
                        __ldg(reinterpret_cast<const float*>(P.col_ptr[c]) + a0[k] + len[k] + lane));
        }
    }
    const uint32_t total = (uint32_t)len[0] * 16u + (uint32_t)(len[1] + (HAS_EL ? len[2] : 0)) * 12u;
    // One elected lane issues all copies.  Under elect.sync (and with operands that come from warp reductions, hence
    // uniform registers) each copy is one UBLKCP; under `lane == 0` the compiler wraps every copy in a loop over the
    // lanes that might be active.
    if (elect_one()) {
        uint64_t* bar = nullptr;
        const uint32_t bar_a = region_a;
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar_a), "r"(total) : "memory");
        (void)bar;
#pragma unroll
        for (int c = 0; c < (HAS_EL ? NCOL : 7); ++c) {
            const int k = c < 4 ? 0 : (c < 7 ? 1 : 2);
            if (len[k] != 0)
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                 region_a + (uint32_t)P.col_dst[c]),
                             "l"(P.col_ptr[c] + ((long long)a0[k] << 2)), "r"((uint32_t)len[k] << 2), "r"(bar_a)
                             : "memory");
        }
    }
    return true;
}

// [profile phase: kernel setup]
// NW: weight columns of an event kept in registers (1, or HEPK_MAX_WVAR for launches with several columns)
template <bool CALIB, bool HAS_EL, int MAXT, int FEAT, int NW = 1>
__global__ void __launch_bounds__(MAXT, 1) chain_kernel(const __grid_constant__ ChainParams P)
{
    extern __shared__ __align__(128) unsigned char smem_raw[];
    ChainShared S;
    chain_shared_layout(P, CALIB, smem_raw, &S);
    const int tid = threadIdx.x, nthr = blockDim.x;
    const int warp = __reduce_min_sync(0xffffffffu, tid >> 5);  // through a warp reduction: its result lives in a uniform register, and so does every address derived from it
    const int lane = tid & 31, nwarp = nthr >> 5;
    unsigned char* R = smem_raw + P.shared_bytes + (size_t)warp * P.region_bytes;   // this warp's staging region
    uint64_t* bar = (uint64_t*)R;

    // ---- one-time setup: barrier, axis edges, calibration tables, zeroed histograms
    if (lane == 0) {
        mbar_init(bar, 1);
        fence_mbar_init();
    }
    if (lane < 2 * N_BUCKETS) ((int*)(R + P.bucket_off))[lane] = 0;
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        for (int i = tid; i <= nb; i += nthr) S.edges[P.edge_prefix[ob] + i] = P.axis_edges[ob][i];
    }
    if (CALIB) {
        for (int i = tid; i <= P.cal_npt; i += nthr) S.cal_pt_edges[i] = P.cal_pt_edges[i];
        for (int i = tid; i <= P.cal_neta; i += nthr) S.cal_eta_edges[i] = P.cal_eta_edges[i];
        for (int i = tid; i < P.cal_npt * P.cal_neta; i += nthr) S.cal_table[i] = P.cal_table[i];
    }
    {
        const int spv = P.obs_prefix[HEPK_N_OBS];
        if (P.hist_acc) for (int i = tid; i < spv * P.V * P.WS; i += nthr) S.h_bins[i] = 0u;
        if (P.evw_table) {
            for (int i = tid; i <= P.evw_nbins; i += nthr) S.evw_edges[i] = P.evw_edges[i];
            for (int i = tid; i < P.evw_nbins; i += nthr) S.evw_table[i] = P.evw_table[i];
        }
        if (tid == 0) {
            float sc, sc2;
            hist_scales(P, sc, sc2);
            S.wscale[0] = sc; S.wscale[1] = sc2;
            *S.scan = 0u;
            *S.next = 0u;
        }
    }
    __syncthreads();
    // per axis: is the arithmetic bin guess of slot_lean safe?  (|(edges[i] - lo) * inv - i| <= 0.5 for every edge)
#pragma unroll
    for (int ob = 0; ob < HEPK_N_OBS; ++ob) {
        if (!P.axis_edges[ob]) continue;
        const int nb = P.axis_nbins[ob];
        const float* ed = S.edges + P.edge_prefix[ob];
        const float lo = ed[0], hi = ed[nb];
        const float inv = (float)nb / (hi - lo);
        bool ok = (hi > lo) && (inv > 0.0f) && (inv < CUDART_INF_F);
        for (int i = tid; i <= nb; i += nthr) ok = ok && (fabsf((ed[i] - lo) * inv - (float)i) <= 0.5f);
        ok = __syncthreads_and(ok);
        if (tid == 0) {
            S.axis_lo[ob] = lo;
            S.axis_inv[ob] = ok ? inv : 0.0f;
        }
    }
    if (CALIB) {
#pragma unroll
        for (int ax = 0; ax < 2; ++ax) {
            const float* ed = ax == 0 ? S.cal_pt_edges : S.cal_eta_edges;
            const int nb = ax == 0 ? P.cal_npt : P.cal_neta;
            const float lo = ed[0], hi = ed[nb];
            const float inv1 = (float)nb / (hi - lo);
            const float l0 = __log2f(lo), inv2 = (float)nb / (__log2f(hi) - l0);
            bool ok1 = (hi > lo) && (inv1 > 0.0f) && (inv1 < CUDART_INF_F);
            bool ok2 = (lo > 0.0f) && (hi > lo) && (inv2 > 0.0f) && (inv2 < CUDART_INF_F);
            for (int i = tid; i <= nb; i += nthr) {
                ok1 = ok1 && (fabsf((ed[i] - lo) * inv1 - (float)i) <= 0.45f);
                ok2 = ok2 && (fabsf((__log2f(ed[i]) - l0) * inv2 - (float)i) <= 0.45f);
            }
            ok1 = __syncthreads_and(ok1);
            ok2 = __syncthreads_and(ok2);
            if (tid == 0) {
                S.cal_axis[4 * ax + 0] = ok1 ? 1.0f : (ok2 ? 2.0f : 0.0f);
                S.cal_axis[4 * ax + 1] = ok1 ? lo : l0;
                S.cal_axis[4 * ax + 2] = ok1 ? inv1 : inv2;
            }
        }
    }
    __syncthreads();

    // this warp's buffers (shared-memory byte addresses)
    const uint32_t region_a = smem_u32(R);
    const uint32_t order_a = region_a + (uint32_t)P.order_off;
    const uint32_t lep_a = region_a + (uint32_t)P.lep_off;
    const uint32_t corr_a = region_a + (uint32_t)P.corr_off;
    const uint32_t bucket_a = region_a + (uint32_t)P.bucket_off;
    const int V = CALIB ? P.V : 1;
    // FEAT >= 0: the launch's feature word is known at compile time (the common analysis shape; one weight column),
    // so everything it does not ask for is compiled out
    const unsigned feat = FEAT >= 0 ? (unsigned)FEAT : chain_features(P);

    // [profile phase: tile hand-out, prefetch of offsets and weights]
    // Tile hand-out.  Every CTA owns a contiguous range of tiles and its warps draw from it through a shared-memory
    // ticket, so a scheduler with one warp more than its neighbours (or a warp that met long events) simply takes
    // fewer tiles; the last eighth of the launch is handed out by a global counter so that no SM idles at the end.
    const bool dyn = P.tile_counter != nullptr;
    // (tile indices fit 32 bits: the host refuses launches of 2^31 tiles or more)
    const unsigned int NT = (unsigned int)P.n_tiles;
    const unsigned int per_cta = dyn ? (NT - NT / 8u) / gridDim.x : (NT + gridDim.x - 1u) / gridDim.x;
    const unsigned int n_static = dyn ? per_cta * gridDim.x : NT;
    const unsigned int cta_lo = blockIdx.x * per_cta;
    const uint32_t next_a = smem_u32(S.next);
    unsigned int ticket = 0;          // of the tile taken last: also picks the slice of bins this warp checks next
    auto take_tile = [&]() -> unsigned int {
        unsigned int i = 0;
        if (elect_one()) i = atom_add_shared_u32(next_a, 1u);
        i = __reduce_max_sync(0xffffffffu, i);      // the elected lane's value, in a uniform register
        ticket = i;
        if (i < per_cta) return min(cta_lo + i, NT);
        if (!dyn) return NT;
        unsigned int g = 0;
        if (elect_one()) g = atom_add_global_u32(P.tile_counter, 1u);
        g = __reduce_max_sync(0xffffffffu, g);
        return g < NT - n_static ? n_static + g : NT;
    };
    unsigned int tile = take_tile();
    uint32_t parity = 0;
    int bsel = 0;
    bool fit = false;
    EventOffsets eo;
    eo.j0 = eo.j1 = eo.m0 = eo.m1 = eo.q0 = eo.q1 = 0;
    // object counts of a tile from the per-lane offsets (lanes past the last event hold offsets[n_events])
    auto tile_counts = [&](const EventOffsets& o, int (&lo)[3], int (&cnt)[3]) {
        // offsets do not decrease: lane 0 holds the smallest start, lane 31 the largest end.  Warp reductions rather
        // than shuffles: their results are uniform registers, so the slice arithmetic runs on the uniform datapath
        lo[0] = __reduce_min_sync(0xffffffffu, o.j0); cnt[0] = __reduce_max_sync(0xffffffffu, o.j1) - lo[0];
        lo[1] = __reduce_min_sync(0xffffffffu, o.m0); cnt[1] = __reduce_max_sync(0xffffffffu, o.m1) - lo[1];
        lo[2] = HAS_EL ? __reduce_min_sync(0xffffffffu, o.q0) : 0;
        cnt[2] = HAS_EL ? __reduce_max_sync(0xffffffffu, o.q1) - lo[2] : 0;
    };
    int lo[3] = {0, 0, 0}, cnt[3] = {0, 0, 0};      // first object and object count of the current tile's slices (uniform)
    if (tile < NT) {
        load_event_offsets<HAS_EL>(P, tile, lane, eo);
        tile_counts(eo, lo, cnt);
        fit = P.n_col > 0 && issue_tile<HAS_EL>(P, smem_u32(R), lane, lo, cnt);
    }

    unsigned int tile_next = take_tile();

    for (; tile < NT;) {
        const long long e0 = (long long)tile * TILE_EVENTS;
        const long long rest = P.n_events - e0;
        const int ne = rest < TILE_EVENTS ? (int)rest : TILE_EVENTS;
        const bool has_next = tile_next < NT;
        float wt[NW];                                                    // weights of the lane's event, loaded early
        float evf = 1.0f;                                                // its weight factor from the lookup
        if ((feat & F_EVW) && (feat & (F_SUMW | F_SUMW2)) && lane < ne) evf = evw_factor(P, S, e0 + lane);
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            wt[w] = 1.0f;
            if ((feat & F_WEIGHTS) && (feat & (F_SUMW | F_SUMW2)) && lane < ne && w < P.W)
                wt[w] = __ldg(P.weights + (long long)w * P.w_stride + e0 + lane);
            if (feat & F_EVW) wt[w] = __fmul_rn(wt[w], evf);             // one float32 multiply (exact class)
        }
        EventOffsets neo;      // (without a next tile the current one is read again: harmless, and no branch)
        load_event_offsets<HAS_EL>(P, has_next ? tile_next : tile, lane, neo);
        bool staged = fit;
        bool released = false;
        fit = false;
        int nlo[3] = {0, 0, 0}, ncnt[3] = {0, 0, 0};                    // the same for the next tile

        if (staged) {
            // [profile phase: phase 0: tile geometry, buckets]
            // ---- phase 0: one lane per event.  Offsets are in registers.
            const int jb = lo[0], mb = lo[1], qb = lo[2];
            const int njt = cnt[0];
            // shared-memory byte addresses; the columns of one collection share alignment and sit STRIDE apart
            const uint32_t a_jpt = region_a + (uint32_t)P.col_dst[0] + 4u * (unsigned)((jb + P.sh_add[0]) & 3);
            const uint32_t a_mpt = region_a + (uint32_t)P.col_dst[4] + 4u * (unsigned)((mb + P.sh_add[4]) & 3);
            const uint32_t a_ept = region_a + (uint32_t)P.col_dst[7] + 4u * (unsigned)((qb + P.sh_add[7]) & 3);
            const uint32_t js = (uint32_t)P.col_stride[0], ms = (uint32_t)P.col_stride[1], es = (uint32_t)P.col_stride[2];
            const uint32_t d_corr0 = corr_a - a_jpt;     // calibration factor of the jet whose pt sits at address x: x + d_corr0
            const bool live = lane < ne;
            const int kj0 = live ? eo.j0 - jb : 0, nj = live ? eo.j1 - eo.j0 : 0;
            const int km0 = eo.m0 - mb, nm = live ? eo.m1 - eo.m0 : 0;
            const int kq0 = eo.q0 - qb, nq = (HAS_EL && live) ? eo.q1 - eo.q0 : 0;
            const int c = nm + nq;          // every lepton gets a list entry; unselected ones can never match
            const int npair = (c + 1) >> 1; // the list is padded to pairs with an entry that can never match
            // every event's list starts at an even entry (16-byte aligned pairs): the running lepton count plus one
            // possible pad entry per earlier event, rounded up to even
            const int l0 = live ? (km0 + kq0 + lane + 1) & ~1 : 0;
            const unsigned longm = __ballot_sync(0xffffffffu, nj > TAIL_CUT);   // events whose tail the warp shares
            // bucket the event's jets by its number of lepton pairs: position inside the bucket from a shared-memory
            // counter (any order inside a bucket will do), bucket bases from the eight totals
            const int key = npair < N_BUCKETS - 1 ? npair : N_BUCKETS - 1;
            const uint32_t bk = bucket_a + (uint32_t)bsel * (4u * N_BUCKETS);
            int pos = 0;
            if (nj > 0) pos = (int)atom_add_shared_u32(bk + 4u * (unsigned)key, (unsigned)nj);
            if (lane < N_BUCKETS) sts_u32(bucket_a + (uint32_t)(bsel ^ 1) * (4u * N_BUCKETS) + 4u * lane, 0u);   // other set, for the next tile
            // an event with more leptons than the packed word can count: the whole tile goes the slow way
            staged = !__any_sync(0xffffffffu, c > MAX_LEP_EVENT);
            mbar_wait(bar, parity);
            parity ^= 1u;
            if (staged) {
                // [profile phase: phase 0: lepton list]
                // combined (eta, phi) list of the event: muons then electrons; eta = +inf marks "not selected"
                // (deta^2 = inf, so dR^2 = inf or NaN and the minimum below ignores it).  Straight-line predicated
                // code for the first few leptons of each kind (a divergent loop costs more than the work it does).
                uint32_t out = lep_a + 8u * (unsigned)l0;            // (l0 <= MAX_LIST by the capacities)
                float lep_pt_min = P.lep_pt_min;
                // pinned in registers: the predicated blocks below would otherwise each recompute the address and reload the cut
                asm volatile("" : "+r"(out), "+f"(lep_pt_min));
                {
                    const uint32_t a = a_mpt + 4u * (unsigned)km0;
                    constexpr int UNR_M = 5;
#pragma unroll
                    for (int k = 0; k < UNR_M; ++k)
                        if (k < nm) {
                            const float pt = lds_f32(a + 4u * k), eta = lds_f32(a + ms + 4u * k), phi = lds_f32(a + 2 * ms + 4u * k);
                            sts_v2(out + 8u * k, pt > lep_pt_min ? eta : CUDART_INF_F, phi);
                        }
#pragma unroll 1
                    for (int k = UNR_M; k < nm; ++k) {
                        const float pt = lds_f32(a + 4u * k), eta = lds_f32(a + ms + 4u * k), phi = lds_f32(a + 2 * ms + 4u * k);
                        sts_v2(out + 8u * k, pt > lep_pt_min ? eta : CUDART_INF_F, phi);
                    }
                }
                if (HAS_EL) {
                    const uint32_t a = a_ept + 4u * (unsigned)kq0;
                    const uint32_t oe = out + 8u * (unsigned)nm;
                    constexpr int UNR_E = 4;
#pragma unroll
                    for (int k = 0; k < UNR_E; ++k)
                        if (k < nq) {
                            const float pt = lds_f32(a + 4u * k), eta = lds_f32(a + es + 4u * k), phi = lds_f32(a + 2 * es + 4u * k);
                            sts_v2(oe + 8u * k, pt > lep_pt_min ? eta : CUDART_INF_F, phi);
                        }
#pragma unroll 1
                    for (int k = UNR_E; k < nq; ++k) {
                        const float pt = lds_f32(a + 4u * k), eta = lds_f32(a + es + 4u * k), phi = lds_f32(a + 2 * es + 4u * k);
                        sts_v2(oe + 8u * k, pt > lep_pt_min ? eta : CUDART_INF_F, phi);
                    }
                }
                if (c & 1) sts_v2(out + 8u * (unsigned)c, CUDART_INF_F, 0.0f);     // pad entry
                // [profile phase: phase 0: permutation]
                __syncwarp();       // bucket totals complete
                const int4 t0 = lds_v4i(bk), t1 = lds_v4i(bk + 16);
                int base = 0;
                base += key > 0 ? t0.x : 0; base += key > 1 ? t0.y : 0; base += key > 2 ? t0.z : 0; base += key > 3 ? t0.w : 0;
                base += key > 4 ? t1.x : 0; base += key > 5 ? t1.y : 0; base += key > 6 ? t1.z : 0;
                {
                    // per jet: byte offset in its column [10:0], byte offset [23:11] and byte length [31:24] of the list
                    unsigned int word = (unsigned)(kj0 << 2) | ((unsigned)l0 << 14) | ((unsigned)npair << 28);
                    const uint32_t a0 = order_a + 4u * (unsigned)(base + pos);
                    uint32_t a = a0;
                    const uint32_t aend = a + 4u * (unsigned)(nj < TAIL_CUT ? nj : TAIL_CUT);
                    const unsigned int word0 = word;
                    if ((aend - a) & 4u) { sts_u32(a, word); a += 4; word += 4; }       // odd count: one word first, then pairs
#pragma unroll 1
                    for (; a != aend; a += 8, word += 8) { sts_u32(a, word); sts_u32(a + 4, word + 4); }
                    // long events: the rest of their words, one per lane
                    for (unsigned lm = longm; lm; lm &= lm - 1) {
                        const int src = __ffs(lm) - 1;
                        const uint32_t as = __shfl_sync(0xffffffffu, a0, src);
                        const unsigned int ws = __shfl_sync(0xffffffffu, word0, src);
                        const int ns = __shfl_sync(0xffffffffu, nj, src);
                        for (int k = TAIL_CUT + lane; k < ns; k += 32) sts_u32(as + 4u * (unsigned)k, ws + 4u * (unsigned)k);
                    }
                }
                __syncwarp();

                // [profile phase: phase 1: dR and cuts (lane = jet)]
                // ---- phase 1: one lane per jet, in bucket order (neighbouring lanes: same lepton count)
                const uint32_t aend1 = order_a + 4u * (unsigned)njt;
#pragma unroll 1
                // the column bases are uniform registers (they derive from warp reductions), so a jet's three loads and
                // its store address as [offset + uniform base] without any per-jet address arithmetic
                const uint32_t u_jpt = __reduce_min_sync(0xffffffffu, a_jpt), u_jeta = __reduce_min_sync(0xffffffffu, a_jpt + js),
                               u_jphi = __reduce_min_sync(0xffffffffu, a_jpt + 2 * js);
                for (uint32_t ao = order_a + 4u * lane; ao < aend1; ao += 128) {
                    const unsigned int word = lds_u32(ao);
                    const uint32_t oj = word & 0x7ffu;
                    const uint32_t aj = u_jpt + oj;
                    const float pt = lds_f32(u_jpt + oj), eta = lds_f32(u_jeta + oj), phi = lds_f32(u_jphi + oj);
                    uint32_t al = (word >> 11) & 0x1fffu;
                    const uint32_t alend = al + (word >> 24);
                    float dmin = CUDART_INF_F;
#pragma unroll 1
                    for (; al != alend; al += 16) {
                        const float4 l = lds_v4(lep_a + al);
                        dmin = fminf(dmin, fminf(dr2_packed(make_float2(eta, phi), make_float2(l.x, l.y)),
                                                 dr2_packed(make_float2(eta, phi), make_float2(l.z, l.w))));
                    }
                    if (!CALIB) {
                        // pt if (pt > pt_min && |eta| < eta_max && !(dmin < dr2_max)) else -inf: one chained predicate
                        float r;
                        asm("{\n\t"
                            ".reg .pred p;\n\t"
                            ".reg .f32 ae;\n\t"
                            "abs.f32 ae, %2;\n\t"
                            "setp.gt.f32 p, %1, %4;\n\t"
                            "setp.lt.and.f32 p, ae, %5, p;\n\t"
                            "setp.geu.and.f32 p, %3, %6, p;\n\t"
                            "selp.f32 %0, %1, 0fFF800000, p;\n\t"
                            "}"
                            : "=f"(r)
                            : "f"(pt), "f"(eta), "f"(dmin), "f"(P.jet_pt_min), "f"(P.jet_abs_eta_max), "f"(P.dr2_max));
                        sts_f32(aj, r);
                    } else {
                        const bool base_ok = (fabsf(eta) < P.jet_abs_eta_max) && !(dmin < P.dr2_max);
                        const int bx = find_bin_fast(pt, smem_u32(S.cal_pt_edges), P.cal_npt, smem_u32(S.cal_axis));
                        const int by = find_bin_fast(eta, smem_u32(S.cal_eta_edges), P.cal_neta, smem_u32(S.cal_axis) + 16u);
                        sts_f32(aj + d_corr0, lds_f32(smem_u32(S.cal_table) + 4u * (unsigned)(bx * P.cal_neta + by)));
                        if (!base_ok) sts_f32(aj, CUDART_NAN_F);
                    }
                }
                __syncwarp();
                // [profile phase: jet mask output]
                if (P.out_jet_mask) {
                    // clean-jet mask, jets in their original order (coalesced bytes), from the verdicts just stored
                    const long long lj0 = __ldg(P.off[0] + e0) - P.jbase;
                    for (int j = lane; j < njt; j += 32) {
                        const float p = lds_f32(a_jpt + 4u * (unsigned)j);
                        if (!CALIB) {
                            P.out_jet_mask[lj0 + j] = (p > -CUDART_INF_F) ? 1 : 0;
                        } else {
                            const float cf = lds_f32(a_jpt + d_corr0 + 4u * (unsigned)j);
                            for (int v = 0; v < V; ++v)      // p is NaN when the jet failed eta / dR
                                P.out_jet_mask[(long long)v * P.jn + lj0 + j] =
                                    (__fmul_rn(p, __fmul_rn(cf, P.scales[v])) > P.jet_pt_min) ? 1 : 0;
                        }
                    }
                }

                // [profile phase: phase 2: per-event reductions (lane = event)]
                // ---- phase 2: one lane per event (lanes past the last event run with nj = 0)
                const uint32_t a_ev = a_jpt + 4u * (unsigned)kj0;
                const uint32_t d_corr = d_corr0;
                for (int v = 0; v < V; ++v) {
                    const float sv = P.scales[v];
                    EventAcc a;
                    a.init();
                    {
                        // two jets per iteration (an odd count takes one jet first)
                        uint32_t ap = a_ev;
                        const int nmain = nj < TAIL_CUT ? nj : TAIL_CUT;
                        int k = 0;
                        auto value = [&](uint32_t at) {
                            float p = lds_f32(at);
                            if (CALIB) p = __fmul_rn(p, __fmul_rn(lds_f32(at + d_corr), sv));     // NaN when the jet failed eta / dR
                            return p;
                        };
                        constexpr bool NEED_MIN = (FEAT < 0) || ((FEAT & (int)(F_MINPT | (F_OBS0 << HEPK_OBS_MINPT))) != 0);
                        if (nmain & 1) {
                            a.template push_lean<NEED_MIN>(value(ap), P.jet_pt_min, 0);
                            ap += 4;
                            k = 1;
                        }
#pragma unroll 1
                        for (; k != nmain; k += 2, ap += 8) {
                            const float p0 = value(ap), p1 = value(ap + 4);
                            a.template push_lean<NEED_MIN>(p0, P.jet_pt_min, k);
                            a.template push_lean<NEED_MIN>(p1, P.jet_pt_min, k + 1);
                        }
                    }
                    // long events: jets beyond TAIL_CUT, 32 at a time, one per lane, reduced over the warp and folded
                    // into the owner's state (their indices are larger than every index seen so far, and the two
                    // best are pushed in (value desc, index asc) order, so the first-index tie rule still holds)
                    for (unsigned lm = longm; lm; lm &= lm - 1) {
                        const int src = __ffs(lm) - 1;
                        const uint32_t as = __shfl_sync(0xffffffffu, a_ev, src);
                        const int ns = __shfl_sync(0xffffffffu, nj, src);
                        for (int kb = TAIL_CUT; kb < ns; kb += 32) {
                            const int k = kb + lane;
                            float p = -CUDART_INF_F;
                            if (k < ns) {
                                p = lds_f32(as + 4u * (unsigned)k);
                                if (CALIB) p = __fmul_rn(p, __fmul_rn(lds_f32(as + 4u * (unsigned)k + d_corr), sv));
                            }
                            const bool ok = p > P.jet_pt_min;
                            const unsigned okm = __ballot_sync(0xffffffffu, ok);
                            if (okm == 0u) continue;
                            double ps = ok ? (double)p : 0.0;
#pragma unroll
                            for (int o = 16; o >= 1; o >>= 1) ps += __shfl_xor_sync(0xffffffffu, ps, o);
                            const unsigned u = ok ? ord_key(p) : 0u;
                            const unsigned k1 = __reduce_max_sync(0xffffffffu, u);
                            const int j1 = __reduce_min_sync(0xffffffffu, u == k1 ? k : 0x7fffffff);
                            const unsigned u2 = k == j1 ? 0u : u;
                            const unsigned k2 = __reduce_max_sync(0xffffffffu, u2);
                            const int j2 = __reduce_min_sync(0xffffffffu, (u2 == k2 && u2 != 0u) ? k : 0x7fffffff);
                            const unsigned kmin = __reduce_min_sync(0xffffffffu, ok ? u : 0xffffffffu);
                            if (lane == src) {
                                a.cnt += __popc(okm);
                                a.sum += ps;
                                a.mn = fminf(a.mn, ord_value(kmin));
                                a.push_top(ord_value(k1), j1);
                                if (k2 != 0u) a.push_top(ord_value(k2), j2);
                            }
                        }
                    }
                    // [profile phase: phase 2: leading pair, release, next TMA issue]
                    float e1 = 0, p1 = 0, m1 = 0, e2 = 0, p2 = 0, m2 = 0;
                    if (a.i2 >= 0) {
                        const uint32_t x = a_ev + 4u * (unsigned)a.i1, y = a_ev + 4u * (unsigned)a.i2;
                        e1 = lds_f32(x + js); p1 = lds_f32(x + 2 * js); m1 = lds_f32(x + 3 * js);
                        e2 = lds_f32(y + js); p2 = lds_f32(y + 2 * js); m2 = lds_f32(y + 3 * js);
                    }
                    if (v == V - 1) {
                        // the staging region is dead from here: start the next tile's copies under the finishing math
                        fence_proxy_async_smem();
                        __syncwarp();
                        if (has_next) {
                            tile_counts(neo, nlo, ncnt);
                            fit = P.n_col > 0 && issue_tile<HAS_EL>(P, region_a, lane, nlo, ncnt);
                        }
                        released = true;
                    }
                    // [profile phase: finish_event call]
                    if (live)
                        finish_event<NW>(P, S, feat, e0 + lane, v, wt, evf, a.cnt, (float)a.sum, a.mn, a.b1, a.b2, a.i1, a.i2, e1, p1, m1, e2, p2, m2);
                }
            }
            bsel ^= 1;
        }
        // [profile phase: tile epilogue, overflow scan]
        if (!released) {
            fence_proxy_async_smem();
            __syncwarp();
            if (has_next) {
                tile_counts(neo, nlo, ncnt);
                fit = P.n_col > 0 && issue_tile<HAS_EL>(P, smem_u32(R), lane, nlo, ncnt);
            }
        }
        if (!staged && lane < ne) chain_event_global<CALIB>(P, smem_raw, e0 + lane);
        __syncwarp();
        eo = neo;
#pragma unroll
        for (int k = 0; k < 3; ++k) { lo[k] = nlo[k]; cnt[k] = ncnt[k]; }
        tile = tile_next;
        tile_next = take_tile();

        if (P.hist_acc) {
            // every finished tile checks one slice of the CTA's bins for values about to leave the int32 range
            const unsigned int t = ticket % SCAN_SLICES;      // tickets are consecutive: 32 finished tiles cover all slices
            const int n = P.obs_prefix[HEPK_N_OBS] * P.V * P.WS;
            const int len = (n + SCAN_SLICES - 1) / SCAN_SLICES;
            const int i0 = (int)t * len;
            flush_bins(P, S, i0, i0 + len < n ? i0 + len : n, lane, 32, false);
        }
    }
    // [profile phase: final flush]
    __syncthreads();
    if (P.hist_acc) flush_bins(P, S, 0, P.obs_prefix[HEPK_N_OBS] * P.V * P.WS, tid, nthr, true);
}

// Range of the launch's weights: max |w|, min non-zero |w| (bits of a non-negative float order like unsigned
// integers) and a flag for non-finite values, into the workspace header; the same for the event-weight table.
// The minima are kept as the COMPLEMENT of their bits and updated with atomicMax, so the caller's memset of the header to
// zero is the whole initialisation (0 = "no non-zero value seen").  w == nullptr: every weight is 1.
__global__ void chain_weight_range_kernel(const float* __restrict__ w, long long n, long long stride, int rows,
                                          const float* __restrict__ table, int nt, unsigned int* __restrict__ hdr)
{
    // p: `nrow` rows of `cnt` values, `rs` apart
    auto fold = [&](const float* p, long long cnt, long long rs, int nrow, int imax, int imin) {
        float m = 0.0f, mn = CUDART_INF_F;
        bool bad = false;
        auto take = [&](float x) {
            const float a = fabsf(x);
            bad = bad || !(a < CUDART_INF_F);
            m = fmaxf(m, a);
            if (a > 0.0f) mn = fminf(mn, a);
        };
        const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x, nt_ = (long long)gridDim.x * blockDim.x;
        for (int r = 0; r < nrow; ++r) {
            const float* q = p + r * rs;
            // 16-byte loads over the aligned body of the row, four in flight per thread; scalar head and tail
            const long long head = min((long long)((4 - ((reinterpret_cast<uintptr_t>(q) >> 2) & 3)) & 3), cnt);
            const long long n4 = (cnt - head) >> 2;
            const float4* q4 = reinterpret_cast<const float4*>(q + head);
            long long g = t0;
            for (; g + 3 * nt_ < n4; g += 4 * nt_) {
                const float4 a = __ldg(q4 + g), b = __ldg(q4 + g + nt_), c = __ldg(q4 + g + 2 * nt_), e = __ldg(q4 + g + 3 * nt_);
                take(a.x); take(a.y); take(a.z); take(a.w); take(b.x); take(b.y); take(b.z); take(b.w);
                take(c.x); take(c.y); take(c.z); take(c.w); take(e.x); take(e.y); take(e.z); take(e.w);
            }
            for (; g < n4; g += nt_) { const float4 a = __ldg(q4 + g); take(a.x); take(a.y); take(a.z); take(a.w); }
            for (long long i = t0; i < head; i += nt_) take(q[i]);
            for (long long i = head + 4 * n4 + t0; i < cnt; i += nt_) take(q[i]);
        }
        const unsigned int b = __reduce_max_sync(0xffffffffu, __float_as_uint(m));
        const unsigned int c = __reduce_min_sync(0xffffffffu, __float_as_uint(mn));
        if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(hdr + HDR_BAD, 1u);
        if ((threadIdx.x & 31) == 0) {
            if (b) atomicMax(hdr + imax, b);
            if (c != 0x7f800000u) atomicMax(hdr + imin, ~c);
        }
    };
    if (w) fold(w, n, stride, rows, HDR_WMAX, HDR_WMIN);
    else if (blockIdx.x == 0 && threadIdx.x == 0) { hdr[HDR_WMAX] = __float_as_uint(1.0f); hdr[HDR_WMIN] = ~__float_as_uint(1.0f); }
    if (table) fold(table, nt, nt, 1, HDR_TMAX, HDR_TMIN);
}

// The caller's arrays from the accumulators: word (v, o, slot, col) of the internal layout goes to
// sumw / sumw2 [v][o][w][slot] (float32(float64(old) + sum)) or counts [v][o][slot] (+=).
__global__ void chain_finalize_hist(const __grid_constant__ ChainParams P)
{
    float sc, sc2;
    hist_scales(P, sc, sc2);
    const int spv = P.obs_prefix[HEPK_N_OBS];
    const long long n = (long long)spv * P.V * P.WS;
    const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const int col = (int)(i % P.WS);
    const long long r = i / P.WS;                   // (v, o, slot) as v * spv + prefix[o] + slot
    const int v = (int)(r / spv), q = (int)(r % spv);
    int o = 0;
#pragma unroll
    for (int k = 1; k < HEPK_N_OBS; ++k)
        if (P.axis_edges[k] && q >= P.obs_prefix[k]) o = k;
    while (!P.axis_edges[o]) ++o;                   // the first active observable has prefix 0
    const int slot = q - P.obs_prefix[o], nb2 = P.axis_nbins[o] + 2;
    if (col == P.col_cnt) {
        P.hist_counts[r] += P.hist_acc[i];
        return;
    }
    if (col >= P.ncol) return;                      // padding column
    const bool sq = P.col_w2 >= 0 && col >= P.col_w2;
    if (sq && ((col - P.col_w2) & 1)) return;       // remainder column: handled with its value column
    if (!sq && !P.hist_sumw) return;                // sumw columns exist but only sumw2 was asked for
    const int w = sq ? (col - P.col_w2) >> 1 : col;
    float* dst = (sq ? P.hist_sumw2 : P.hist_sumw) + ((long long)v * spv + P.obs_prefix[o]) * P.W + (long long)w * nb2 + slot;
    const float s = sq ? sc2 : sc;
    double add;
    if (s == 0.0f) add = __longlong_as_double(P.hist_acc[i]);
    else if (sq) add = ((double)P.hist_acc[i] + (double)P.hist_acc[i + 1] * (1.0 / 1048576.0)) / (double)s;
    else add = (double)P.hist_acc[i] / (double)s;
    *dst = (float)((double)*dst + add);
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
    if (d->evw_table) {
        HEPK_REQUIRE(d->evw_x && d->evw_edges, "event-weight lookup: x or edges is NULL");
        HEPK_REQUIRE(d->evw_nbins >= 1 && d->evw_nbins <= 4096, "event-weight lookup: 1..4096 bins");
    }
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


// Internal histogram layout (ChainParams): columns of a slot row and the padded row length.
struct HistLayout { int ncol, ws, col_w2, col_cnt; long long n_words; };
static HistLayout hist_layout(const hepk_chain_desc* d)
{
    HistLayout h;
    const long long sp = hist_slots_per_variant(d);
    const int W = d->n_wvar;
    const bool w1 = d->hist_sumw != nullptr, w2 = d->hist_sumw2 != nullptr, cn = d->hist_counts != nullptr;
    h.ncol = 0; h.col_w2 = -1; h.col_cnt = -1;
    if (sp > 0 && (w1 || w2 || cn)) {
        h.ncol = (w1 || w2) ? W : 0;         // sumw columns are kept (unused) when only sumw2 is asked for
        if (w2) { h.col_w2 = h.ncol; h.ncol += 2 * W; }        // value and rounding-remainder column per weight
        if (cn) { h.col_cnt = h.ncol; h.ncol += 1; }
    }
    // an odd row length spreads the rows of a column over all shared-memory banks; pad when it costs little
    h.ws = h.ncol;
    if (h.ncol > 0 && (h.ncol & 1) == 0 && sp * d->n_variants * (h.ncol + 1) * 4 <= 32 * 1024) h.ws = h.ncol + 1;
    h.n_words = sp * d->n_variants * h.ws;
    return h;
}

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
    P.col_stride[0] = (cap_j + 8) * 4; P.col_stride[1] = (cap_m + 8) * 4; P.col_stride[2] = (cap_e + 8) * 4;
    // the jet permutation overlays the lepton column buffers: they are dead once the lepton list is built, and
    // the permutation is written after that and read until the region is released
    P.order_off = P.col_dst[4];
    if (o < (size_t)P.order_off + (size_t)cap_j * 4) o = (size_t)P.order_off + (size_t)cap_j * 4;
    P.lep_off = take((size_t)(cap_m + cap_e + LIST_PAD) * 8);
    P.corr_off = take(calib ? (size_t)(cap_j + 8) * 4 : 0);
    P.bucket_off = take(2 * N_BUCKETS * 4);
    return (int)dev::align_up(o, 128);
}

// plan_warps != nullptr: only work out the CTA shape (warps per SM; 0 = does not fit) and return.
static int32_t chain_launch(const hepk_chain_desc* d, void* workspace, cudaStream_t st, int* plan_warps, bool keep_weight_range = false)
{
    if (plan_warps) *plan_warps = 0;
    ChainParams P;
    memset(&P, 0, sizeof(P));
    P.n_events = d->n_events;
    P.n_tiles = (d->n_events + TILE_EVENTS - 1) / TILE_EVENTS;
    if (P.n_tiles >= (1ll << 31)) {          // the kernel indexes tiles with 32 bits (the offsets alone would be > 500 GB)
        if (plan_warps) return HEPK_OK;
        set_error("hepk_analysis_chain: n_events = %lld is beyond the 2^36 a launch supports", (long long)d->n_events);
        return HEPK_ERR_UNSUPPORTED;
    }
    P.w_stride = d->weights_stride > 0 ? d->weights_stride : d->n_events;
    P.out_stride = d->out_stride > 0 ? d->out_stride : d->n_events;
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
    const HistLayout hl = hist_layout(d);
    const bool want_hist = hl.ncol > 0;
    P.WS = hl.ws; P.ncol = hl.ncol; P.col_w2 = hl.col_w2; P.col_cnt = hl.col_cnt;
    const long long n_words = hl.n_words;
    P.hist_hdr = want_hist ? (unsigned int*)workspace : nullptr;
    P.hist_acc = want_hist ? (long long*)((char*)workspace + HDR_WORDS * 4) : nullptr;
    P.hist_sumw = want_hist ? d->hist_sumw : nullptr;
    P.hist_sumw2 = want_hist ? d->hist_sumw2 : nullptr;
    P.hist_counts = want_hist ? (long long*)d->hist_counts : nullptr;
    P.evw_x = d->evw_x; P.evw_edges = d->evw_edges; P.evw_table = d->evw_table; P.evw_nbins = d->evw_nbins;

    // staging capacities per 32-event tile from the mean multiplicities: mean + k sigma of a Poisson-like tile total
    // (a tile that does not fit takes the per-event path).  Leptons: k = 4.  Jets: k = 8, because jet multiplicities
    // have tails (BASELINE.json configs 2-4: 1 % of the events carry 30-40 jets), a tile that overflows contains
    // several such events, and on the per-event path one of them holds its warp for ~100 us: measured as a straggler
    // SM 12-18 % behind the rest at the end of a launch.
    const double nev = (double)(d->n_events > 0 ? d->n_events : 1);
    auto cap_for = [&](double mean, int floor_, double k) {
        const double t = TILE_EVENTS * mean;
        long long c = (long long)(t + k * sqrt(2.0 * t + 1.0)) + 8;
        return c < floor_ ? floor_ : (int)c;
    };
    const int cap_j4 = round_up4(cap_for((double)d->jets.n_objects / nev, 64, 4.0));
    int cap_j = round_up4(d->tune_cap_jets > 0 ? d->tune_cap_jets : cap_for((double)d->jets.n_objects / nev, 64, 8.0));
    int cap_m = round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons : cap_for((double)d->muons.n_objects / nev, 32, 4.0));
    int cap_e = has_el ? round_up4(d->tune_cap_leptons > 0 ? d->tune_cap_leptons
                                                              : cap_for((double)d->electrons.n_objects / nev, 32, 4.0)) : 0;
    if (cap_j < 16) cap_j = 16;
    if (cap_j > MAX_JETS_TILE) cap_j = MAX_JETS_TILE;      // the jet's byte offset is packed in 11 bits
    if (cap_m < 4) cap_m = 4;
    if (has_el && cap_e < 4) cap_e = 4;
    if (cap_m > 492) cap_m = 492;        // the list start (in bytes) is packed in 13 bits
    if (cap_e > 492) cap_e = 492;        // 2 * 492 + LIST_PAD <= MAX_LIST, multiple of 4

    const int smem_max = max_smem_optin();
    const int shared_bytes = (int)dev::chain_shared_layout(P, calib, nullptr, nullptr);
    if (shared_bytes + 1024 > smem_max) {
        if (plan_warps) return HEPK_OK;
        set_error("hepk_analysis_chain: histograms need %d bytes of shared memory (max %d)", shared_bytes, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    int region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
    // large histogram sets leave room for few warps: below 16 per SM the warps matter more than the rare overflowing
    // tile, and the jet buffers go back to 4 sigma
    if (d->tune_cap_jets <= 0 && (smem_max - shared_bytes) / region < 16 && cap_j > cap_j4) {
        cap_j = cap_j4;
        region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
    }
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
        if (plan_warps) return HEPK_OK;
        set_error("hepk_analysis_chain: %d + %d bytes of shared memory needed (max %d)", shared_bytes, region, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    P.shared_bytes = shared_bytes;
    P.region_bytes = region;
    // the kernel addresses the columns of a collection at a fixed stride from the first one, which needs them to
    // share their alignment modulo 16 bytes; otherwise every tile takes the per-event path
    P.n_col = NCOL;
    for (int c = 0; c < NCOL; ++c) {
        const int first = P.col_coll[c] == 0 ? 0 : (P.col_coll[c] == 1 ? 4 : 7);
        if (P.col_ptr[c] && P.col_ptr[first] && P.col_mis[c] != P.col_mis[first]) P.n_col = 0;
    }
    // the staged path indexes with 32-bit object counts
    const long long big = 0x7fffffffll - 64;
    if (d->jets.n_objects > big || d->muons.n_objects > big || (has_el && d->electrons.n_objects > big)) P.n_col = 0;
    P.col_n32[0] = (int)(d->jets.n_objects > big ? big : d->jets.n_objects);
    P.col_n32[1] = (int)(d->muons.n_objects > big ? big : d->muons.n_objects);
    P.col_n32[2] = has_el ? (int)(d->electrons.n_objects > big ? big : d->electrons.n_objects) : 0;

    // CTA shape: as many warps per SM as shared memory allows (up to 20), in as few CTAs as possible so that
    // the privatised histograms are shared by many warps
    const int sm_total = smem_max + 1024;              // per SM; each CTA also pays 1 KB of system shared memory
    int best_ctas = 1, best_wpc = 1, best_total = 0;
    const int max_warps_sm = d->tune_warps_per_sm > 0 ? d->tune_warps_per_sm : 20;
    for (int ctas = 1; ctas <= 4; ++ctas) {
        if (d->tune_ctas_per_sm > 0 && ctas != d->tune_ctas_per_sm && !(ctas == 1 && d->tune_ctas_per_sm > 4)) continue;
        int budget = sm_total / ctas - 1024;
        if (budget > smem_max) budget = smem_max;
        int wpc = (budget - shared_bytes) / region;
        if (wpc > 24) wpc = 24;
        if (wpc * ctas > max_warps_sm) wpc = max_warps_sm / ctas;
        if (d->tune_warps_per_cta > 0 && wpc > d->tune_warps_per_cta) wpc = d->tune_warps_per_cta;
        if (wpc < 1) continue;
        if (wpc * ctas > best_total) { best_total = wpc * ctas; best_ctas = ctas; best_wpc = wpc; }
    }
    const int wpc = best_wpc;
    if (plan_warps) {
        *plan_warps = best_total;
        return HEPK_OK;
    }
    // Shared memory the chosen shape leaves unused also goes to the jet buffers (fewer overflowing tiles still).
    if (d->tune_cap_jets <= 0) {
        int budget = sm_total / best_ctas - 1024;
        if (budget > smem_max) budget = smem_max;
        while (cap_j + 4 <= MAX_JETS_TILE && cap_j + 4 <= 2 * cap_j4) {
            const int r = chain_region_layout(P, d, calib, cap_j + 4, cap_m, cap_e);
            if (shared_bytes + wpc * r > budget) break;
            cap_j += 4;
        }
        region = chain_region_layout(P, d, calib, cap_j, cap_m, cap_e);
        P.region_bytes = region;
    }
    const size_t smem = (size_t)shared_bytes + (size_t)wpc * region;
    P.tile_counter = want_hist ? P.hist_hdr + HDR_TILE : nullptr;

    // two register budgets: up to 20 warps per CTA (96 registers per thread, no spills) or up to 24 (80)
    void (*kern)(ChainParams);
#define HEPK_PICK(MAXT, FEAT)                                                                                        \
    (calib ? (has_el ? dev::chain_kernel<true, true, MAXT, FEAT> : dev::chain_kernel<true, false, MAXT, FEAT>)     \
           : (has_el ? dev::chain_kernel<false, true, MAXT, FEAT> : dev::chain_kernel<false, false, MAXT, FEAT>))
    // the common analysis shape (njet, argmax, ht, maxpt, mjj per event; HT and leading-pt histograms with counts and
    // one weight column) has a build with its feature word as a compile-time constant
    constexpr int FEAT_COMMON = (int)(dev::F_NJET | dev::F_ARGMAX | dev::F_HT | dev::F_MAXPT | dev::F_MJJ |
                                      (dev::F_OBS0 << HEPK_OBS_HT) | (dev::F_OBS0 << HEPK_OBS_MAXPT) | dev::F_COUNTS |
                                      dev::F_SUMW | dev::F_WEIGHTS);
    unsigned feat_host = 0;
    if (d->out_njet) feat_host |= dev::F_NJET;
    if (d->out_argmax) feat_host |= dev::F_ARGMAX;
    if (d->out_ht) feat_host |= dev::F_HT;
    if (d->out_maxpt) feat_host |= dev::F_MAXPT;
    if (d->out_minpt) feat_host |= dev::F_MINPT;
    if (d->out_mjj) feat_host |= dev::F_MJJ;
    if (d->out_subpt) feat_host |= dev::F_SUBPT;
    for (int o = 0; o < HEPK_N_OBS; ++o)
        if (d->axis_edges[o]) feat_host |= dev::F_OBS0 << o;
    if (P.col_cnt >= 0) feat_host |= dev::F_COUNTS;
    if (P.hist_acc && P.hist_sumw) feat_host |= dev::F_SUMW;
    if (P.col_w2 >= 0) feat_host |= dev::F_SUMW2;
    if (P.evw_table) feat_host |= dev::F_EVW;
    if (d->weights) feat_host |= dev::F_WEIGHTS;
    if (P.W > 1) feat_host |= dev::F_MULTIW;
    const bool common = (int)feat_host == FEAT_COMMON && !d->out_jet_mask && has_el && !d->tune_generic_build;
#define HEPK_PICK_COMMON(MAXT) (calib ? dev::chain_kernel<true, true, MAXT, FEAT_COMMON> : dev::chain_kernel<false, true, MAXT, FEAT_COMMON>)
    // several weight columns and few warps (large histograms): a build that keeps the event's weights in registers
    const bool multiw = P.W > 1 && d->weights && wpc <= 16;
    // The histograms-only shape (the paper's own output: all six observables, counts and weighted sums
    // over several weight columns, no per-event arrays) also has its feature word fixed at compile time: the generic
    // build is ~13,000 instructions of which such a launch executes ~4,000, scattered among the rest, and it spent
    // more time waiting for instruction fetches than for anything else (profiles/r02: stall `no_instruction`).
    constexpr int FEAT_HISTS = (int)((dev::F_OBS0 * 63u) | dev::F_COUNTS | dev::F_SUMW | dev::F_WEIGHTS | dev::F_MULTIW);
    const bool hists_shape = multiw && (int)feat_host == FEAT_HISTS && !d->out_jet_mask && has_el && !d->tune_generic_build;
    if (hists_shape)
        kern = calib ? dev::chain_kernel<true, true, 512, FEAT_HISTS, HEPK_MAX_WVAR> : dev::chain_kernel<false, true, 512, FEAT_HISTS, HEPK_MAX_WVAR>;
    else if (multiw)
        kern = calib ? (has_el ? dev::chain_kernel<true, true, 512, -1, HEPK_MAX_WVAR> : dev::chain_kernel<true, false, 512, -1, HEPK_MAX_WVAR>)
                     : (has_el ? dev::chain_kernel<false, true, 512, -1, HEPK_MAX_WVAR> : dev::chain_kernel<false, false, 512, -1, HEPK_MAX_WVAR>);
    else if (wpc <= 20) kern = common ? HEPK_PICK_COMMON(640) : HEPK_PICK(640, -1);
    else kern = common ? HEPK_PICK_COMMON(768) : HEPK_PICK(768, -1);
#undef HEPK_PICK_COMMON
#undef HEPK_PICK
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    HEPK_CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, wpc * 32, smem));
    if (occ < 1) occ = 1;
    if (occ > best_ctas) occ = best_ctas;
    long long grid = (long long)sm_count() * occ;
    const long long need = (P.n_tiles + wpc - 1) / wpc;
    if (grid > need) grid = need;
    if (grid < 1) grid = 1;

    if (want_hist && keep_weight_range) {
        // a later group of variants of the same call: the weights (and their range in the header) are the same
        HEPK_CUDA_TRY(cudaMemsetAsync(P.hist_hdr + HDR_TILE, 0, 4, st));
        HEPK_CUDA_TRY(cudaMemsetAsync(P.hist_acc, 0, (size_t)n_words * 8, st));
    } else if (want_hist) {
        HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, HDR_WORDS * 4 + (size_t)n_words * 8, st));
        const long long nw = (long long)P.W * P.n_events;
        long long blocks = (nw + 256 * 8 - 1) / (256 * 8);
        if (blocks > 4 * sm_count()) blocks = 4 * sm_count();
        if (blocks < 1) blocks = 1;
        dev::chain_weight_range_kernel<<<(unsigned)blocks, 256, 0, st>>>(d->weights, P.n_events, P.w_stride, P.W, d->evw_table,
                                                                         d->evw_nbins, P.hist_hdr); count_launch();
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    profile_mark(st, 0);
    kern<<<(unsigned)grid, wpc * 32, smem, st>>>(P); count_launch();
    profile_mark(st, 1);
    HEPK_CUDA_TRY(cudaGetLastError());
    if (want_hist) {
        dev::chain_finalize_hist<<<(unsigned)((n_words + 255) / 256), 256, 0, st>>>(P); count_launch();
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    return HEPK_OK;
}

}  // namespace hepk

extern "C" size_t hepk_chain_workspace_bytes(const hepk_chain_desc* d)
{
    if (!d || d->n_variants < 1 || d->n_wvar < 1) return 0;
    return hepk::HDR_WORDS * 4 + (size_t)hepk::hist_layout(d).n_words * 8 + 8;      // header + 64-bit accumulators
}

extern "C" int32_t hepk_analysis_chain(const hepk_chain_desc* d, void* workspace, size_t workspace_bytes, void* stream)
{
    using namespace hepk;
    const int32_t rc = chain_validate(d);
    if (rc != HEPK_OK) return rc;
    if (d->n_events == 0) return HEPK_OK;
    if (hist_layout(d).ncol > 0) {
        HEPK_REQUIRE(workspace != nullptr, "workspace is NULL");
        HEPK_REQUIRE(workspace_bytes >= hepk_chain_workspace_bytes(d), "workspace too small");
    }
    // Variants are independent given the variant-independent first half of the chain, and the privatised histograms
    // of all variants share the SM's shared memory with the warps' staging regions.  When they leave room for fewer
    // than 12 warps (large histogram sets), or do not fit at all, the variants are run in groups, one launch per
    // group: the first half is recomputed per group, which costs less than running at a fraction of the occupancy.
    const int V = d->n_variants;
    int group = V;
    if (d->tune_variants_per_pass > 0) group = d->tune_variants_per_pass < V ? d->tune_variants_per_pass : V;
    else if (V > 1 && hist_layout(d).ncol > 0) {
        int best_g = 0, best_w = 0;
        for (int g = V; g >= 1; --g) {
            hepk_chain_desc t = *d;
            t.n_variants = g;
            int w = 0;
            if (chain_launch(&t, workspace, nullptr, &w) != HEPK_OK) w = 0;
            if (w >= 12) { best_g = g; best_w = w; break; }
            if (w > best_w) { best_g = g; best_w = w; }
        }
        if (best_g == 0) best_g = V;         // nothing fits: let the launch report the error
        group = best_g;
    }
    if (group >= V) return chain_launch(d, workspace, (cudaStream_t)stream, nullptr);
    const long long spv = hist_slots_per_variant(d), N = d->out_stride > 0 ? d->out_stride : d->n_events, W = d->n_wvar;
    for (int v0 = 0; v0 < V; v0 += group) {
        hepk_chain_desc t = *d;
        t.n_variants = v0 + group <= V ? group : V - v0;
        for (int v = 0; v < t.n_variants; ++v) t.calib_scales[v] = d->calib_scales[v0 + v];
        if (t.out_njet) t.out_njet += v0 * N;
        if (t.out_argmax) t.out_argmax += v0 * N;
        if (t.out_ht) t.out_ht += v0 * N;
        if (t.out_maxpt) t.out_maxpt += v0 * N;
        if (t.out_minpt) t.out_minpt += v0 * N;
        if (t.out_mjj) t.out_mjj += v0 * N;
        if (t.out_subpt) t.out_subpt += v0 * N;
        if (t.out_jet_mask) t.out_jet_mask += v0 * d->jets.n_objects;
        if (t.hist_sumw) t.hist_sumw += v0 * spv * W;
        if (t.hist_sumw2) t.hist_sumw2 += v0 * spv * W;
        if (t.hist_counts) t.hist_counts += v0 * spv;
        const int32_t r = chain_launch(&t, workspace, (cudaStream_t)stream, nullptr, v0 > 0);
        if (r != HEPK_OK) return r;
    }
    return HEPK_OK;
}
