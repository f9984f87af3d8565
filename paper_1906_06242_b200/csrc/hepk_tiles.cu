// hepk_tiles.cu — the per-event single kernels that walk jagged collections (include/hepk.h):
//   hepk_segmented_reduce_{sum,max,min,count,argmax} (variant 2, "block-per-tile"), hepk_deltar_mask, hepk_pair_invmass,
//   hepk_select_opposite_sign.
//
// One streaming skeleton serves them all.  A CTA is a handful of AUTONOMOUS warps; a warp owns a double-buffered
// staging region of shared memory with one mbarrier per buffer and streams tiles of 32 x H events through it (a lane
// owns H consecutive events; H is 4 for the light reductions, whose cost per tile is mostly the tile's own
// bookkeeping, and 1 otherwise):
//   * the offsets of a tile are read one tile ahead (H + 1 consecutive entries per lane) and reduced over the warp
//     (REDUX: the slice bounds come back in uniform registers);
//   * one elected lane issues one 1-D bulk copy (cp.async.bulk, SASS UBLKCP) per column for the tile's slice, 16-byte
//     aligned on both sides by starting at the aligned element below the slice; the consumer adds the same shift;
//   * while those bytes fly, the warp works on the tile that landed before: there is no CTA-wide barrier after the
//     set-up, and every input byte is read from HBM once.
// The buffers have a fixed capacity; a launch whose collections are dense enough to overflow them with 32 lanes per tile
// takes 16, 8, ... lanes per tile instead (decided on the device from offsets[n_events], so no call ever waits for a
// read-back).  A tile whose slices still do not fit (giant events), or cannot be aligned at the very ends of the
// arrays, goes a warp-per-event way straight from global memory (same arithmetic, same results).
#include <math.h>
#include <string.h>

#include <type_traits>

#include "hepk_common.cuh"

namespace hepk {

constexpr int WT_EVENTS = 32;      // events per warp tile and event-per-lane, at most
constexpr int WT_MAX_COL = 6;      // staged columns per tile

// Staged columns come in four classes: float32 / uint8 columns of collection 0, then of collection 1.  The columns of
// a class must share their alignment modulo 16 bytes (else the launch takes the global path), so one slice geometry
// per class serves all of them.  How many columns each class has is a compile-time property of the kernel (Shape).
struct TileParams {
    long long n_events;
    const long long* off[2];
    long long base[2];
    int cap[2];                    // slice capacity per collection, in objects
    int staged;                    // 0: every tile takes the global path
    const char* ptr[WT_MAX_COL];   // element 0 of each column (content index 0), classes in order
    int dst[WT_MAX_COL];           // byte offset of each column's buffer inside a stage
    int mis[4];                    // per class: (address / element size) mod (16 / element size)
    int stage_bytes;               // one stage: mbarrier at +0, column buffers from +16
    int extra_off, warp_bytes;     // per-warp scratch after the two stages; bytes per warp
};

template <int H_, int NC_, int NF0_, int NB0_, int NF1_ = 0, int NB1_ = 0>
struct TileShape {
    static constexpr int H = H_;         // consecutive events per lane
    static constexpr int NC = NC_;
    static constexpr int NCOL = NF0_ + NB0_ + NF1_ + NB1_;
    static constexpr int NCA = NCOL > 0 ? NCOL : 1;      // length of the address array handed to the op
    __host__ __device__ static constexpr int count(int q) { return q == 0 ? NF0_ : (q == 1 ? NB0_ : (q == 2 ? NF1_ : NB1_)); }
    __host__ __device__ static constexpr int first(int q) { return q == 0 ? 0 : (q == 1 ? NF0_ : (q == 2 ? NF0_ + NB0_ : NF0_ + NB0_ + NF1_)); }
};

namespace dev {

__device__ __forceinline__ bool elect_one_lane()
{
    unsigned int pred;
    asm volatile("{\n\t.reg .pred p;\n\telect.sync _|p, 0xffffffff;\n\tselp.u32 %0, 1, 0, p;\n\t}" : "=r"(pred));
    return pred != 0u;
}
__device__ __forceinline__ float lds_f(uint32_t a)
{
    float r;
    asm volatile("ld.shared.f32 %0, [%1];" : "=f"(r) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ unsigned int lds_b(uint32_t a)
{
    unsigned int r;
    asm volatile("ld.shared.u8 %0, [%1];" : "=r"(r) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ unsigned int lds_w(uint32_t a)
{
    unsigned int r;
    asm volatile("ld.shared.u32 %0, [%1];" : "=r"(r) : "r"(a) : "memory");
    return r;
}
__device__ __forceinline__ void sts_b(uint32_t a, unsigned int v) { asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts_w(uint32_t a, unsigned int v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }

// Offsets of the lane's H events of tile `tile` (low words; differences inside a tile are exact): o[c][h] = offsets
// of event lane * H + h of the tile, h = 0 .. H.  Events past the tile's last one repeat its end offset (empty events).
template <int NC, int H>
__device__ __forceinline__ void tile_load_offsets(const TileParams& P, unsigned int tile, int evt, int lane, int (&o)[NC][H + 1])
{
    const long long t0 = (long long)tile * evt;
    int lim = evt;
    if (t0 + evt > P.n_events) lim = (int)(P.n_events - t0);       // only the last tile can be ragged (uniform branch)
#pragma unroll
    for (int h = 0; h <= H; ++h) {
        const int d = lane * H + h < lim ? lane * H + h : lim;
#pragma unroll
        for (int c = 0; c < NC; ++c) o[c][h] = (int)__ldg(P.off[c] + t0 + d);
    }
}

// Slice bounds of the tile (uniform) and the bulk copies of its columns into the stage at shared address `stage_a`.
// Returns false (nothing issued) when a slice does not fit.  Called by all 32 lanes, converged.
template <class SH>
__device__ __forceinline__ bool tile_issue(const TileParams& P, const int (&n_obj)[SH::NC], uint32_t stage_a,
                                           const int (&o)[SH::NC][SH::H + 1], int (&lo)[SH::NC], int (&cnt)[SH::NC])
{
#pragma unroll
    for (int c = 0; c < SH::NC; ++c) {        // offsets do not decrease: lane 0 holds the smallest start, lane 31 the largest end
        lo[c] = __reduce_min_sync(0xffffffffu, o[c][0]);
        cnt[c] = __reduce_max_sync(0xffffffffu, o[c][SH::H]) - lo[c];
    }
    // Per class: the slice [l0, l0 + n) sits in the window [A, A + len) whose ends are 16-byte aligned in memory; the
    // part [bA, bB) of the window that lies inside the array goes by bulk copy.  Only at the very ends of an array can
    // bA > A or bB < A + len; the few elements of the slice outside [bA, bB) are then moved by ordinary loads.
    int bad = 0, edge = 0;
    int A[4], bA[4], bB[4];
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        A[q] = bA[q] = bB[q] = 0;
        if (SH::count(q) == 0) continue;
        const int c = q >> 1;
        const int per16 = (q & 1) ? 16 : 4;
        const int l0 = (int)((unsigned)lo[c] - (unsigned)P.base[c]);
        const int sh = (l0 + P.mis[q]) & (per16 - 1);
        const int n = cnt[c];
        const int len = n != 0 ? (n + sh + per16 - 1) & ~(per16 - 1) : 0;
        A[q] = n != 0 ? l0 - sh : 0;
        bA[q] = A[q];
        bB[q] = A[q] + len;
        // fits: 0 <= n <= capacity, and the slice lies inside the collection (sign bits, no branches)
        bad |= n | (P.cap[c] - n) | l0 | (n_obj[c] - l0 - n);
        edge |= A[q] | (n_obj[c] - bB[q]);          // negative: the window reaches past an end of the array
    }
    if (bad < 0) return false;
    if (edge < 0) {          // (uniform, rare) clip the bulk windows to the array; slice elements outside them by ordinary loads
        const int lane = (int)(threadIdx.x & 31u);
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            if (SH::count(q) == 0) continue;
            const int c = q >> 1;
            const int per16 = (q & 1) ? 16 : 4, es = (q & 1) ? 1 : 4;
            const int l0 = (int)((unsigned)lo[c] - (unsigned)P.base[c]);
            if (A[q] < 0) bA[q] = A[q] + per16;
            if (bB[q] > n_obj[c]) bB[q] = A[q] + ((n_obj[c] - A[q]) & ~(per16 - 1));
            if (bB[q] < bA[q]) bB[q] = bA[q];
            for (int j = lane; j < cnt[c]; j += 32) {
                const int g = l0 + j;
                if (g >= bA[q] && g < bB[q]) continue;
#pragma unroll
                for (int i = 0; i < SH::count(q); ++i) {
                    const int k = SH::first(q) + i;
                    const uint32_t d = stage_a + (uint32_t)P.dst[k] + (uint32_t)((g - A[q]) * es);
                    if (es == 4) sts_w(d, __ldg(reinterpret_cast<const unsigned int*>(P.ptr[k]) + g));
                    else sts_b(d, (unsigned int)__ldg(reinterpret_cast<const unsigned char*>(P.ptr[k]) + g));
                }
            }
        }
    }
    uint32_t total = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) total += (uint32_t)((bB[q] - bA[q]) * ((q & 1) ? 1 : 4) * SH::count(q));
    if (elect_one_lane()) {
        asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(stage_a), "r"(total) : "memory");
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            const int es = (q & 1) ? 1 : 4;
            if (SH::count(q) == 0 || bB[q] == bA[q]) continue;
#pragma unroll
            for (int j = 0; j < SH::count(q); ++j) {
                const int k = SH::first(q) + j;
                asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                                 stage_a + (uint32_t)P.dst[k] + (uint32_t)((bA[q] - A[q]) * es)),
                             "l"(P.ptr[k] + (long long)bA[q] * es), "r"((uint32_t)((bB[q] - bA[q]) * es)), "r"(stage_a)
                             : "memory");
            }
        }
    }
    return true;
}

// Shared addresses of tile-local element 0 of every column in the stage at `stage_a`.
template <class SH>
__device__ __forceinline__ void tile_col_addrs(const TileParams& P, uint32_t stage_a, const int (&lo)[SH::NC], uint32_t (&ca)[SH::NCA])
{
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        if (SH::count(q) == 0) continue;
        const int c = q >> 1;
        const int per16 = (q & 1) ? 16 : 4, es = (q & 1) ? 1 : 4;
        const int l0 = (int)((unsigned)lo[c] - (unsigned)P.base[c]);
        const uint32_t sh = (uint32_t)(((l0 + P.mis[q]) & (per16 - 1)) * es);
#pragma unroll
        for (int j = 0; j < SH::count(q); ++j) ca[SH::first(q) + j] = stage_a + (uint32_t)P.dst[SH::first(q) + j] + sh;
    }
    // pinned: the compiler would otherwise recompute these few adds from the parameters at every use inside the loops
#pragma unroll
    for (int k = 0; k < SH::NCOL; ++k) asm volatile("" : "+r"(ca[k]));
}

// The streaming loop.  Op provides
//   void staged(const TileParams&, const uint32_t (&ca)[NCOL], uint32_t extra_a, long long e0, int ne, int lane,
//               const int (&o)[NC][H + 1], const int (&lo)[NC], const int (&cnt)[NC]);
//   void global(const TileParams&, long long e0, int ne, int lane);
// e0: first event of the tile, ne: its events; event lane * H + h of the tile belongs to lane `lane`.
template <class SH, class Op>
__device__ __forceinline__ void tile_stream(const TileParams& P, Op& op)
{
    constexpr int NC = SH::NC, H = SH::H;
    extern __shared__ __align__(128) unsigned char smem_raw[];
    const int tid = threadIdx.x;
    const int warp = __reduce_min_sync(0xffffffffu, tid >> 5);      // uniform register
    const int lane = tid & 31, nwarp = blockDim.x >> 5;
    const uint32_t region_a = smem_u32(smem_raw) + (uint32_t)warp * (uint32_t)P.warp_bytes;
    const uint32_t extra_a = region_a + (uint32_t)P.extra_off;
    if (lane == 0) {
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(region_a));
        asm volatile("mbarrier.init.shared::cta.b64 [%0], 1;" ::"r"(region_a + (uint32_t)P.stage_bytes));
        fence_mbar_init();
    }
    __syncwarp();
    // events per tile: 32 lanes x H unless the collections are so dense that such a slice would overflow the buffers
    int n_obj[NC];
    int evt = WT_EVENTS * H;
    bool staged = P.staged != 0;
#pragma unroll
    for (int c = 0; c < NC; ++c) {
        const long long n = __ldg(P.off[c] + P.n_events) - P.base[c];
        if (n < 0 || n > 0x7fffffffll - 64) staged = false;          // the staging indexes with 32 bits
        n_obj[c] = staged ? (int)n : 0;
        const float mean = (float)n / (float)P.n_events;
        while (evt > H && (float)evt * mean + 4.0f * sqrtf(2.0f * (float)evt * mean + 1.0f) + 8.0f > (float)P.cap[c]) evt >>= 1;
    }
    const long long nt64 = (P.n_events + evt - 1) / evt;           // (the host refuses launches of 2^31 32-event tiles or more)
    const unsigned int NT = nt64 > 0xfffffff0ll ? 0xfffffff0u : (unsigned int)nt64;
    const unsigned int stride = gridDim.x * (unsigned)nwarp;
    unsigned int tile = blockIdx.x * (unsigned)nwarp + (unsigned)warp;
    if (tile >= NT) return;
    int o[NC][H + 1], lo[NC], cnt[NC];
    int po[NC][H + 1];                        // offsets of the next tile
    uint32_t parity = 0u;                     // bit s: phase of stage s's barrier
    uint32_t stage_a = region_a, other_a = region_a + (uint32_t)P.stage_bytes;
    tile_load_offsets<NC, H>(P, tile, evt, lane, o);
    bool fit = staged && tile_issue<SH>(P, n_obj, stage_a, o, lo, cnt);
    unsigned int next = tile + stride < NT && tile + stride > tile ? tile + stride : NT;
    if (next < NT) tile_load_offsets<NC, H>(P, next, evt, lane, po);
    while (true) {
        // the next tile's copies go into the other stage (its previous contents were consumed an iteration ago)
        int nlo[NC], ncnt[NC];
        bool nfit = false;
        unsigned int next2 = NT;
        int qo[NC][H + 1];
        if (next < NT) {
            fence_proxy_async_smem();
            __syncwarp();
            nfit = staged && tile_issue<SH>(P, n_obj, other_a, po, nlo, ncnt);
            next2 = next + stride < NT && next + stride > next ? next + stride : NT;
            if (next2 < NT) tile_load_offsets<NC, H>(P, next2, evt, lane, qo);
        }
        const long long e0 = (long long)tile * evt;
        const long long rest = P.n_events - e0;
        const int ne = rest < evt ? (int)rest : evt;
        if (fit) {
            const uint32_t ph = stage_a == region_a ? (parity & 1u) : (parity >> 1);
            asm volatile(
                "{\n"
                ".reg .pred p;\n"
                "WAIT_%=:\n"
                "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
                "@p bra DONE_%=;\n"
                "bra WAIT_%=;\n"
                "DONE_%=:\n"
                "}\n" ::"r"(stage_a), "r"(ph)
                : "memory");
            parity ^= stage_a == region_a ? 1u : 2u;
            uint32_t ca[SH::NCA];
            tile_col_addrs<SH>(P, stage_a, lo, ca);
            op.staged(P, ca, extra_a, e0, ne, lane, o, lo, cnt);
        } else {
            op.global(P, e0, ne, lane);
        }
        __syncwarp();
        if (next >= NT) break;
        tile = next; next = next2; fit = nfit;
        { const uint32_t t = stage_a; stage_a = other_a; other_a = t; }
#pragma unroll
        for (int c = 0; c < NC; ++c) {
            lo[c] = nlo[c]; cnt[c] = ncnt[c];
#pragma unroll
            for (int h = 0; h <= H; ++h) { o[c][h] = po[c][h]; po[c][h] = qo[c][h]; }
        }
    }
}

// =========================================================================================== segmented reductions
enum { OP_SUM = 0, OP_MAX = 1, OP_MIN = 2, OP_COUNT = 3, OP_ARGMAX = 4 };

template <int OP> struct RedOut { typedef float type; };
template <> struct RedOut<OP_COUNT> { typedef int type; };
template <> struct RedOut<OP_ARGMAX> { typedef int type; };

// Running state of one reduction (the oracle's update rules); merge() combines partial states so that count / max /
// min / argmax do not depend on the order of combination.  Sums accumulate in float64 and are rounded once.
template <int OP>
struct RedAcc {
    float v;
    double s;
    int i;
    __device__ __forceinline__ void init()
    {
        v = (OP == OP_MAX || OP == OP_ARGMAX) ? -CUDART_INF_F : (OP == OP_MIN ? CUDART_INF_F : 0.f);
        s = 0.0;
        i = OP == OP_ARGMAX ? -1 : 0;
    }
    // element k of the event, taken iff `take` (branch-free: the staged loop runs it predicated)
    __device__ __forceinline__ void push(float x, int k, bool take)
    {
        if (OP == OP_SUM) s += (double)(take ? x : 0.f);           // (+0.0 leaves any sum unchanged, -0.0 + 0.0 included: the sum starts at +0.0)
        else if (OP == OP_COUNT) i += take ? 1 : 0;
        else if (OP == OP_MAX) { if (take && x > v) v = x; }       // a NaN compares false: skipped
        else if (OP == OP_MIN) { if (take && x < v) v = x; }
        else { if (take && x == x && (i < 0 || x > v)) { v = x; i = k; } }     // k ascending within a thread (full rule)
    }
    // argmax only: the rule without its "the first non-NaN element is always taken" clause.  Starting from v = -inf it
    // differs from push() only when no element exceeds -inf; the caller then redoes the event with push().
    __device__ __forceinline__ void push_gt(float x, int k)
    {
        if (x > v) { v = x; i = k; }
    }
    __device__ __forceinline__ void merge(const RedAcc& o)
    {
        if (OP == OP_SUM) s += o.s;
        else if (OP == OP_COUNT) i += o.i;
        else if (OP == OP_MAX) { if (o.v > v) v = o.v; }
        else if (OP == OP_MIN) { if (o.v < v) v = o.v; }
        else { if (o.i >= 0 && (i < 0 || o.v > v || (o.v == v && o.i < i))) { v = o.v; i = o.i; } }
    }
    __device__ __forceinline__ typename RedOut<OP>::type result() const
    {
        if (OP == OP_COUNT || OP == OP_ARGMAX) return (typename RedOut<OP>::type)i;
        if (OP == OP_SUM) return (typename RedOut<OP>::type)(float)s;
        return (typename RedOut<OP>::type)v;
    }
    __device__ __forceinline__ void warp_reduce()
    {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            RedAcc o;
            o.v = __shfl_xor_sync(0xffffffffu, v, d);
            o.i = __shfl_xor_sync(0xffffffffu, i, d);
            o.s = OP == OP_SUM ? __shfl_xor_sync(0xffffffffu, s, d) : 0.0;
            merge(o);
        }
    }
};

template <int OP, bool HAS_MASK>
struct ReduceOp {
    // events per lane: these kernels do little per event, so tiles are large (count stages one byte per element at most
    // and can afford 128 events per tile)
    static constexpr int H = OP == OP_COUNT ? 4 : 2;
    typedef TileShape<H, 1, OP != OP_COUNT ? 1 : 0, HAS_MASK ? 1 : 0> Shape;
    const float* data;
    const unsigned char* mask_rows;
    const unsigned char* mask_content;
    typename RedOut<OP>::type* out;

    // value that leaves the reduction unchanged (what a masked-out element is replaced with)
    __device__ static __forceinline__ float neutral()
    {
        return OP == OP_MAX ? -CUDART_INF_F : (OP == OP_MIN ? CUDART_INF_F : (OP == OP_ARGMAX ? CUDART_NAN_F : 0.f));
    }
    __device__ __forceinline__ void staged(const TileParams&, const uint32_t (&ca)[Shape::NCA], uint32_t extra_a,
                                           long long e0, int ne, int lane, const int (&o)[1][H + 1],
                                           const int (&lo)[1], const int (&cnt)[1])
    {
        constexpr bool DATA = OP != OP_COUNT;
        // count over a mask: a flat pass turns the tile's mask bytes into a bit string (one ballot per 32 elements), and
        // an event's count is the population count of its bit range
        constexpr bool BITS = OP == OP_COUNT && HAS_MASK;
        unsigned bit0 = 0;                    // bit of the tile's first element in the string
        if (BITS) {
            // Four mask bytes per lane (one 32-bit load from the 4-byte-aligned address at or below the first element),
            // folded into a nibble; the nibbles of eight neighbouring lanes make a word of the string.  Bits of bytes
            // in front of the first element or behind the last one are whatever the buffer holds: no range covers them.
            bit0 = ca[0] & 3u;
            const uint32_t a4 = ca[0] - bit0;
            const int nb = cnt[0] + (int)bit0;
            const unsigned shl = 4u * ((unsigned)lane & 7u);
            uint32_t wa = extra_a + 4u * ((unsigned)lane >> 3);
            int i0 = 0;
            for (; i0 < nb; i0 += 128, wa += 16u) {
                const int i = i0 + 4 * lane;
                unsigned w = 0u;
                if (i < nb) w = lds_w(a4 + (unsigned)i);
                const unsigned t = (w | ((w & 0x7f7f7f7fu) + 0x7f7f7f7fu)) & 0x80808080u;      // high bit of every non-zero byte
                unsigned v = (((t >> 7) * 0x01020408u) >> 24) << shl;                            // ... gathered: bit b = byte b
                v |= __shfl_xor_sync(0xffffffffu, v, 1);
                v |= __shfl_xor_sync(0xffffffffu, v, 2);
                v |= __shfl_xor_sync(0xffffffffu, v, 4);
                if (((unsigned)lane & 7u) == 0u) sts_w(wa, v);
            }
            if (lane == 0) sts_w(extra_a + 4u * (unsigned)(i0 >> 5), 0u);        // (a range may end exactly at a word boundary)
            __syncwarp();
        }
        constexpr int TAIL = 16;          // elements of an event beyond this many are reduced by the whole warp
        constexpr unsigned ES = DATA ? 4u : 1u;
        // Flat pass, one lane per element: a masked-out element becomes the reduction's neutral value, so the
        // per-event loops below never look at the mask.  (count: the mask byte itself is what is summed.)
        if (DATA && HAS_MASK) {
            for (int j = lane; j < cnt[0]; j += 32)
                if (!lds_b(ca[1] + (unsigned)j))
                    asm volatile("st.shared.f32 [%0], %1;" ::"r"(ca[0] + 4u * (unsigned)j), "f"(neutral()) : "memory");
            __syncwarp();
        }
        auto value = [&](uint32_t a, bool& take) {
            if (DATA) { take = true; return lds_f(a); }
            take = lds_b(a) != 0u;
            return 0.f;
        };
        typename RedOut<OP>::type res[H];
#pragma unroll
        for (int h = 0; h < H; ++h) {
            const int ev = lane * H + h;              // event of the tile
            int n = o[0][h + 1] - o[0][h];            // (0 for events past the tile's end)
            if (mask_rows && ev < ne && !__ldg(mask_rows + e0 + ev)) n = 0;
            RedAcc<OP> acc;
            acc.init();
            if (!DATA && !HAS_MASK) {
                acc.i = n;
            } else if (BITS) {
                int pos = o[0][h] - lo[0] + (int)bit0, rem = n, c = 0;
                while (rem > 0) {
                    const int take = rem < 32 ? rem : 32;
                    const uint32_t wa = extra_a + 4u * (unsigned)(pos >> 5);
                    unsigned v = __funnelshift_r(lds_w(wa), lds_w(wa + 4u), (unsigned)(pos & 31));
                    if (take < 32) v &= (1u << take) - 1u;
                    c += __popc(v);
                    pos += take; rem -= take;
                }
                acc.i = c;
            } else {
                const uint32_t a0 = ca[0] + ES * (unsigned)(o[0][h] - lo[0]);
                const int nmain = n < TAIL ? n : TAIL;
                uint32_t ad = a0;
                int k = 0;
                bool t0, t1;
                if (nmain & 1) {
                    const float x = value(ad, t0);
                    if (OP == OP_ARGMAX) acc.push_gt(x, 0); else acc.push(x, 0, t0);
                    k = 1; ad += ES;
                }
#pragma unroll 1
                for (; k < nmain; k += 2, ad += 2 * ES) {          // two elements per iteration
                    const float x0 = value(ad, t0), x1 = value(ad + ES, t1);
                    if (OP == OP_ARGMAX) { acc.push_gt(x0, k); acc.push_gt(x1, k + 1); }
                    else { acc.push(x0, k, t0); acc.push(x1, k + 1, t1); }
                }
                if (OP == OP_ARGMAX && acc.i < 0 && nmain > 0) {   // nothing above -inf: the full rule (rare)
                    acc.init();
                    for (int kk = 0; kk < nmain; ++kk) acc.push(lds_f(a0 + ES * (unsigned)kk), kk, true);
                }
                // long events: the rest of their elements, 32 at a time, one per lane, folded into the owner's state
                for (unsigned lm = __ballot_sync(0xffffffffu, n > TAIL); lm; lm &= lm - 1) {
                    const int src = __ffs(lm) - 1;
                    const uint32_t as = __shfl_sync(0xffffffffu, a0, src);
                    const int ns = __shfl_sync(0xffffffffu, n, src);
                    RedAcc<OP> part;
                    part.init();
                    for (int kk = TAIL + lane; kk < ns; kk += 32) {
                        const float x = value(as + ES * (unsigned)kk, t0);
                        part.push(x, kk, t0);
                    }
                    part.warp_reduce();
                    if (lane == src) acc.merge(part);
                }
            }
            res[h] = acc.result();
        }
        // a lane's H results are neighbours in memory: one vector store when the whole group is live
        typename RedOut<OP>::type* dst = out + e0 + lane * H;
        typedef typename std::conditional<H >= 4, int4, int2>::type V;
        static_assert(H == 2 || H == 4 || H == 8, "the vector stores cover 2, 4 or 8 results");
        if (lane * H + H <= ne && (reinterpret_cast<uintptr_t>(dst) & (sizeof(V) - 1)) == 0) {
#pragma unroll
            for (int q = 0; q < (int)(H * 4 / sizeof(V)); ++q) reinterpret_cast<V*>(dst)[q] = reinterpret_cast<const V*>(res)[q];
        } else {
#pragma unroll
            for (int h = 0; h < H; ++h)
                if (lane * H + h < ne) dst[h] = res[h];
        }
    }
    // Straight from global memory, 32 events at a time: one lane per event (the paper's loop shape) for events of up
    // to 64 particles, the whole warp striding over the particles of a larger one.
    __device__ __forceinline__ void global(const TileParams& P, long long e0, int ne, int lane)
    {
        for (int b = 0; b < ne; b += 32) {
            const long long e = e0 + b + lane;
            const bool live = b + lane < ne;
            long long g0 = 0, g1 = 0;
            if (live && (!mask_rows || mask_rows[e])) { g0 = P.off[0][e]; g1 = P.off[0][e + 1]; }
            const bool big = g1 - g0 > 64;
            RedAcc<OP> acc;
            acc.init();
            if (!big)
                for (long long g = g0; g < g1; ++g) {
                    const long long i = g - P.base[0];
                    acc.push(OP == OP_COUNT ? 0.f : data[i], (int)(g - g0), !mask_content || mask_content[i] != 0);
                }
            for (unsigned lm = __ballot_sync(0xffffffffu, big); lm; lm &= lm - 1) {
                const int src = __ffs(lm) - 1;
                const long long s0 = __shfl_sync(0xffffffffu, g0, src), s1 = __shfl_sync(0xffffffffu, g1, src);
                RedAcc<OP> part;
                part.init();
                for (long long g = s0 + lane; g < s1; g += 32) {
                    const long long i = g - P.base[0];
                    part.push(OP == OP_COUNT ? 0.f : data[i], (int)(g - s0), !mask_content || mask_content[i] != 0);
                }
                part.warp_reduce();
                if (lane == src) acc = part;
            }
            if (live) out[e] = acc.result();
        }
    }
};

template <int OP, bool HAS_MASK>
__global__ void __launch_bounds__(256, 4) segreduce_stream_kernel(const __grid_constant__ TileParams P, ReduceOp<OP, HAS_MASK> op)
{
    tile_stream<typename ReduceOp<OP, HAS_MASK>::Shape>(P, op);
}

// Variant 1: one warp per event, lanes stride over the event's particles (coalesced), shuffle reduction.
template <int OP>
__global__ void __launch_bounds__(256) segreduce_warp_kernel(const float* __restrict__ data, const long long* __restrict__ offsets,
                                                             long long n_events, long long base,
                                                             const unsigned char* __restrict__ mask_rows,
                                                             const unsigned char* __restrict__ mask_content,
                                                             typename RedOut<OP>::type* __restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long e = warp0; e < n_events; e += nwarps) {
        RedAcc<OP> acc;
        acc.init();
        if (!mask_rows || mask_rows[e]) {
            const long long g0 = offsets[e], g1 = offsets[e + 1];
            for (long long g = g0 + lane; g < g1; g += 32) {
                const long long i = g - base;
                if (mask_content && !mask_content[i]) continue;
                acc.push(OP == OP_COUNT ? 0.f : data[i], (int)(g - g0), true);
            }
        }
        acc.warp_reduce();
        if (lane == 0) out[e] = acc.result();
    }
}

// =========================================================================================== deltar_mask
// Staged columns: eta1, phi1, (sel1), eta2, phi2, (sel2).  Per-warp scratch: one word per event (its collection-2
// range) and one byte per collection-1 object of the tile (the lane of its event).
template <bool S1, bool S2>
struct DeltarOp {
    typedef TileShape<1, 2, 2, S1 ? 1 : 0, 2, S2 ? 1 : 0> Shape;
    const float *eta1, *phi1, *eta2, *phi2;
    const unsigned char *sel1, *sel2;
    unsigned char* out;
    float dr2_max;

    __device__ __forceinline__ void staged(const TileParams& P, const uint32_t (&ca)[Shape::NCA], uint32_t extra_a, long long, int ne,
                                           int lane, const int (&o)[2][2], const int (&lo)[2], const int (&cnt)[2])
    {
        const uint32_t a_e1 = ca[0], a_p1 = ca[1], a_s1 = S1 ? ca[2] : 0u;
        const uint32_t a_e2 = ca[S1 ? 3 : 2], a_p2 = ca[S1 ? 4 : 3], a_s2 = S2 ? ca[S1 ? 5 : 4] : 0u;
        const uint32_t range_a = extra_a, evid_a = extra_a + 4u * WT_EVENTS;
        const bool live = lane < ne;
        const int k0 = o[0][0] - lo[0], n1 = live ? o[0][1] - o[0][0] : 0;
        const int m0 = o[1][0] - lo[1], n2 = live ? o[1][1] - o[1][0] : 0;
        // byte range of the event's collection-2 objects inside a float column (begin, end), 16 bits each
        sts_w(range_a + 4u * (unsigned)lane, (unsigned)(4 * m0) | ((unsigned)(4 * (m0 + n2)) << 16));
        if (S2) {       // an unselected object of collection 2 can never match: eta = NaN
            for (int m = lane; m < cnt[1]; m += 32)
                if (!lds_b(a_s2 + (unsigned)m)) asm volatile("st.shared.u32 [%0], %1;" ::"r"(a_e2 + 4u * (unsigned)m), "r"(0x7fc00000u) : "memory");
        }
        {
            uint32_t a = evid_a + (unsigned)k0;
            const uint32_t aend = a + (unsigned)n1;
            if (n1 & 1) { sts_b(a, (unsigned)lane); a += 1; }
#pragma unroll 1
            for (; a != aend; a += 2) { sts_b(a, (unsigned)lane); sts_b(a + 1, (unsigned)lane); }
        }
        __syncwarp();
        const long long l1 = (long long)(int)((unsigned)lo[0] - (unsigned)P.base[0]);
        unsigned char* dst = out + l1;
#pragma unroll 1
        for (int j = lane; j < cnt[0]; j += 32) {
            const float eta = lds_f(a_e1 + 4u * (unsigned)j), phi = lds_f(a_p1 + 4u * (unsigned)j);
            const unsigned int r = lds_w(range_a + 4u * lds_b(evid_a + (unsigned)j));
            uint32_t b = r & 0xffffu;
            const uint32_t e = r >> 16;
            float dmin = CUDART_INF_F;
#pragma unroll 1
            for (; b != e; b += 4) dmin = fminf(dmin, dr2_exact(eta, phi, lds_f(a_e2 + b), lds_f(a_p2 + b)));   // fminf skips a NaN
            bool matched = dmin < dr2_max;
            if (S1) matched = matched && lds_b(a_s1 + (unsigned)j) != 0u;
            dst[j] = matched ? 1 : 0;
        }
    }
    __device__ __forceinline__ void match_range(const TileParams& P, long long g0, long long g1, long long gs, long long h0, long long h1) const
    {
        for (long long g = g0; g < g1; g += gs) {
            const long long j = g - P.base[0];
            bool matched = false;
            if (!sel1 || sel1[j]) {
                const float eta = eta1[j], phi = phi1[j];
                for (long long h = h0; h < h1 && !matched; ++h) {
                    const long long m = h - P.base[1];
                    if (sel2 && !sel2[m]) continue;
                    matched = dr2_exact(eta, phi, eta2[m], phi2[m]) < dr2_max;
                }
            }
            out[j] = matched ? 1 : 0;
        }
    }
    // Straight from global memory: one lane per event (the paper's nested loop) for events of up to 64 collection-1
    // objects, the whole warp striding over the objects of a larger one.
    __device__ __forceinline__ void global(const TileParams& P, long long e0, int ne, int lane)
    {
        for (int b = 0; b < ne; b += 32) {
            const long long e = e0 + b + lane;
            const bool live = b + lane < ne;
            long long g0 = 0, g1 = 0, h0 = 0, h1 = 0;
            if (live) { g0 = P.off[0][e]; g1 = P.off[0][e + 1]; h0 = P.off[1][e]; h1 = P.off[1][e + 1]; }
            const bool big = g1 - g0 > 64;
            if (!big) match_range(P, g0, g1, 1, h0, h1);
            for (unsigned lm = __ballot_sync(0xffffffffu, big); lm; lm &= lm - 1) {
                const int src = __ffs(lm) - 1;
                const long long s0 = __shfl_sync(0xffffffffu, g0, src), s1 = __shfl_sync(0xffffffffu, g1, src);
                const long long t0 = __shfl_sync(0xffffffffu, h0, src), t1 = __shfl_sync(0xffffffffu, h1, src);
                match_range(P, s0 + lane, s1, 32, t0, t1);
            }
        }
    }
};

template <bool S1, bool S2>
__global__ void __launch_bounds__(256, 4) deltar_stream_kernel(const __grid_constant__ TileParams P, DeltarOp<S1, S2> op)
{
    tile_stream<typename DeltarOp<S1, S2>::Shape>(P, op);
}

// =========================================================================================== pair_invmass
// Staged columns: pt, eta, phi, mass, (mask).  One lane per event.
template <bool HAS_MASK>
struct InvmassOp {
    typedef TileShape<1, 1, 4, HAS_MASK ? 1 : 0> Shape;
    const float *pt, *eta, *phi, *mass;
    const unsigned char* mask;
    float* out_mass;
    int *out_i1, *out_i2;

    __device__ __forceinline__ void staged(const TileParams&, const uint32_t (&ca)[Shape::NCA], uint32_t, long long e0, int ne, int lane,
                                           const int (&o)[1][2], const int (&lo)[1], const int (&cnt)[1])
    {
        const bool live = lane < ne;
        const int k0 = o[0][0] - lo[0], n = live ? o[0][1] - o[0][0] : 0;
        // masked-out jets become NaN in a flat pass (one lane per jet), so the per-event loop never looks at the mask
        if (HAS_MASK) {
            for (int j = lane; j < cnt[0]; j += 32)
                if (!lds_b(ca[4] + (unsigned)j)) sts_w(ca[0] + 4u * (unsigned)j, 0x7fc00000u);
            __syncwarp();
        }
        constexpr int TAIL = 16;          // jets of an event beyond this many are taken by the whole warp
        Top2 top;
        top.init();
        const uint32_t a0 = ca[0] + 4u * (unsigned)k0;
        const int nmain = n < TAIL ? n : TAIL;
#pragma unroll 1
        for (int k = 0; k < nmain; ++k) top.push_any(lds_f(a0 + 4u * (unsigned)k), k);
        for (unsigned lm = __ballot_sync(0xffffffffu, n > TAIL); lm; lm &= lm - 1) {
            const int src = __ffs(lm) - 1;
            const uint32_t as = __shfl_sync(0xffffffffu, a0, src);
            const int ns = __shfl_sync(0xffffffffu, n, src);
            // 32 jets at a time, one per lane: the two best of the chunk by (value desc, index asc), folded into the
            // owner's state in that order (their indices exceed every index seen so far, so the tie rule holds)
            for (int kb = TAIL; kb < ns; kb += 32) {
                const int k = kb + lane;
                const float p = k < ns ? lds_f(as + 4u * (unsigned)k) : CUDART_NAN_F;
                const bool ok = p == p;
                // order-preserving key: a < b <=> key(a) < key(b); 0 marks "no value"
                const unsigned bits = p == 0.f ? 0u : __float_as_uint(p);      // (-0 and +0 are one value)
                const unsigned u = ok ? (bits ^ ((unsigned)((int)bits >> 31) | 0x80000000u)) : 0u;
                const unsigned k1 = __reduce_max_sync(0xffffffffu, u);
                const int j1 = __reduce_min_sync(0xffffffffu, (ok && u == k1) ? k : 0x7fffffff);
                const unsigned u2 = k == j1 ? 0u : u;
                const unsigned k2 = __reduce_max_sync(0xffffffffu, u2);
                const int j2 = __reduce_min_sync(0xffffffffu, (u2 != 0u && u2 == k2) ? k : 0x7fffffff);
                if (lane == src) {
                    if (k1 != 0u) top.push_any(__uint_as_float(k1 ^ ((k1 & 0x80000000u) ? 0x80000000u : 0xffffffffu)), j1);
                    if (k2 != 0u) top.push_any(__uint_as_float(k2 ^ ((k2 & 0x80000000u) ? 0x80000000u : 0xffffffffu)), j2);
                }
            }
        }
        float m = 0.f;
        if (top.i2 >= 0) {
            const unsigned a = 4u * (unsigned)(k0 + top.i1), c = 4u * (unsigned)(k0 + top.i2);
            m = pair_mass_lean(top.b1, lds_f(ca[1] + a), lds_f(ca[2] + a), lds_f(ca[3] + a),
                               top.b2, lds_f(ca[1] + c), lds_f(ca[2] + c), lds_f(ca[3] + c));
        }
        if (live) {
            out_mass[e0 + lane] = m;
            if (out_i1) out_i1[e0 + lane] = top.i1;
            if (out_i2) out_i2[e0 + lane] = top.i2;
        }
    }
    // the paper's loop shape: one lane per event, global memory
    __device__ __forceinline__ void global(const TileParams& P, long long e0, int ne, int lane)
    {
        if (lane >= ne) return;
        const long long e = e0 + lane, g0 = P.off[0][e], g1 = P.off[0][e + 1];
        Top2 top;
        top.init();
        for (long long g = g0; g < g1; ++g) {
            const long long i = g - P.base[0];
            if (mask && !mask[i]) continue;
            top.push_any(pt[i], (int)(g - g0));
        }
        float m = 0.f;
        if (top.i2 >= 0) {
            const long long a = g0 - P.base[0] + top.i1, c = g0 - P.base[0] + top.i2;
            m = pair_mass_f32(top.b1, eta[a], phi[a], mass[a], top.b2, eta[c], phi[c], mass[c]);
        }
        out_mass[e] = m;
        if (out_i1) out_i1[e] = top.i1;
        if (out_i2) out_i2[e] = top.i2;
    }
};

template <bool HAS_MASK>
__global__ void __launch_bounds__(256, 2) invmass_stream_kernel(const __grid_constant__ TileParams P, InvmassOp<HAS_MASK> op)
{
    tile_stream<typename InvmassOp<HAS_MASK>::Shape>(P, op);
}

// =========================================================================================== select_opposite_sign
// Staged columns: pt, charge (int32, moved as 32-bit words), (mask).  One lane per event finds the leading object and
// the best object of each sign; the two chosen objects are marked in a per-warp byte buffer that a flat pass writes out
// (coalesced bytes, every object of the tile).
struct OppSignPick {
    int lead, bpos, bneg;
    float plead, ppos, pneg;
    int qlead;
    __device__ __forceinline__ void init() { lead = bpos = bneg = -1; plead = ppos = pneg = 0.f; qlead = 0; }
    // strict > keeps the first index among equal pt; NaN skipped
    __device__ __forceinline__ void push(float p, int q, int k)
    {
        if (p != p) return;
        if (lead < 0 || p > plead) { lead = k; plead = p; qlead = q; }
        if (q > 0 && (bpos < 0 || p > ppos)) { bpos = k; ppos = p; }
        if (q < 0 && (bneg < 0 || p > pneg)) { bneg = k; pneg = p; }
    }
    __device__ __forceinline__ int partner() const
    {
        if (lead < 0) return -1;
        return qlead > 0 ? bneg : (qlead < 0 ? bpos : -1);      // charge 0 has no opposite sign
    }
};

template <bool HAS_MASK>
struct OppSignOp {
    static constexpr int H = 4;          // (lepton collections are sparse: 128 events per tile)
    typedef TileShape<H, 1, 2, HAS_MASK ? 1 : 0> Shape;
    const float* pt;
    const int* charge;
    const unsigned char *mask_rows, *mask;
    unsigned char* out;

    __device__ __forceinline__ void staged(const TileParams& P, const uint32_t (&ca)[Shape::NCA], uint32_t extra_a, long long e0, int ne,
                                           int lane, const int (&o)[1][H + 1], const int (&lo)[1], const int (&cnt)[1])
    {
        const int nw = (cnt[0] + 3) >> 2;
        for (int j = lane; j < nw; j += 32) sts_w(extra_a + 4u * (unsigned)j, 0u);
        __syncwarp();
#pragma unroll
        for (int h = 0; h < H; ++h) {
            const int ev = lane * H + h;
            const int k0 = o[0][h] - lo[0];
            int n = o[0][h + 1] - o[0][h];
            if (mask_rows && ev < ne && !__ldg(mask_rows + e0 + ev)) n = 0;
            OppSignPick pk;
            pk.init();
            uint32_t ap = ca[0] + 4u * (unsigned)k0, aq = ca[1] + 4u * (unsigned)k0, am = HAS_MASK ? ca[2] + (unsigned)k0 : 0u;
#pragma unroll 1
            for (int k = 0; k < n; ++k, ap += 4, aq += 4, am += 1) {
                if (HAS_MASK && !lds_b(am)) continue;
                pk.push(lds_f(ap), (int)lds_w(aq), k);
            }
            const int part = pk.partner();
            if (part >= 0) {
                sts_b(extra_a + (unsigned)(k0 + pk.lead), 1u);
                sts_b(extra_a + (unsigned)(k0 + part), 1u);
            }
        }
        __syncwarp();
        unsigned char* dst = out + (long long)(int)((unsigned)lo[0] - (unsigned)P.base[0]);
        for (int j = lane; j < cnt[0]; j += 32) dst[j] = (unsigned char)lds_b(extra_a + (unsigned)j);
    }
    // the paper's loop shape: one lane per event, global memory
    __device__ __forceinline__ void global(const TileParams& P, long long e0, int ne, int lane)
    {
        for (int b = 0; b < ne; b += 32) {
            if (b + lane >= ne) continue;
            const long long e = e0 + b + lane;
            const long long g0 = P.off[0][e], g1 = P.off[0][e + 1];
            OppSignPick pk;
            pk.init();
            if (!mask_rows || mask_rows[e])
                for (long long g = g0; g < g1; ++g) {
                    const long long i = g - P.base[0];
                    if (mask && !mask[i]) continue;
                    pk.push(pt[i], charge[i], (int)(g - g0));
                }
            const int part = pk.partner();
            for (long long g = g0; g < g1; ++g) {
                const int k = (int)(g - g0);
                out[g - P.base[0]] = (part >= 0 && (k == pk.lead || k == part)) ? 1 : 0;
            }
        }
    }
};

template <bool HAS_MASK>
__global__ void __launch_bounds__(256, 4) oppsign_stream_kernel(const __grid_constant__ TileParams P, OppSignOp<HAS_MASK> op)
{
    tile_stream<typename OppSignOp<HAS_MASK>::Shape>(P, op);
}

}  // namespace dev

// ------------------------------------------------------------------------------------------ host side
struct TileLayout {
    TileParams P;
    int warps_per_cta, grid;
    size_t smem;
};

// Fill the staging geometry.  n_cls[q]: columns per class (float32 / uint8 of collection 0, then of collection 1),
// ptr: their pointers in that order; cap_coll: slice capacity per collection; extra: per-warp scratch bytes.
static int32_t tile_layout(TileLayout& L, long long n_events, int n_coll, const int64_t* const* off, const int64_t* base,
                           const int (&n_cls)[4], const void* const* ptr, const int* cap_coll, int extra_bytes, int max_warps_sm)
{
    TileParams& P = L.P;
    memset(&P, 0, sizeof(P));
    P.n_events = n_events;
    const long long nt = (n_events + WT_EVENTS - 1) / WT_EVENTS;
    if (nt >= (1ll << 31)) {
        set_error("n_events = %lld is beyond the 2^36 a launch supports", n_events);
        return HEPK_ERR_UNSUPPORTED;
    }
    P.staged = 1;
    for (int c = 0; c < n_coll; ++c) {
        P.off[c] = (const long long*)off[c];
        P.base[c] = base[c];
        P.cap[c] = cap_coll[c];
    }
    size_t o = 16;
    int k = 0;
    for (int q = 0; q < 4; ++q) {
        const int es = (q & 1) ? 1 : 4;
        for (int j = 0; j < n_cls[q]; ++j, ++k) {
            const uintptr_t addr = reinterpret_cast<uintptr_t>(ptr[k]);
            const int mis = (int)((addr / (uintptr_t)es) % (uintptr_t)(16 / es));
            if (addr % (uintptr_t)es) P.staged = 0;                 // not even element-aligned
            if (j == 0) P.mis[q] = mis;
            else if (mis != P.mis[q]) P.staged = 0;                 // the columns of a class must share their alignment
            P.ptr[k] = (const char*)ptr[k];
            o = (o + 15) / 16 * 16;
            P.dst[k] = (int)o;
            o += (size_t)(cap_coll[q >> 1] + 32) * (size_t)es;
        }
    }
    P.stage_bytes = (int)((o + 127) / 128 * 128);
    P.extra_off = 2 * P.stage_bytes;
    P.warp_bytes = P.extra_off + (extra_bytes + 127) / 128 * 128;
    const int smem_max = max_smem_optin();
    // warps per SM: as many as fit (each CTA also pays 1 KB of system shared memory), in CTAs of up to 8 warps
    int best_ctas = 1, best_wpc = 1, best_total = 0;
    for (int ctas = 1; ctas <= 8; ++ctas) {
        int budget = (smem_max + 1024) / ctas - 1024;
        if (budget > smem_max) budget = smem_max;
        int wpc = budget / P.warp_bytes;
        if (wpc > 8) wpc = 8;
        if (wpc * ctas > max_warps_sm) wpc = max_warps_sm / ctas;
        if (wpc < 1) continue;
        if (wpc * ctas > best_total) { best_total = wpc * ctas; best_ctas = ctas; best_wpc = wpc; }
    }
    if (best_total == 0) {
        set_error("a tile needs %d bytes of shared memory (max %d)", P.warp_bytes, smem_max);
        return HEPK_ERR_UNSUPPORTED;
    }
    L.warps_per_cta = best_wpc;
    L.smem = (size_t)best_wpc * P.warp_bytes;
    long long grid = (long long)sm_count() * best_ctas;
    const long long need = (nt + best_wpc - 1) / best_wpc;
    if (grid > need) grid = need;
    L.grid = (int)(grid < 1 ? 1 : grid);
    return HEPK_OK;
}

template <class Kern, class Op>
static int32_t tile_launch(Kern kern, const TileLayout& L, const Op& op, cudaStream_t st)
{
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)L.smem));
    kern<<<L.grid, L.warps_per_cta * 32, L.smem, st>>>(L.P, op); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

// Slice capacities (objects per tile).  Fixed: the kernels adapt the number of events per tile to them (a tile of E
// events is taken when E * mean + 4 sqrt(2 E mean + 1) + 8 objects fit: 32-event tiles up to a mean of 9.7 objects
// per event at 416, 8.8 at 384, 1.9 at 112).  They are sized for the warps they leave room for, measured on
// BASELINE.json configs[2]: deltar_mask 416/160 -> 416/112 takes 20 warps per SM instead of 18 (0.465 -> 0.421 ms per
// 10 M events; 400/128 0.423, 384/128 0.438: with fewer than ~410 jets a few dozen tiles per launch overflow into the
// lane-per-event path and the warps that meet them finish last), pair_invmass 416 -> 384 takes 16 instead of 15
// (0.399 -> 0.374 ms).
constexpr int CAP_REDUCE = 672, CAP_DR_1 = 416, CAP_DR_2 = 112, CAP_MASS = 384;      // (reductions: 64 events per tile)

template <int OP>
static int32_t segreduce_dispatch(const float* data, const int64_t* offsets, int64_t n_events, int64_t base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, void* out, int32_t variant,
                                  void* stream)
{
    typedef typename dev::RedOut<OP>::type T;
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(variant >= 0 && variant <= 2, "unknown variant");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out, "offsets/out is NULL");
    HEPK_REQUIRE(OP == dev::OP_COUNT || data, "data is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (variant == HEPK_VARIANT_WARP_PER_EVENT) {
        auto kern = dev::segreduce_warp_kernel<OP>;
        long long blocks = (n_events + 7) / 8;
        const long long maxb = (long long)sm_count() * 32;
        if (blocks > maxb) blocks = maxb;
        kern<<<(unsigned)blocks, 256, 0, st>>>(data, (const long long*)offsets, n_events, base, mask_rows, mask_content, (T*)out); count_launch();
        HEPK_CUDA_TRY(cudaGetLastError());
        return HEPK_OK;
    }
    const bool has_data = OP != dev::OP_COUNT;
    const void* ptr[2] = {nullptr, nullptr};
    int k = 0;
    if (has_data) ptr[k++] = data;
    if (mask_content) ptr[k++] = mask_content;
    const int n_cls[4] = {has_data ? 1 : 0, mask_content ? 1 : 0, 0, 0};
    const int64_t* offs[1] = {offsets};
    const int64_t bases[1] = {base};
    const int caps[1] = {OP == dev::OP_COUNT ? 2 * CAP_REDUCE : CAP_REDUCE};
    TileLayout L;
    const int32_t rc = tile_layout(L, n_events, 1, offs, bases, n_cls, ptr, caps, OP == dev::OP_COUNT ? caps[0] / 8 + 16 : 0, 32);
    if (rc != HEPK_OK) return rc;
    if (mask_content) {
        dev::ReduceOp<OP, true> op;
        op.data = data; op.mask_rows = mask_rows; op.mask_content = mask_content; op.out = (T*)out;
        return tile_launch(dev::segreduce_stream_kernel<OP, true>, L, op, st);
    }
    dev::ReduceOp<OP, false> op;
    op.data = data; op.mask_rows = mask_rows; op.mask_content = nullptr; op.out = (T*)out;
    return tile_launch(dev::segreduce_stream_kernel<OP, false>, L, op, st);
}

template <bool S1, bool S2>
static int32_t deltar_launch(const TileLayout& L, const float* eta1, const float* phi1, const uint8_t* sel1, const float* eta2,
                             const float* phi2, const uint8_t* sel2, float dr_max, uint8_t* out, cudaStream_t st)
{
    dev::DeltarOp<S1, S2> op;
    op.eta1 = eta1; op.phi1 = phi1; op.eta2 = eta2; op.phi2 = phi2; op.sel1 = sel1; op.sel2 = sel2;
    op.out = out;
    op.dr2_max = dr_max * dr_max;      // float32 product (exact class)
    return tile_launch(dev::deltar_stream_kernel<S1, S2>, L, op, st);
}

template <bool M>
static int32_t invmass_launch(const TileLayout& L, const float* pt, const float* eta, const float* phi, const float* mass,
                              const uint8_t* mask, float* out_mass, int32_t* out_i1, int32_t* out_i2, cudaStream_t st)
{
    dev::InvmassOp<M> op;
    op.pt = pt; op.eta = eta; op.phi = phi; op.mass = mass; op.mask = mask;
    op.out_mass = out_mass; op.out_i1 = out_i1; op.out_i2 = out_i2;
    return tile_launch(dev::invmass_stream_kernel<M>, L, op, st);
}

}  // namespace hepk

using namespace hepk;

#define HEPK_DEFINE_SEGREDUCE(NAME, OP, T)                                                                             \
    extern "C" int32_t hepk_segmented_reduce_##NAME(const float* data, const int64_t* offsets, int64_t n_events,       \
                                                    int64_t content_base, const uint8_t* mask_rows,                   \
                                                    const uint8_t* mask_content, T* out, int32_t variant, void* stream) \
    {                                                                                                                  \
        return segreduce_dispatch<OP>(data, offsets, n_events, content_base, mask_rows, mask_content, out, variant,    \
                                      stream);                                                                         \
    }
HEPK_DEFINE_SEGREDUCE(sum, dev::OP_SUM, float)
HEPK_DEFINE_SEGREDUCE(max, dev::OP_MAX, float)
HEPK_DEFINE_SEGREDUCE(min, dev::OP_MIN, float)
HEPK_DEFINE_SEGREDUCE(count, dev::OP_COUNT, int32_t)
HEPK_DEFINE_SEGREDUCE(argmax, dev::OP_ARGMAX, int32_t)

extern "C" int32_t hepk_deltar_mask(const float* eta1, const float* phi1, const int64_t* offsets1, int64_t base1, const uint8_t* sel1,
                                    const float* eta2, const float* phi2, const int64_t* offsets2, int64_t base2, const uint8_t* sel2,
                                    int64_t n_events, float dr_max, uint8_t* out_matched, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets1 && offsets2, "offsets is NULL");
    const void* ptr[6];
    int k = 0;
    ptr[k++] = eta1; ptr[k++] = phi1;
    if (sel1) ptr[k++] = sel1;
    ptr[k++] = eta2; ptr[k++] = phi2;
    if (sel2) ptr[k++] = sel2;
    const int n_cls[4] = {2, sel1 ? 1 : 0, 2, sel2 ? 1 : 0};
    const int64_t* offs[2] = {offsets1, offsets2};
    const int64_t bases[2] = {base1, base2};
    const int caps[2] = {CAP_DR_1, CAP_DR_2};
    TileLayout L;
    const int32_t rc = tile_layout(L, n_events, 2, offs, bases, n_cls, ptr, caps, 4 * WT_EVENTS + caps[0] + 32, 32);
    if (rc != HEPK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (sel1 && sel2) return deltar_launch<true, true>(L, eta1, phi1, sel1, eta2, phi2, sel2, dr_max, out_matched, st);
    if (sel1) return deltar_launch<true, false>(L, eta1, phi1, sel1, eta2, phi2, sel2, dr_max, out_matched, st);
    if (sel2) return deltar_launch<false, true>(L, eta1, phi1, sel1, eta2, phi2, sel2, dr_max, out_matched, st);
    return deltar_launch<false, false>(L, eta1, phi1, sel1, eta2, phi2, sel2, dr_max, out_matched, st);
}

extern "C" int32_t hepk_pair_invmass(const float* pt, const float* eta, const float* phi, const float* mass,
                                     const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_content,
                                     float* out_mass, int32_t* out_i1, int32_t* out_i2, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out_mass, "offsets/out_mass is NULL");
    const void* ptr[5] = {pt, eta, phi, mass, mask_content};
    const int n_cls[4] = {4, mask_content ? 1 : 0, 0, 0};
    const int64_t* offs[1] = {offsets};
    const int64_t bases[1] = {content_base};
    const int caps[1] = {CAP_MASS};
    TileLayout L;
    const int32_t rc = tile_layout(L, n_events, 1, offs, bases, n_cls, ptr, caps, 0, 32);
    if (rc != HEPK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (mask_content) return invmass_launch<true>(L, pt, eta, phi, mass, mask_content, out_mass, out_i1, out_i2, st);
    return invmass_launch<false>(L, pt, eta, phi, mass, mask_content, out_mass, out_i1, out_i2, st);
}

extern "C" int32_t hepk_select_opposite_sign(const float* pt, const int32_t* charge, const int64_t* offsets, int64_t n_events,
                                             int64_t content_base, const uint8_t* mask_rows, const uint8_t* mask_content,
                                             uint8_t* out_mask, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && charge && out_mask, "offsets/charge/out_mask is NULL");
    // objects per 128-event tile (the kernel takes fewer lanes per tile for denser collections: 128-event tiles up to a
    // mean of 1.9 objects per event); 352 leaves room for 32 warps per SM, 416 for 28 (0.099 -> 0.095 ms per 10 M events)
    constexpr int CAP = 352;
    const void* ptr[3] = {pt, charge, mask_content};
    const int n_cls[4] = {2, mask_content ? 1 : 0, 0, 0};
    const int64_t* offs[1] = {offsets};
    const int64_t bases[1] = {content_base};
    const int caps[1] = {CAP};
    TileLayout L;
    const int32_t rc = tile_layout(L, n_events, 1, offs, bases, n_cls, ptr, caps, CAP + 64, 32);
    if (rc != HEPK_OK) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    if (mask_content) {
        dev::OppSignOp<true> op;
        op.pt = pt; op.charge = charge; op.mask_rows = mask_rows; op.mask = mask_content; op.out = out_mask;
        return tile_launch(dev::oppsign_stream_kernel<true>, L, op, st);
    }
    dev::OppSignOp<false> op;
    op.pt = pt; op.charge = charge; op.mask_rows = mask_rows; op.mask = nullptr; op.out = out_mask;
    return tile_launch(dev::oppsign_stream_kernel<false>, L, op, st);
}
