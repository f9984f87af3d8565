// hepk_hist_lanes.cuh — the fill kernel for small one-dimensional histograms, shared by hepk_fill_histogram
// (hepk_kernels.cu) and hepk_fill_histogram_w2 (hepk_hist.cu); PAPER.md:L109 `fill_histogram`.
#pragma once
#include "hepk_common.cuh"

namespace hepk {
namespace dev {

// Small histograms: every LANE of every warp owns a private copy of the bins (cell [warp][slot][lane], so a warp's 32
// updates fall into 32 different banks whatever the slots are): no atomics, no same-bin or bank conflicts, and a lane's
// float32 partial sum covers only n / (threads of the grid) entries.  The copies are added up in float64 at the end of
// the CTA and merged into the caller's arrays with one atomic per slot.
// MODE 0: counts only (also serves the sums when there are no weights: w = 1), 1: sumw only, 2: sumw and counts (8-byte
// cells), 3: sumw, sumw2 and counts (16-byte cells).
// Where the result goes: ACC false -> float atomics on the caller's sumw and 64-bit integer atomics on counts
// (hepk_fill_histogram); ACC true -> float64 / int64 atomics on the rows of a workspace that a finalize kernel adds to
// the caller's arrays (hepk_fill_histogram_w2: rows of WS words, columns 0 = sumw, col_w2, col_cnt; -1 = absent).
struct LaneHistOut {
    float* sumw;
    unsigned long long* counts;
    long long* acc;
    int WS, want_sumw, col_w2, col_cnt;
    // ACC only: the CTA that finishes last adds the rows to the caller's arrays itself (float32(float64(old) + sum);
    // counts +=), which saves the launch of a finalize kernel behind a 25-40 us fill.  `done` counts finished CTAs (a
    // zeroed word of the workspace); nullptr: the caller runs the finalize kernel.
    unsigned int* done;
    float *fin_sumw, *fin_sumw2;
    long long* fin_counts;
};

template <int MODE> struct LaneCell { using type = unsigned int; };
template <> struct LaneCell<2> { using type = uint2; };
template <> struct LaneCell<3> { using type = uint4; };

template <int MODE, bool VEC, bool ACC>
__global__ void __launch_bounds__(256, 1) fill_hist_lanes_kernel(const float* __restrict__ data, const float* __restrict__ weights,
                                                                 long long n, const float* __restrict__ edges, int nbins,
                                                                 const LaneHistOut o)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    using Cell = typename LaneCell<MODE>::type;
    // s_pad[0] = -inf, s_pad[1 + i] = edges[i], s_pad[nbins + 2] = NaN (nothing, not even +inf, is >= it): slot s holds
    // s_pad[s] <= x < s_pad[s + 1]
    float* s_pad = (float*)smem_raw;
    float* s_edges = s_pad + 1;
    const int ns = nbins + 2, nwarps = blockDim.x >> 5;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const float4 one4 = make_float4(1.f, 1.f, 1.f, 1.f);
    const long long n4 = n / 4;
    const float4* d4 = (const float4*)data;
    const float4* w4 = (const float4*)weights;
    // The first three batches are requested before anything else: the set-up below (clearing ~200 KB of shared memory,
    // classifying the axis) then runs under the first DRAM round trip instead of in front of it.
    float4 xa[4], wa[4], xb[4], wb[4], xc[4], wc[4];
    long long gf = t0;                                    // first group of the next batch to fetch
    auto try_fetch = [&](float4 (&x)[4], float4 (&w)[4]) {
        if (!VEC || gf + 3 * stride >= n4) return false;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            x[k] = __ldg(d4 + gf + k * stride);
            w[k] = MODE != 0 ? __ldg(w4 + gf + k * stride) : one4;
        }
        gf += 4 * stride;
        return true;
    };
    bool va = try_fetch(xa, wa), vb = try_fetch(xb, wb), vc = try_fetch(xc, wc);
    // the padded edges once more with a copy per lane ([slot][lane]: the +-1 step's two loads hit 32 different banks,
    // where 32 lanes reading 32 different words of one copy would conflict 3-4 ways)
    float* s_rep = (float*)(smem_raw + (((size_t)(nbins + 3) * 4 + 15) & ~(size_t)15));
    Cell* cells = (Cell*)(s_rep + (size_t)(nbins + 3) * 32);
    for (int i = threadIdx.x; i <= nbins; i += blockDim.x) s_edges[i] = edges[i];
    if (threadIdx.x == 0) { s_pad[0] = -CUDART_INF_F; s_pad[nbins + 2] = CUDART_NAN_F; }
    {
        uint4* z = (uint4*)cells;
        const int nz = (int)((size_t)nwarps * ns * 32 * sizeof(Cell) / 16);
        for (int i = threadIdx.x; i < nz; i += blockDim.x) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    __syncthreads();
    for (int i = threadIdx.x; i < (nbins + 3) * 32; i += blockDim.x) s_rep[i] = s_pad[i >> 5];
    const AxisGuess ax = classify_axis(s_edges, nbins);          // (its barriers also publish s_rep)
    Cell* mine = cells + (size_t)(threadIdx.x >> 5) * ns * 32 + (threadIdx.x & 31);
    const float* my_pad = s_rep + (threadIdx.x & 31);
    const float top = (float)(nbins + 1);
    auto run = [&](auto axis_tag) {
    constexpr int AXIS = decltype(axis_tag)::value;       // 0: search, 1: uniform in x, 2: uniform in log2 x
    auto slot_of = [&](float v) {
        if (AXIS == 0) {
            int s = 1 + find_bin_clamped(v, s_edges, nbins);
            s = (v < s_edges[0]) ? 0 : s;
            return !(v < s_edges[nbins]) ? nbins + 1 : s;
        }
        // arithmetic guess in slot units, good to +-1 (classify_axis), then one step against the padded edges.
        // NaN: fminf(NaN, top) = top, and no comparison moves it -> overflow slot.
        float pos;
        if (AXIS == 1) pos = fmaf(v - ax.lo, ax.inv, 1.0f);
        else pos = v > 0.0f ? fmaf(__log2f(v) - ax.lo, ax.inv, 1.0f) : (v != v ? top : 0.0f);
        int s = (int)fmaxf(fminf(pos, top), 0.0f);
        const float e0 = my_pad[s * 32], e1 = my_pad[s * 32 + 32];
        s += (v >= e1) ? 1 : 0;
        s -= (v < e0) ? 1 : 0;
        return s;
    };
    auto update = [&](int s, float wv) {
        Cell* c = mine + s * 32;
        if (MODE == 0) *(unsigned int*)c += 1u;
        else if (MODE == 1) *(float*)c += wv;
        else if (MODE == 2) { uint2 v = *(uint2*)c; v.x = __float_as_uint(__uint_as_float(v.x) + wv); v.y += 1u; *(uint2*)c = v; }
        else {
            uint4 v = *(uint4*)c;
            v.x = __float_as_uint(__uint_as_float(v.x) + wv);
            v.y = __float_as_uint(fmaf(wv, wv, __uint_as_float(v.y)));
            v.z += 1u;
            *(uint4*)c = v;
        }
    };
    // Four updates with their loads issued together (one shared-memory round trip instead of four; used where few warps
    // fit and that latency is exposed): an entry whose slot equals an earlier one of the four takes that entry's new
    // value instead of what it loaded, and the stores go out in order, so the last store to a slot carries all of its
    // entries, added in the same order as one by one.
    auto update4 = [&](int s0, int s1, int s2, int s3, float w0, float w1, float w2, float w3) {
        if constexpr (MODE != 3) {
            update(s0, w0); update(s1, w1); update(s2, w2); update(s3, w3);
        } else {
            uint4 *c0 = mine + s0 * 32, *c1 = mine + s1 * 32, *c2 = mine + s2 * 32, *c3 = mine + s3 * 32;
            uint4 v0 = *c0, v1 = *c1, v2 = *c2, v3 = *c3;
            auto bump = [&](uint4 v, float wv) {
                v.x = __float_as_uint(__uint_as_float(v.x) + wv);
                v.y = __float_as_uint(fmaf(wv, wv, __uint_as_float(v.y)));
                v.z += 1u;
                return v;
            };
            auto pick = [&](bool c, const uint4& a, const uint4& b) { return make_uint4(c ? a.x : b.x, c ? a.y : b.y, c ? a.z : b.z, 0u); };
            const uint4 n0 = bump(v0, w0);
            v1 = pick(s1 == s0, n0, v1);
            const uint4 n1 = bump(v1, w1);
            v2 = pick(s2 == s1, n1, pick(s2 == s0, n0, v2));
            const uint4 n2 = bump(v2, w2);
            v3 = pick(s3 == s2, n2, pick(s3 == s1, n1, pick(s3 == s0, n0, v3)));
            const uint4 n3 = bump(v3, w3);
            *c0 = n0; *c1 = n1; *c2 = n2; *c3 = n3;
        }
    };
    auto add4 = [&](const float4& x, const float4& w) {
        const int s0 = slot_of(x.x), s1 = slot_of(x.y), s2 = slot_of(x.z), s3 = slot_of(x.w);
        update(s0, w.x); update(s1, w.y); update(s2, w.z); update(s3, w.w);
    };
    // The slots of a batch are all found BEFORE its first update: the compiler must assume that an update may alias
    // the edges (both live in shared memory), so interleaving the two would serialise every edge load behind a store.
    auto add16 = [&](const float4 (&x)[4], const float4 (&w)[4]) {
        int sl[16];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            sl[4 * k] = slot_of(x[k].x); sl[4 * k + 1] = slot_of(x[k].y); sl[4 * k + 2] = slot_of(x[k].z); sl[4 * k + 3] = slot_of(x[k].w);
        }
#pragma unroll
        for (int k = 0; k < 4; ++k) update4(sl[4 * k], sl[4 * k + 1], sl[4 * k + 2], sl[4 * k + 3], w[k].x, w[k].y, w[k].z, w[k].w);
    };
    if (VEC) {
        // batches of 4 x 2 16-byte loads per thread in three register buffers: two batches are in flight while one is
        // filled (one CTA of <= 8 warps per SM: the loads in flight have to come from depth, not from occupancy)
        while (va) {
            add16(xa, wa); va = try_fetch(xa, wa);
            if (!vb) break;
            add16(xb, wb); vb = try_fetch(xb, wb);
            if (!vc) break;
            add16(xc, wc); vc = try_fetch(xc, wc);
        }
        for (long long g = gf; g < n4; g += stride) add4(__ldg(d4 + g), MODE != 0 ? __ldg(w4 + g) : one4);
        for (long long i = n4 * 4 + t0; i < n; i += stride) update(slot_of(data[i]), MODE != 0 ? weights[i] : 1.f);
    } else {
        for (long long i = t0; i < n; i += stride) update(slot_of(data[i]), MODE != 0 ? weights[i] : 1.f);
    }
    };
    if (ax.mode == 1) run(std::integral_constant<int, 1>{});
    else if (ax.mode == 2 && s_edges[0] >= 1.0e-30f) run(std::integral_constant<int, 2>{});
    else run(std::integral_constant<int, 0>{});
    __syncthreads();
    // merge: thread -> (slot, part); part p adds up the copies of warps p, p + parts, ...
    const int parts = ns * 4 <= (int)blockDim.x ? 4 : (ns * 2 <= (int)blockDim.x ? 2 : 1);
    for (int idx = threadIdx.x; idx < ns * parts; idx += blockDim.x) {
        const int s = idx % ns, part = idx / ns;
        double tot = 0.0, tot2 = 0.0;
        unsigned long long cnt = 0;
        for (int w = part; w < nwarps; w += parts) {
            const Cell* row = cells + ((size_t)w * ns + s) * 32;
#pragma unroll 8
            for (int j = 0; j < 32; ++j) {
                const Cell c = row[(j + threadIdx.x) & 31];          // rotated: the lanes of a warp read different banks
                if constexpr (MODE == 0) cnt += c;
                else if constexpr (MODE == 1) tot += (double)__uint_as_float(c);
                else if constexpr (MODE == 2) { tot += (double)__uint_as_float(c.x); cnt += c.y; }
                else { tot += (double)__uint_as_float(c.x); tot2 += (double)__uint_as_float(c.y); cnt += c.z; }
            }
        }
        if (MODE == 0) tot = tot2 = (double)cnt;
        if (ACC) {
            long long* row = o.acc + (long long)s * o.WS;
            if (o.want_sumw && tot != 0.0) atomicAdd((double*)row, tot);
            if (o.col_w2 >= 0 && tot2 != 0.0) atomicAdd((double*)(row + o.col_w2), tot2);
            if (o.col_cnt >= 0 && cnt) atomicAdd((unsigned long long*)(row + o.col_cnt), cnt);
        } else {
            if (o.sumw && tot != 0.0) atomicAdd(o.sumw + s, (float)tot);
            if (o.counts && cnt) atomicAdd(o.counts + s, cnt);
        }
    }
    if constexpr (ACC) {
        if (o.done) {
            __shared__ unsigned int s_last;
            __threadfence();                     // this thread's atomics on the rows are visible before the CTA reports in
            __syncthreads();
            if (threadIdx.x == 0) s_last = atomicAdd(o.done, 1u) == gridDim.x - 1 ? 1u : 0u;
            __syncthreads();
            if (s_last) {
                __threadfence();
                for (int s = threadIdx.x; s < ns; s += blockDim.x) {
                    const long long* row = o.acc + (long long)s * o.WS;
                    if (o.want_sumw && o.fin_sumw) o.fin_sumw[s] = (float)((double)o.fin_sumw[s] + __longlong_as_double(__ldcg(row)));
                    if (o.col_w2 >= 0) o.fin_sumw2[s] = (float)((double)o.fin_sumw2[s] + __longlong_as_double(__ldcg(row + o.col_w2)));
                    if (o.col_cnt >= 0) o.fin_counts[s] += __ldcg(row + o.col_cnt);
                }
            }
        }
    }
}


// shared memory of a launch with `warps` warps per CTA: padded edges, their per-lane copy, the cells
__host__ __device__ inline size_t lane_hist_head_bytes(int nbins)
{
    return (((size_t)(nbins + 3) * 4 + 15) & ~(size_t)15) + (size_t)(nbins + 3) * 128;
}
__host__ __device__ inline size_t lane_hist_warp_bytes(int nbins, int mode)
{
    return (size_t)(nbins + 2) * 32 * (mode == 3 ? 16 : (mode == 2 ? 8 : 4));
}

}  // namespace dev
}  // namespace hepk
