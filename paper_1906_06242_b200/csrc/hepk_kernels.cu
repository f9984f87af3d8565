// hepk_kernels.cu — the single kernels of include/hepk.h:
//   select_mask, lookup_binned, fill_histogram           (flat, 128-bit vectorised streaming)
//   segmented_reduce_{sum,max,min,count,argmax}          (warp-per-event and block-per-tile variants)
//   deltar_mask, pair_invmass                            (tiles of events staged through shared memory)
#include <string.h>

#include "hepk_common.cuh"

namespace hepk {
namespace dev {

// =========================================================================================== select_mask
// Vector path: one thread = 16 consecutive objects = 4+4 LDG.128 in flight and one STG.128 of mask bytes.
__global__ void __launch_bounds__(256) select_mask_vec(const float4* __restrict__ pt, const float4* __restrict__ eta,
                                                       long long n, float pt_min, float eta_max,
                                                       uint4* __restrict__ out)
{
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;   // group of 16
    const long long i0 = g * 16;
    if (i0 >= n) return;
    if (i0 + 16 <= n) {
        float4 p[4], e[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) p[k] = __ldg(pt + g * 4 + k);
        if (eta) {
#pragma unroll
            for (int k = 0; k < 4; ++k) e[k] = __ldg(eta + g * 4 + k);
        } else {
#pragma unroll
            for (int k = 0; k < 4; ++k) e[k] = make_float4(0.f, 0.f, 0.f, 0.f);
        }
        const float em = eta ? eta_max : CUDART_INF_F;
        unsigned int w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const unsigned int b0 = (p[k].x > pt_min && fabsf(e[k].x) < em) ? 1u : 0u;
            const unsigned int b1 = (p[k].y > pt_min && fabsf(e[k].y) < em) ? 1u : 0u;
            const unsigned int b2 = (p[k].z > pt_min && fabsf(e[k].z) < em) ? 1u : 0u;
            const unsigned int b3 = (p[k].w > pt_min && fabsf(e[k].w) < em) ? 1u : 0u;
            w[k] = b0 | (b1 << 8) | (b2 << 16) | (b3 << 24);
        }
        out[g] = make_uint4(w[0], w[1], w[2], w[3]);
    } else {
        const float* ps = (const float*)pt;
        const float* es = (const float*)eta;
        unsigned char* os = (unsigned char*)out;
        for (long long i = i0; i < n; ++i)
            os[i] = (ps[i] > pt_min && (!es || fabsf(es[i]) < eta_max)) ? 1 : 0;
    }
}

__global__ void __launch_bounds__(256) select_mask_scalar(const float* __restrict__ pt, const float* __restrict__ eta,
                                                          long long n, float pt_min, float eta_max,
                                                          unsigned char* __restrict__ out)
{
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x)
        out[i] = (pt[i] > pt_min && (!eta || fabsf(eta[i]) < eta_max)) ? 1 : 0;
}

// =========================================================================================== lookup_binned
// Edges and table staged in shared memory once per (persistent) CTA; 4 objects per thread per step.
template <bool VEC>
__global__ void __launch_bounds__(256) lookup_kernel(const float* __restrict__ x, const float* __restrict__ y, long long n,
                                                     const float* __restrict__ edges_x, int nx,
                                                     const float* __restrict__ edges_y, int ny,
                                                     const float* __restrict__ table, float* __restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_ex = (float*)smem_raw;
    float* s_ey = s_ex + (nx + 1);
    float* s_t = s_ey + (y ? ny + 1 : 0);
    const int nyy = y ? ny : 1;
    for (int i = threadIdx.x; i <= nx; i += blockDim.x) s_ex[i] = edges_x[i];
    if (y) for (int i = threadIdx.x; i <= ny; i += blockDim.x) s_ey[i] = edges_y[i];
    for (int i = threadIdx.x; i < nx * nyy; i += blockDim.x) s_t[i] = table[i];
    __syncthreads();
    const AxisGuess ax = classify_axis(s_ex, nx);
    AxisGuess ay;
    ay.mode = 0; ay.lo = 0.f; ay.inv = 0.f;
    if (y) ay = classify_axis(s_ey, ny);
    auto look = [&](float xv, float yv) {
        const int bx = find_bin_guess(xv, s_ex, nx, ax);
        const int by = y ? find_bin_guess(yv, s_ey, ny, ay) : 0;
        return s_t[bx * nyy + by];
    };
    const long long stride = (long long)gridDim.x * blockDim.x;
    if (VEC) {
        const long long n4 = n / 4;
        for (long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x; g < n4; g += stride) {
            const float4 xv = __ldg((const float4*)x + g);
            const float4 yv = y ? __ldg((const float4*)y + g) : make_float4(0.f, 0.f, 0.f, 0.f);
            float4 r;
            r.x = look(xv.x, yv.x); r.y = look(xv.y, yv.y); r.z = look(xv.z, yv.z); r.w = look(xv.w, yv.w);
            ((float4*)out)[g] = r;
        }
        for (long long i = n4 * 4 + (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            out[i] = look(x[i], y ? y[i] : 0.f);
    } else {
        for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += stride)
            out[i] = look(x[i], y ? y[i] : 0.f);
    }
}

// =========================================================================================== fill_histogram
// Per-CTA privatised bins in shared memory (float32 sums + uint32 counts), merged into the global arrays
// with atomics at the end of each chunk of CHUNK_ITERS grid-stride steps.
template <bool VEC>
__global__ void __launch_bounds__(256) fill_hist_kernel(const float* __restrict__ data, const float* __restrict__ weights,
                                                        long long n, const float* __restrict__ edges, int nbins,
                                                        float* __restrict__ sumw, unsigned long long* __restrict__ counts)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_edges = (float*)smem_raw;
    float* s_sumw = s_edges + (nbins + 1);
    unsigned int* s_cnt = (unsigned int*)(s_sumw + (nbins + 2));
    for (int i = threadIdx.x; i <= nbins; i += blockDim.x) s_edges[i] = edges[i];
    for (int i = threadIdx.x; i < nbins + 2; i += blockDim.x) { s_sumw[i] = 0.f; s_cnt[i] = 0u; }
    __syncthreads();
    const float lo = s_edges[0];
    const float inv_w = (float)nbins / (s_edges[nbins] - lo);
    auto add = [&](float xv, float wv) {
        const int s = hist_slot(xv, s_edges, nbins, lo, inv_w);
        if (sumw) red_shared_add_f32(&s_sumw[s], wv);
        if (counts) red_shared_add_u32(&s_cnt[s], 1u);
    };
    auto flush = [&]() {
        __syncthreads();
        for (int i = threadIdx.x; i < nbins + 2; i += blockDim.x) {
            if (sumw) { const float v = s_sumw[i]; if (v != 0.f) { atomicAdd(sumw + i, v); s_sumw[i] = 0.f; } }
            if (counts) { const unsigned int c = s_cnt[i]; if (c) { atomicAdd(counts + i, (unsigned long long)c); s_cnt[i] = 0u; } }
        }
        __syncthreads();
    };
    constexpr int CHUNK_ITERS = 32;
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (VEC) {
        const long long n4 = n / 4;
        const long long iters = (n4 + stride - 1) / stride;
        for (long long it = 0; it < iters; ++it) {
            const long long g = t0 + it * stride;
            if (g < n4) {
                const float4 xv = __ldg((const float4*)data + g);
                const float4 wv = weights ? __ldg((const float4*)weights + g) : make_float4(1.f, 1.f, 1.f, 1.f);
                add(xv.x, wv.x); add(xv.y, wv.y); add(xv.z, wv.z); add(xv.w, wv.w);
            }
            if ((it + 1) % CHUNK_ITERS == 0) flush();
        }
        for (long long i = n4 * 4 + t0; i < n; i += stride) add(data[i], weights ? weights[i] : 1.f);
    } else {
        const long long iters = (n + stride - 1) / stride;
        for (long long it = 0; it < iters; ++it) {
            const long long i = t0 + it * stride;
            if (i < n) add(data[i], weights ? weights[i] : 1.f);
            if ((it + 1) % (4 * CHUNK_ITERS) == 0) flush();
        }
    }
    flush();
}

// =========================================================================================== segmented reductions
enum { OP_SUM = 0, OP_MAX = 1, OP_MIN = 2, OP_COUNT = 3, OP_ARGMAX = 4 };

template <int OP> struct OutT { typedef float type; };
template <> struct OutT<OP_COUNT> { typedef int type; };
template <> struct OutT<OP_ARGMAX> { typedef int type; };

// Running state of one reduction.  push() follows the oracle's update rules; merge() combines partial
// states so that count / max / min / argmax do not depend on the order of combination.
template <int OP>
struct Acc {
    float v;
    int i;
    __device__ __forceinline__ void init()
    {
        v = OP == OP_MAX ? -CUDART_INF_F : (OP == OP_MIN ? CUDART_INF_F : 0.f);
        i = OP == OP_ARGMAX ? -1 : 0;
    }
    __device__ __forceinline__ void push(float x, int k)
    {
        if (OP == OP_SUM) v += x;
        else if (OP == OP_COUNT) i += 1;
        else if (OP == OP_MAX) { if (x > v) v = x; }
        else if (OP == OP_MIN) { if (x < v) v = x; }
        else { if (x == x && (i < 0 || x > v)) { v = x; i = k; } }     // k ascending within a thread
    }
    __device__ __forceinline__ void merge(float ov, int oi)
    {
        if (OP == OP_SUM) v += ov;
        else if (OP == OP_COUNT) i += oi;
        else if (OP == OP_MAX) { if (ov > v) v = ov; }
        else if (OP == OP_MIN) { if (ov < v) v = ov; }
        else { if (oi >= 0 && (i < 0 || ov > v || (ov == v && oi < i))) { v = ov; i = oi; } }
    }
    __device__ __forceinline__ typename OutT<OP>::type result() const
    {
        if (OP == OP_COUNT || OP == OP_ARGMAX) return (typename OutT<OP>::type)i;
        return (typename OutT<OP>::type)v;
    }
    __device__ __forceinline__ void warp_reduce()
    {
#pragma unroll
        for (int d = 16; d > 0; d >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, v, d);
            const int oi = __shfl_xor_sync(0xffffffffu, i, d);
            merge(ov, oi);
        }
    }
};

// Variant 1: one warp per event, lanes stride over the event's particles (coalesced), shuffle reduction.
template <int OP>
__global__ void __launch_bounds__(256) segreduce_warp_kernel(const float* __restrict__ data, const long long* __restrict__ offsets,
                                                             long long n_events, long long base,
                                                             const unsigned char* __restrict__ mask_rows,
                                                             const unsigned char* __restrict__ mask_content,
                                                             typename OutT<OP>::type* __restrict__ out)
{
    const int lane = threadIdx.x & 31;
    const long long warp0 = ((long long)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const long long nwarps = ((long long)gridDim.x * blockDim.x) >> 5;
    for (long long e = warp0; e < n_events; e += nwarps) {
        Acc<OP> acc;
        acc.init();
        if (!mask_rows || mask_rows[e]) {
            const long long g0 = offsets[e], g1 = offsets[e + 1];
            for (long long g = g0 + lane; g < g1; g += 32) {
                const long long i = g - base;
                if (mask_content && !mask_content[i]) continue;
                acc.push(OP == OP_COUNT ? 0.f : data[i], (int)(g - g0));
            }
        }
        acc.warp_reduce();
        if (lane == 0) out[e] = acc.result();
    }
}

// Variant 2: a tile of TILE events per step; the tile's data (and content-mask) slice is staged into shared
// memory by bulk copies, then one thread reduces one event; outputs are written coalesced.
template <int OP, int TILE>
__global__ void __launch_bounds__(TILE) segreduce_tile_kernel(const float* __restrict__ data, const long long* __restrict__ offsets,
                                                              long long n_events, long long base,
                                                              const unsigned char* __restrict__ mask_rows,
                                                              const unsigned char* __restrict__ mask_content,
                                                              typename OutT<OP>::type* __restrict__ out, int cap)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* bar = (uint64_t*)smem_raw;
    int* loc = (int*)(smem_raw + 16);
    float* s_data = (float*)(smem_raw + 16 + ((TILE + 1) * 4 + 15) / 16 * 16);
    unsigned char* s_mask = (unsigned char*)(s_data + cap);
    __shared__ float red_v[TILE / 32];
    __shared__ int red_i[TILE / 32];
    const int tid = threadIdx.x;
    const bool need_data = OP != OP_COUNT;
    if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
    __syncthreads();
    uint32_t parity = 0;
    const long long n_total = offsets[n_events] - base;
    const long long n_tiles = (n_events + TILE - 1) / TILE;
    const int capm = cap - 40;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long e0 = tile * TILE;
        const int ne = (int)((n_events - e0) < TILE ? (n_events - e0) : TILE);
        const long long gb = offsets[e0];
        for (int i = tid; i <= ne; i += TILE) loc[i] = (int)(offsets[e0 + i] - gb);
        __syncthreads();
        int ev0 = 0;
        while (ev0 < ne) {
            const int b = loc[ev0];
            int n_fit;
            if (loc[ne] - b <= capm) n_fit = ne - ev0;
            else n_fit = __syncthreads_count(tid >= ev0 && tid < ne && loc[tid + 1] - b <= capm);
            if (n_fit == 0) {
                // one event larger than the buffer: the whole CTA strides over it in global memory
                const long long e = e0 + ev0;
                Acc<OP> acc;
                acc.init();
                if (!mask_rows || mask_rows[e]) {
                    const long long g0 = gb + b, g1 = gb + loc[ev0 + 1];
                    for (long long g = g0 + tid; g < g1; g += TILE) {
                        const long long i = g - base;
                        if (mask_content && !mask_content[i]) continue;
                        acc.push(need_data ? data[i] : 0.f, (int)(g - g0));
                    }
                }
                acc.warp_reduce();
                if ((tid & 31) == 0) { red_v[tid >> 5] = acc.v; red_i[tid >> 5] = acc.i; }
                __syncthreads();
                if (tid == 0) {
                    Acc<OP> t;
                    t.v = red_v[0]; t.i = red_i[0];
                    for (int w = 1; w < TILE / 32; ++w) t.merge(red_v[w], red_i[w]);
                    out[e] = t.result();
                }
                ev0 += 1;
                __syncthreads();
                continue;
            }
            const int ev1 = ev0 + n_fit;
            const int nd = loc[ev1] - b;
            const long long l0 = gb + b - base;
            long long a0;
            int sh_d = 0, sh_m = 0;
            uint32_t bytes = 0;
            if (tid == 0) fence_proxy_async_smem();
            if (need_data) { bytes += stage_column(s_data, data, l0, l0 + nd, n_total, bar, tid, 0, &a0); sh_d = (int)(l0 - a0); }
            if (mask_content) { bytes += stage_column(s_mask, mask_content, l0, l0 + nd, n_total, bar, tid, 0, &a0); sh_m = (int)(l0 - a0); }
            if (tid == 0) mbar_arrive_expect_tx(bar, bytes);
            mbar_wait(bar, parity);
            parity ^= 1u;
            __syncthreads();
            if (tid < n_fit) {
                const long long e = e0 + ev0 + tid;
                Acc<OP> acc;
                acc.init();
                if (!mask_rows || mask_rows[e]) {
                    const int k0 = loc[ev0 + tid] - b, k1 = loc[ev0 + tid + 1] - b;
                    for (int k = k0; k < k1; ++k) {
                        if (mask_content && !s_mask[k + sh_m]) continue;
                        acc.push(need_data ? s_data[k + sh_d] : 0.f, k - k0);
                    }
                }
                out[e] = acc.result();
            }
            fence_proxy_async_smem();
            __syncthreads();
            ev0 = ev1;
        }
    }
}

// =========================================================================================== deltar_mask
template <int TILE>
__global__ void __launch_bounds__(TILE) deltar_tile_kernel(const float* __restrict__ eta1, const float* __restrict__ phi1,
                                                           const long long* __restrict__ off1, long long base1,
                                                           const unsigned char* __restrict__ sel1,
                                                           const float* __restrict__ eta2, const float* __restrict__ phi2,
                                                           const long long* __restrict__ off2, long long base2,
                                                           const unsigned char* __restrict__ sel2,
                                                           long long n_events, float dr2_max,
                                                           unsigned char* __restrict__ out, int cap1, int cap2)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* bar = (uint64_t*)smem_raw;
    int* loc1 = (int*)(smem_raw + 16);
    int* loc2 = loc1 + (TILE + 1);
    unsigned char* p = smem_raw + 16 + (2 * (TILE + 1) * 4 + 15) / 16 * 16;
    float* s_eta1 = (float*)p; p += (size_t)cap1 * 4;
    float* s_phi1 = (float*)p; p += (size_t)cap1 * 4;
    float* s_eta2 = (float*)p; p += (size_t)cap2 * 4;
    float* s_phi2 = (float*)p; p += (size_t)cap2 * 4;
    unsigned short* evid = (unsigned short*)p; p += (size_t)cap1 * 2;
    unsigned char* s_sel1 = p; p += cap1;
    unsigned char* s_sel2 = p;
    const int tid = threadIdx.x;
    if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
    __syncthreads();
    uint32_t parity = 0;
    const long long n1 = off1[n_events] - base1, n2 = off2[n_events] - base2;
    const long long n_tiles = (n_events + TILE - 1) / TILE;
    const int c1 = cap1 - 40, c2 = cap2 - 40;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long e0 = tile * TILE;
        const int ne = (int)((n_events - e0) < TILE ? (n_events - e0) : TILE);
        const long long gb1 = off1[e0], gb2 = off2[e0];
        for (int i = tid; i <= ne; i += TILE) { loc1[i] = (int)(off1[e0 + i] - gb1); loc2[i] = (int)(off2[e0 + i] - gb2); }
        __syncthreads();
        int ev0 = 0;
        while (ev0 < ne) {
            const int b1 = loc1[ev0], b2 = loc2[ev0];
            int n_fit;
            if (loc1[ne] - b1 <= c1 && loc2[ne] - b2 <= c2) n_fit = ne - ev0;
            else n_fit = __syncthreads_count(tid >= ev0 && tid < ne && loc1[tid + 1] - b1 <= c1 && loc2[tid + 1] - b2 <= c2);
            if (n_fit == 0) {
                // one event larger than the buffers: the CTA strides over its collection-1 objects in global memory
                const long long g0 = gb1 + b1, g1 = gb1 + loc1[ev0 + 1];
                const long long h0 = gb2 + b2, h1 = gb2 + loc2[ev0 + 1];
                for (long long g = g0 + tid; g < g1; g += TILE) {
                    const long long j = g - base1;
                    bool matched = false;
                    if (!sel1 || sel1[j]) {
                        const float eta = eta1[j], phi = phi1[j];
                        for (long long h = h0; h < h1 && !matched; ++h) {
                            const long long m = h - base2;
                            if (sel2 && !sel2[m]) continue;
                            matched = dr2_exact(eta, phi, eta2[m], phi2[m]) < dr2_max;
                        }
                    }
                    out[j] = matched ? 1 : 0;
                }
                ev0 += 1;
                __syncthreads();
                continue;
            }
            const int ev1 = ev0 + n_fit;
            const int na = loc1[ev1] - b1, nb = loc2[ev1] - b2;
            const long long l1 = gb1 + b1 - base1, l2 = gb2 + b2 - base2;
            long long a0;
            int sh_e1, sh_p1, sh_e2, sh_p2, sh_s1 = 0, sh_s2 = 0;
            uint32_t bytes = 0;
            if (tid == 0) fence_proxy_async_smem();
            bytes += stage_column(s_eta1, eta1, l1, l1 + na, n1, bar, tid, 0, &a0); sh_e1 = (int)(l1 - a0);
            bytes += stage_column(s_phi1, phi1, l1, l1 + na, n1, bar, tid, 0, &a0); sh_p1 = (int)(l1 - a0);
            bytes += stage_column(s_eta2, eta2, l2, l2 + nb, n2, bar, tid, 0, &a0); sh_e2 = (int)(l2 - a0);
            bytes += stage_column(s_phi2, phi2, l2, l2 + nb, n2, bar, tid, 0, &a0); sh_p2 = (int)(l2 - a0);
            if (sel1) { bytes += stage_column(s_sel1, sel1, l1, l1 + na, n1, bar, tid, 0, &a0); sh_s1 = (int)(l1 - a0); }
            if (sel2) { bytes += stage_column(s_sel2, sel2, l2, l2 + nb, n2, bar, tid, 0, &a0); sh_s2 = (int)(l2 - a0); }
            if (tid == 0) mbar_arrive_expect_tx(bar, bytes);
            if (tid < n_fit) {
                const int k0 = loc1[ev0 + tid] - b1, k1 = loc1[ev0 + tid + 1] - b1;
                for (int k = k0; k < k1; ++k) evid[k] = (unsigned short)tid;
            }
            mbar_wait(bar, parity);
            parity ^= 1u;
            __syncthreads();
            if (sel2) {   // unselected objects of collection 2 never match: NaN eta
                for (int m = tid; m < nb; m += TILE)
                    if (!s_sel2[m + sh_s2]) s_eta2[m + sh_e2] = CUDART_NAN_F;
                __syncthreads();
            }
            for (int j = tid; j < na; j += TILE) {
                bool matched = false;
                if (!sel1 || s_sel1[j + sh_s1]) {
                    const float eta = s_eta1[j + sh_e1], phi = s_phi1[j + sh_p1];
                    const int a = ev0 + (int)evid[j];
                    const int m0 = loc2[a] - b2, m1 = loc2[a + 1] - b2;
                    for (int m = m0; m < m1; ++m)
                        matched |= dr2_exact(eta, phi, s_eta2[m + sh_e2], s_phi2[m + sh_p2]) < dr2_max;
                }
                out[l1 + j] = matched ? 1 : 0;
            }
            fence_proxy_async_smem();
            __syncthreads();
            ev0 = ev1;
        }
    }
}

// =========================================================================================== pair_invmass
template <int TILE>
__global__ void __launch_bounds__(TILE) invmass_tile_kernel(const float* __restrict__ pt, const float* __restrict__ eta,
                                                            const float* __restrict__ phi, const float* __restrict__ mass,
                                                            const long long* __restrict__ offsets, long long n_events, long long base,
                                                            const unsigned char* __restrict__ mask,
                                                            float* __restrict__ out_mass, int* __restrict__ out_i1,
                                                            int* __restrict__ out_i2, int cap)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    uint64_t* bar = (uint64_t*)smem_raw;
    int* loc = (int*)(smem_raw + 16);
    unsigned char* p = smem_raw + 16 + ((TILE + 1) * 4 + 15) / 16 * 16;
    float* s_pt = (float*)p; p += (size_t)cap * 4;
    float* s_eta = (float*)p; p += (size_t)cap * 4;
    float* s_phi = (float*)p; p += (size_t)cap * 4;
    float* s_mass = (float*)p; p += (size_t)cap * 4;
    unsigned char* s_mask = p;
    const int tid = threadIdx.x;
    if (tid == 0) { mbar_init(bar, 1); fence_mbar_init(); }
    __syncthreads();
    uint32_t parity = 0;
    const long long n_total = offsets[n_events] - base;
    const long long n_tiles = (n_events + TILE - 1) / TILE;
    const int capm = cap - 40;
    for (long long tile = blockIdx.x; tile < n_tiles; tile += gridDim.x) {
        const long long e0 = tile * TILE;
        const int ne = (int)((n_events - e0) < TILE ? (n_events - e0) : TILE);
        const long long gb = offsets[e0];
        for (int i = tid; i <= ne; i += TILE) loc[i] = (int)(offsets[e0 + i] - gb);
        __syncthreads();
        int ev0 = 0;
        while (ev0 < ne) {
            const int b = loc[ev0];
            int n_fit;
            if (loc[ne] - b <= capm) n_fit = ne - ev0;
            else n_fit = __syncthreads_count(tid >= ev0 && tid < ne && loc[tid + 1] - b <= capm);
            if (n_fit == 0) {
                // one event larger than the buffers: one thread, the paper's loop shape, global memory
                if (tid == 0) {
                    const long long e = e0 + ev0, g0 = gb + b, g1 = gb + loc[ev0 + 1];
                    Top2 top;
                    top.init();
                    for (long long g = g0; g < g1; ++g) {
                        const long long i = g - base;
                        if (mask && !mask[i]) continue;
                        top.push_any(pt[i], (int)(g - g0));
                    }
                    float m = 0.f;
                    if (top.i2 >= 0) {
                        const long long a = g0 - base + top.i1, c = g0 - base + top.i2;
                        m = pair_mass_f32(top.b1, eta[a], phi[a], mass[a], top.b2, eta[c], phi[c], mass[c]);
                    }
                    out_mass[e] = m;
                    if (out_i1) out_i1[e] = top.i1;
                    if (out_i2) out_i2[e] = top.i2;
                }
                ev0 += 1;
                __syncthreads();
                continue;
            }
            const int ev1 = ev0 + n_fit;
            const int nd = loc[ev1] - b;
            const long long l0 = gb + b - base;
            long long a0;
            int sh_pt, sh_eta, sh_phi, sh_mass, sh_m = 0;
            uint32_t bytes = 0;
            if (tid == 0) fence_proxy_async_smem();
            bytes += stage_column(s_pt, pt, l0, l0 + nd, n_total, bar, tid, 0, &a0);     sh_pt = (int)(l0 - a0);
            bytes += stage_column(s_eta, eta, l0, l0 + nd, n_total, bar, tid, 0, &a0);   sh_eta = (int)(l0 - a0);
            bytes += stage_column(s_phi, phi, l0, l0 + nd, n_total, bar, tid, 0, &a0);   sh_phi = (int)(l0 - a0);
            bytes += stage_column(s_mass, mass, l0, l0 + nd, n_total, bar, tid, 0, &a0); sh_mass = (int)(l0 - a0);
            if (mask) { bytes += stage_column(s_mask, mask, l0, l0 + nd, n_total, bar, tid, 0, &a0); sh_m = (int)(l0 - a0); }
            if (tid == 0) mbar_arrive_expect_tx(bar, bytes);
            mbar_wait(bar, parity);
            parity ^= 1u;
            __syncthreads();
            if (tid < n_fit) {
                const long long e = e0 + ev0 + tid;
                const int k0 = loc[ev0 + tid] - b, k1 = loc[ev0 + tid + 1] - b;
                Top2 top;
                top.init();
                for (int k = k0; k < k1; ++k) {
                    if (mask && !s_mask[k + sh_m]) continue;
                    top.push_any(s_pt[k + sh_pt], k - k0);
                }
                float m = 0.f;
                if (top.i2 >= 0) {
                    const int a = k0 + top.i1, c = k0 + top.i2;
                    m = pair_mass_f32(top.b1, s_eta[a + sh_eta], s_phi[a + sh_phi], s_mass[a + sh_mass],
                                      top.b2, s_eta[c + sh_eta], s_phi[c + sh_phi], s_mass[c + sh_mass]);
                }
                out_mass[e] = m;
                if (out_i1) out_i1[e] = top.i1;
                if (out_i2) out_i2[e] = top.i2;
            }
            fence_proxy_async_smem();
            __syncthreads();
            ev0 = ev1;
        }
    }
}

}  // namespace dev

// ------------------------------------------------------------------------------------------ host helpers
static int persistent_grid(const void* kern, int block, size_t smem, long long work_items)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, block, smem) != cudaSuccess || occ < 1) occ = 1;
    long long g = (long long)sm_count() * occ;
    if (g > work_items) g = work_items;
    return (int)(g < 1 ? 1 : g);
}

template <int OP>
static int32_t segreduce_dispatch(const float* data, const int64_t* offsets, int64_t n_events, int64_t base,
                                  const uint8_t* mask_rows, const uint8_t* mask_content, void* out, int32_t variant,
                                  void* stream)
{
    typedef typename dev::OutT<OP>::type T;
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(variant >= 0 && variant <= 2, "unknown variant");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out, "offsets/out is NULL");
    HEPK_REQUIRE(OP == dev::OP_COUNT || data, "data is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (variant == HEPK_VARIANT_WARP_PER_EVENT) {
        auto kern = dev::segreduce_warp_kernel<OP>;
        const long long warps = n_events;
        long long blocks = (warps + 7) / 8;
        const long long maxb = (long long)sm_count() * 32;
        if (blocks > maxb) blocks = maxb;
        kern<<<(unsigned)blocks, 256, 0, st>>>(data, (const long long*)offsets, n_events, base, mask_rows, mask_content, (T*)out); count_launch();
    } else {
        constexpr int TILE = 128;
        const int cap = 2560;
        auto kern = dev::segreduce_tile_kernel<OP, TILE>;
        const size_t smem = 16 + ((TILE + 1) * 4 + 15) / 16 * 16 + (size_t)cap * 4 + cap + 16;
        const int grid = persistent_grid((const void*)kern, TILE, smem, (n_events + TILE - 1) / TILE);
        kern<<<grid, TILE, smem, st>>>(data, (const long long*)offsets, n_events, base, mask_rows, mask_content, (T*)out, cap); count_launch();
    }
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

}  // namespace hepk

using namespace hepk;

extern "C" int32_t hepk_select_mask(const float* pt, const float* eta, int64_t n, float pt_min, float abs_eta_max,
                                    uint8_t* out_mask, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    if (n == 0) return HEPK_OK;
    HEPK_REQUIRE(pt && out_mask, "pt/out_mask is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    if (aligned16(pt) && aligned16(out_mask) && (!eta || aligned16(eta))) {
        const long long groups = (n + 15) / 16;
        dev::select_mask_vec<<<(unsigned)((groups + 255) / 256), 256, 0, st>>>((const float4*)pt, (const float4*)eta, n, pt_min,
                                                                               abs_eta_max, (uint4*)out_mask); count_launch();
    } else {
        long long blocks = (n + 255) / 256;
        const long long maxb = (long long)sm_count() * 16;
        if (blocks > maxb) blocks = maxb;
        dev::select_mask_scalar<<<(unsigned)blocks, 256, 0, st>>>(pt, eta, n, pt_min, abs_eta_max, out_mask); count_launch();
    }
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_lookup_binned(const float* x, const float* y, int64_t n, const float* edges_x, int32_t nx,
                                      const float* edges_y, int32_t ny, const float* table, float* out, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges_x && table && nx >= 1, "edges_x/table is NULL or nx < 1");
    HEPK_REQUIRE(!y || (edges_y && ny >= 1), "edges_y is NULL or ny < 1");
    if (n == 0) return HEPK_OK;
    HEPK_REQUIRE(x && out, "x/out is NULL");
    const size_t smem = ((size_t)(nx + 1) + (y ? ny + 1 : 0) + (size_t)nx * (y ? ny : 1)) * 4;
    if (smem > 200 * 1024) {
        set_error("hepk_lookup_binned: table of %zu bytes does not fit shared memory", smem);
        return HEPK_ERR_UNSUPPORTED;
    }
    cudaStream_t st = (cudaStream_t)stream;
    const bool vec = aligned16(x) && aligned16(out) && (!y || aligned16(y));
    auto kern = vec ? dev::lookup_kernel<true> : dev::lookup_kernel<false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = persistent_grid((const void*)kern, 256, smem, (n + 1023) / 1024);
    kern<<<grid, 256, smem, st>>>(x, y, n, edges_x, nx, edges_y, ny, table, out); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_fill_histogram(const float* data, const float* weights, int64_t n, const float* edges, int32_t nbins,
                                       float* sumw, int64_t* counts, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges && nbins >= 1, "edges is NULL or nbins < 1");
    if (nbins + 2 > 16384) {
        set_error("hepk_fill_histogram: nbins+2 = %d exceeds 16384", nbins + 2);
        return HEPK_ERR_UNSUPPORTED;
    }
    if (n == 0 || (!sumw && !counts)) return HEPK_OK;
    HEPK_REQUIRE(data, "data is NULL");
    const size_t smem = ((size_t)(nbins + 1) + 2 * (size_t)(nbins + 2)) * 4;
    cudaStream_t st = (cudaStream_t)stream;
    const bool vec = aligned16(data) && (!weights || aligned16(weights));
    auto kern = vec ? dev::fill_hist_kernel<true> : dev::fill_hist_kernel<false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = persistent_grid((const void*)kern, 256, smem, (n + 1023) / 1024);
    kern<<<grid, 256, smem, st>>>(data, weights, n, edges, nbins, sumw, (unsigned long long*)counts); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

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
    constexpr int TILE = 128;
    const int cap1 = 2560, cap2 = 1024;
    const size_t smem = 16 + (2 * (TILE + 1) * 4 + 15) / 16 * 16 + (size_t)cap1 * (8 + 2 + 1) + (size_t)cap2 * (8 + 1) + 16;
    auto kern = dev::deltar_tile_kernel<TILE>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = persistent_grid((const void*)kern, TILE, smem, (n_events + TILE - 1) / TILE);
    const float dr2_max = dr_max * dr_max;      // float32 product (exact class)
    kern<<<grid, TILE, smem, (cudaStream_t)stream>>>(eta1, phi1, (const long long*)offsets1, base1, sel1, eta2, phi2,
                                                     (const long long*)offsets2, base2, sel2, n_events, dr2_max,
                                                     out_matched, cap1, cap2); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_pair_invmass(const float* pt, const float* eta, const float* phi, const float* mass,
                                     const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_content,
                                     float* out_mass, int32_t* out_i1, int32_t* out_i2, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out_mass, "offsets/out_mass is NULL");
    constexpr int TILE = 128;
    const int cap = 2560;
    const size_t smem = 16 + ((TILE + 1) * 4 + 15) / 16 * 16 + (size_t)cap * 17 + 16;
    auto kern = dev::invmass_tile_kernel<TILE>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = persistent_grid((const void*)kern, TILE, smem, (n_events + TILE - 1) / TILE);
    kern<<<grid, TILE, smem, (cudaStream_t)stream>>>(pt, eta, phi, mass, (const long long*)offsets, n_events, content_base,
                                                     mask_content, out_mass, out_i1, out_i2, cap); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}
