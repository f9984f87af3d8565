// hepk_kernels.cu — the flat single kernels of include/hepk.h: select_mask, lookup_binned, fill_histogram
// (128-bit vectorised streaming).  The kernels that walk jagged collections are in hepk_tiles.cu.
#include <string.h>

#include "hepk_common.cuh"
#include "hepk_hist_lanes.cuh"

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
    float* s_px = s_t + nx * nyy;              // padded copies of the edges (pad_axis_find, bin form)
    float* s_py = s_px + (nx + 1);
    for (int i = threadIdx.x; i <= nx; i += blockDim.x) s_ex[i] = edges_x[i];
    if (y) for (int i = threadIdx.x; i <= ny; i += blockDim.x) s_ey[i] = edges_y[i];
    for (int i = threadIdx.x; i < nx * nyy; i += blockDim.x) s_t[i] = table[i];
    pad_axis_fill<false>(s_px, edges_x, nx);
    if (y) pad_axis_fill<false>(s_py, edges_y, ny);
    __syncthreads();
    const AxisGuess ax = classify_axis(s_ex, nx);
    AxisGuess ay;
    ay.mode = 1; ay.lo = 0.f; ay.inv = 0.f;
    if (y) ay = classify_axis(s_ey, ny);
    const float top_x = (float)(nx - 1), top_y = (float)(ny - 1);
    const long long stride = (long long)gridDim.x * blockDim.x;
    dispatch_axes(ax.mode, ay.mode, [&](auto tx, auto ty) {
        constexpr int AX = decltype(tx)::value, AY = decltype(ty)::value;
        auto look = [&](float xv, float yv) {
            const int bx = pad_axis_find<AX, false>(xv, s_ex, s_px, nx, ax, top_x);
            const int by = y ? pad_axis_find<AY, false>(yv, s_ey, s_py, ny, ay, top_y) : 0;
            return s_t[bx * nyy + by];
        };
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
    });
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
    const size_t smem = (2 * (size_t)(nx + 1) + (y ? 2 * (size_t)(ny + 1) : 0) + (size_t)nx * (y ? ny : 1)) * 4;
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
    cudaStream_t st = (cudaStream_t)stream;
    const bool vec = aligned16(data) && (!weights || aligned16(weights));
    {
        // lane-private bins when 4-8 warps' worth of copies fit one SM's shared memory
        const int mode = !weights ? 0 : (counts ? (sumw ? 2 : 0) : 1);
        const size_t head = dev::lane_hist_head_bytes(nbins), per_warp = dev::lane_hist_warp_bytes(nbins, mode);
        int warps = (size_t)max_smem_optin() > head ? (int)(((size_t)max_smem_optin() - head) / per_warp) : 0;
        if (warps > 8) warps = 8;
        if (warps >= 4 && n >= (1 << 16) && n < (1ll << 40)) {
            void (*k)(const float*, const float*, long long, const float*, int, dev::LaneHistOut);
            if (mode == 0) k = vec ? dev::fill_hist_lanes_kernel<0, true, false> : dev::fill_hist_lanes_kernel<0, false, false>;
            else if (mode == 1) k = vec ? dev::fill_hist_lanes_kernel<1, true, false> : dev::fill_hist_lanes_kernel<1, false, false>;
            else k = vec ? dev::fill_hist_lanes_kernel<2, true, false> : dev::fill_hist_lanes_kernel<2, false, false>;
            const size_t sm = head + (size_t)warps * per_warp;
            dev::LaneHistOut o;
            o.sumw = sumw; o.counts = (unsigned long long*)counts; o.acc = nullptr;
            o.WS = 0; o.want_sumw = 0; o.col_w2 = -1; o.col_cnt = -1;
            o.done = nullptr; o.fin_sumw = nullptr; o.fin_sumw2 = nullptr; o.fin_counts = nullptr;
            HEPK_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            k<<<sm_count(), warps * 32, sm, st>>>(data, weights, n, edges, nbins, o); count_launch();
            HEPK_CUDA_TRY(cudaGetLastError());
            return HEPK_OK;
        }
    }
    const size_t smem = ((size_t)(nbins + 1) + 2 * (size_t)(nbins + 2)) * 4;
    auto kern = vec ? dev::fill_hist_kernel<true> : dev::fill_hist_kernel<false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const int grid = persistent_grid((const void*)kern, 256, smem, (n + 1023) / 1024);
    kern<<<grid, 256, smem, st>>>(data, weights, n, edges, nbins, sumw, (unsigned long long*)counts); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}
