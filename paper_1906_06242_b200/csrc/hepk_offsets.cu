// hepk_offsets.cu — the remaining generic kernels of the paper's list (include/hepk.h):
// hepk_get_in_offsets, hepk_set_in_offsets and hepk_select_opposite_sign.
//
// All three touch one or two elements per event, so they are bound by the offsets stream (8 B/event, coalesced)
// plus one 32-byte sector per touched element; one thread per event (the paper's own loop shape, Listing 1) is
// the right mapping: there is no per-event work to spread over lanes unless a content mask forces a scan, and
// then the scan is the event's few objects.
#include "hepk_common.cuh"

namespace hepk {
namespace dev {

// column index of the index-th counted element of the event, or -1
__device__ __forceinline__ long long nth_position(long long g0, long long g1, long long base,
                                                  const unsigned char* __restrict__ mask_content, int index)
{
    if (!mask_content) return (g1 - g0 > index) ? g0 + index - base : -1;
    int seen = 0;
    for (long long g = g0; g < g1; ++g) {
        if (!mask_content[g - base]) continue;
        if (seen == index) return g - base;
        ++seen;
    }
    return -1;
}

__global__ void get_in_offsets_kernel(const float* __restrict__ data, const long long* __restrict__ offsets, long long n_events,
                                      long long base, const unsigned char* __restrict__ mask_rows,
                                      const unsigned char* __restrict__ mask_content, int index, float fill,
                                      float* __restrict__ out)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_events; e += (long long)gridDim.x * blockDim.x) {
        float v = fill;
        if (!mask_rows || mask_rows[e]) {
            const long long i = nth_position(__ldg(offsets + e), __ldg(offsets + e + 1), base, mask_content, index);
            if (i >= 0) v = __ldg(data + i);
        }
        out[e] = v;
    }
}

__global__ void set_in_offsets_kernel(float* __restrict__ data, const long long* __restrict__ offsets, long long n_events,
                                      long long base, const unsigned char* __restrict__ mask_rows,
                                      const unsigned char* __restrict__ mask_content, int index,
                                      const float* __restrict__ values, float value)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_events; e += (long long)gridDim.x * blockDim.x) {
        if (mask_rows && !mask_rows[e]) continue;
        const long long i = nth_position(__ldg(offsets + e), __ldg(offsets + e + 1), base, mask_content, index);
        if (i >= 0) data[i] = values ? __ldg(values + e) : value;
    }
}

__global__ void select_opposite_sign_kernel(const float* __restrict__ pt, const int* __restrict__ charge,
                                            const long long* __restrict__ offsets, long long n_events, long long base,
                                            const unsigned char* __restrict__ mask_rows,
                                            const unsigned char* __restrict__ mask_content, unsigned char* __restrict__ out)
{
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_events; e += (long long)gridDim.x * blockDim.x) {
        const long long g0 = __ldg(offsets + e), g1 = __ldg(offsets + e + 1);
        // one pass: leading object, and per sign the best object (strict > keeps the first index among equal pt)
        long long lead = -1, bpos = -1, bneg = -1;
        float plead = 0.f, ppos = 0.f, pneg = 0.f;
        const bool row = !mask_rows || mask_rows[e];
        if (row) {
            for (long long g = g0; g < g1; ++g) {
                const long long i = g - base;
                if (mask_content && !mask_content[i]) continue;
                const float p = __ldg(pt + i);
                if (p != p) continue;
                const int q = __ldg(charge + i);
                if (lead < 0 || p > plead) { lead = i; plead = p; }
                if (q > 0 && (bpos < 0 || p > ppos)) { bpos = i; ppos = p; }
                if (q < 0 && (bneg < 0 || p > pneg)) { bneg = i; pneg = p; }
            }
        }
        long long part = -1;
        if (lead >= 0) {
            const int ql = __ldg(charge + lead);
            part = ql > 0 ? bneg : (ql < 0 ? bpos : -1);      // charge 0 has no opposite sign
        }
        const bool pair = part >= 0;
        for (long long g = g0; g < g1; ++g) {
            const long long i = g - base;
            out[i] = (pair && (i == lead || i == part)) ? 1 : 0;
        }
    }
}

}  // namespace dev

static unsigned grid_for(long long n)
{
    long long blocks = (n + 255) / 256;
    const long long maxb = (long long)sm_count() * 16;
    if (blocks > maxb) blocks = maxb;
    return (unsigned)(blocks < 1 ? 1 : blocks);
}

}  // namespace hepk

using namespace hepk;

extern "C" int32_t hepk_get_in_offsets(const float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                       const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index, float fill,
                                       float* out, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(index >= 0, "index < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out, "offsets/out is NULL");
    dev::get_in_offsets_kernel<<<grid_for(n_events), 256, 0, (cudaStream_t)stream>>>(
        data, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, index, fill, out);
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_set_in_offsets(float* data, const int64_t* offsets, int64_t n_events, int64_t content_base,
                                       const uint8_t* mask_rows, const uint8_t* mask_content, int32_t index,
                                       const float* values, float value, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(index >= 0, "index < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets, "offsets is NULL");
    dev::set_in_offsets_kernel<<<grid_for(n_events), 256, 0, (cudaStream_t)stream>>>(
        data, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, index, values, value);
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_select_opposite_sign(const float* pt, const int32_t* charge, const int64_t* offsets, int64_t n_events,
                                             int64_t content_base, const uint8_t* mask_rows, const uint8_t* mask_content,
                                             uint8_t* out_mask, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && charge && out_mask, "offsets/charge/out_mask is NULL");
    dev::select_opposite_sign_kernel<<<grid_for(n_events), 256, 0, (cudaStream_t)stream>>>(
        pt, charge, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, out_mask);
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

// ------------------------------------------------------------------------------------------ SURVEY.md 8(f-2)
// hepk_lookup_interp and hepk_fill_histogram_2d.  Both stream their inputs once
// (4 B in + 4 B out per element; 8-12 B per entry) with the knots / edges / bins in shared memory.
namespace hepk {
namespace dev {

__global__ void __launch_bounds__(256) lookup_interp_kernel(const float* __restrict__ x, long long n, const float* __restrict__ xs,
                                                            const float* __restrict__ ys, int nk, float* __restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_x = (float*)smem_raw;
    float* s_y = s_x + nk;
    for (int i = threadIdx.x; i < nk; i += blockDim.x) { s_x[i] = xs[i]; s_y[i] = ys[i]; }
    __syncthreads();
    const float x_lo = s_x[0], x_hi = s_x[nk - 1];
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float v = __ldg(x + i);
        float r;
        if (v != v) r = v;
        else if (v <= x_lo) r = s_y[0];
        else if (v >= x_hi) r = s_y[nk - 1];
        else {
            int lo = 0, hi = nk - 1;               // s_x[lo] <= v < s_x[hi]
            while (hi - lo > 1) {
                const int mid = (lo + hi) >> 1;
                if (v >= s_x[mid]) lo = mid; else hi = mid;
            }
            const float x0 = s_x[lo], y0 = s_y[lo];
            const float t = (v - x0) / (s_x[lo + 1] - x0);      // tolerance class: a few float32 roundings
            r = fmaf(t, s_y[lo + 1] - y0, y0);
        }
        out[i] = r;
    }
}

__global__ void __launch_bounds__(256) fill_hist2d_kernel(const float* __restrict__ x, const float* __restrict__ y,
                                                          const float* __restrict__ w, long long n,
                                                          const float* __restrict__ edges_x, int nx,
                                                          const float* __restrict__ edges_y, int ny,
                                                          double* __restrict__ acc, unsigned long long* __restrict__ counts)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_ex = (float*)smem_raw;
    float* s_ey = s_ex + (nx + 1);
    float* s_sumw = s_ey + (ny + 1);
    const int slots = (nx + 2) * (ny + 2);
    unsigned int* s_cnt = (unsigned int*)(s_sumw + slots);
    for (int i = threadIdx.x; i <= nx; i += blockDim.x) s_ex[i] = edges_x[i];
    for (int i = threadIdx.x; i <= ny; i += blockDim.x) s_ey[i] = edges_y[i];
    for (int i = threadIdx.x; i < slots; i += blockDim.x) { s_sumw[i] = 0.f; s_cnt[i] = 0u; }
    __syncthreads();
    const float lox = s_ex[0], invx = (float)nx / (s_ex[nx] - lox);
    const float loy = s_ey[0], invy = (float)ny / (s_ey[ny] - loy);
    auto flush = [&]() {
        __syncthreads();
        for (int i = threadIdx.x; i < slots; i += blockDim.x) {
            if (acc) { const float v = s_sumw[i]; if (v != 0.f) { atomicAdd(acc + i, (double)v); s_sumw[i] = 0.f; } }
            if (counts) { const unsigned int c = s_cnt[i]; if (c) { atomicAdd(counts + i, (unsigned long long)c); s_cnt[i] = 0u; } }
        }
        __syncthreads();
    };
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long iters = (n + stride - 1) / stride;
    for (long long it = 0; it < iters; ++it) {
        const long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x + it * stride;
        if (i < n) {
            const int s = hist_slot(__ldg(x + i), s_ex, nx, lox, invx) * (ny + 2) + hist_slot(__ldg(y + i), s_ey, ny, loy, invy);
            if (acc) atomicAdd(&s_sumw[s], w ? __ldg(w + i) : 1.f);
            if (counts) atomicAdd(&s_cnt[s], 1u);
        }
        if ((it + 1) % 64 == 0) flush();      // bounded float32 partial sums
    }
    flush();
}

// sumw[i] = float32(float64(sumw[i]) + acc[i])
__global__ void hist2d_finalize(float* __restrict__ sumw, const double* __restrict__ acc, int n)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) sumw[i] = (float)((double)sumw[i] + acc[i]);
}

}  // namespace dev
}  // namespace hepk

extern "C" int32_t hepk_lookup_interp(const float* x, int64_t n, const float* xs, const float* ys, int32_t nk, float* out,
                                      void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(xs && ys && nk >= 2, "knots are NULL or fewer than 2");
    if ((size_t)nk * 8 > 200 * 1024) {
        set_error("hepk_lookup_interp: %d knots do not fit 200 KB of shared memory", nk);
        return HEPK_ERR_UNSUPPORTED;
    }
    if (n == 0) return HEPK_OK;
    HEPK_REQUIRE(x && out, "x/out is NULL");
    const size_t smem = (size_t)nk * 8;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(dev::lookup_interp_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dev::lookup_interp_kernel<<<grid_for(n), 256, smem, (cudaStream_t)stream>>>(x, n, xs, ys, nk, out);
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" size_t hepk_hist2d_workspace_bytes(int32_t nx, int32_t ny)
{
    if (nx < 1 || ny < 1) return 0;
    return (size_t)(nx + 2) * (size_t)(ny + 2) * sizeof(double);
}

extern "C" int32_t hepk_fill_histogram_2d(const float* x, const float* y, const float* weights, int64_t n,
                                          const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                                          float* sumw, int64_t* counts, void* workspace, size_t workspace_bytes, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges_x && edges_y && nx >= 1 && ny >= 1, "edges are NULL or an axis has no bins");
    const long long slots = (long long)(nx + 2) * (ny + 2);
    if (slots > 16384) {
        set_error("hepk_fill_histogram_2d: (nx+2)*(ny+2) = %lld exceeds 16384", slots);
        return HEPK_ERR_UNSUPPORTED;
    }
    if (n == 0 || (!sumw && !counts)) return HEPK_OK;
    HEPK_REQUIRE(x && y, "x/y is NULL");
    if (sumw) {
        HEPK_REQUIRE(workspace != nullptr, "workspace is NULL");
        HEPK_REQUIRE(workspace_bytes >= hepk_hist2d_workspace_bytes(nx, ny), "workspace too small");
    }
    cudaStream_t st = (cudaStream_t)stream;
    const size_t smem = ((size_t)(nx + 1) + (size_t)(ny + 1) + 2 * (size_t)slots) * 4;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(dev::fill_hist2d_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (sumw) HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, (size_t)slots * sizeof(double), st));
    unsigned grid = grid_for((n + 3) / 4);
    dev::fill_hist2d_kernel<<<grid, 256, smem, st>>>(x, y, weights, n, edges_x, nx, edges_y, ny, sumw ? (double*)workspace : nullptr,
                                                     (unsigned long long*)counts);
    HEPK_CUDA_TRY(cudaGetLastError());
    if (sumw) {
        dev::hist2d_finalize<<<(unsigned)((slots + 255) / 256), 256, 0, st>>>(sumw, (const double*)workspace, (int)slots);
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    return HEPK_OK;
}
