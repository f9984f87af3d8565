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
