// hepk_offsets.cu — the remaining generic kernels of the paper's list (include/hepk.h):
// hepk_get_in_offsets, hepk_set_in_offsets; the f-2 lookups and the 2-D histogram; hepk_triplet_mass.
// (hepk_select_opposite_sign, reads whole events and lives in hepk_tiles.cu.)
//
// get / set touch one element per event, so they are bound by the offsets stream (8 B/event, coalesced) plus one
// 32-byte sector per touched element; one thread per event (the paper's own loop shape, Listing 1) is the right
// mapping: there is no per-event work to spread over lanes unless a content mask forces a scan, and then the scan
// is the event's few objects.
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

}  // namespace dev

// one wave of resident CTAs (kernels that stage tables once per CTA and merge privatised bins at its end)
static unsigned grid_resident(const void* kern, size_t smem, long long items)
{
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, smem) != cudaSuccess || occ < 1) occ = 1;
    long long blocks = (items + 255) / 256;
    const long long maxb = (long long)sm_count() * occ;
    if (blocks > maxb) blocks = maxb;
    return (unsigned)(blocks < 1 ? 1 : blocks);
}

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
        data, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, index, fill, out); count_launch();
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
        data, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, index, values, value); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

// ------------------------------------------------------------------------------------------ SURVEY.md 8(f-2)
// hepk_lookup_interp and hepk_fill_histogram_2d.  Both stream their inputs once
// (4 B in + 4 B out per element; 8-12 B per entry) with the knots / edges / bins in shared memory.
namespace hepk {
namespace dev {

// Knots in shared memory; the segment is found by the arithmetic bin guess of hepk_lookup_binned when the knots are
// uniform in x or in log2 x (verified at start-up, exact after one +-1 step), else by binary search; four elements per
// thread and step with 16-byte loads and stores when the pointers allow.
template <bool VEC>
__global__ void __launch_bounds__(256) lookup_interp_kernel(const float* __restrict__ x, long long n, const float* __restrict__ xs,
                                                            const float* __restrict__ ys, int nk, float* __restrict__ out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_x = (float*)smem_raw;
    float* s_y = s_x + nk;
    float* s_m = s_y + nk;                                 // slope of segment i (one IEEE division per segment and CTA)
    for (int i = threadIdx.x; i < nk; i += blockDim.x) { s_x[i] = xs[i]; s_y[i] = ys[i]; }
    __syncthreads();
    for (int i = threadIdx.x; i + 1 < nk; i += blockDim.x) s_m[i] = (s_y[i + 1] - s_y[i]) / (s_x[i + 1] - s_x[i]);
    __syncthreads();
    float* s_p = s_m + nk;                                 // padded copy of the knots (pad_axis_find, bin form)
    pad_axis_fill<false>(s_p, xs, nk - 1);
    AxisGuess ax;
    ax.mode = 0; ax.lo = 0.f; ax.inv = 0.f;
    if (nk >= 2) ax = classify_axis(s_x, nk - 1);          // the knots as the edges of nk - 1 segments (its barriers publish s_p)
    const float x_lo = s_x[0], x_hi = s_x[nk - 1];
    const float y_lo = s_y[0], y_hi = s_y[nk - 1];
    const float top = (float)(nk - 2);
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    dispatch_axis(ax.mode, [&](auto tx) {
        constexpr int AX = decltype(tx)::value;
        auto interp = [&](float v) {
            const int lo = pad_axis_find<AX, false>(v, s_x, s_p, nk - 1, ax, top);  // s_x[lo] <= v < s_x[lo + 1] inside the range
            float r = fmaf(v - s_x[lo], s_m[lo], s_y[lo]);       // tolerance class: a few float32 roundings
            r = v <= x_lo ? y_lo : r;
            r = v >= x_hi ? y_hi : r;
            return v != v ? v : r;
        };
        if (VEC) {
            const long long n4 = n >> 2;
            for (long long g = t0; g < n4; g += stride) {
                const float4 v = __ldg(reinterpret_cast<const float4*>(x) + g);
                float4 r;
                r.x = interp(v.x); r.y = interp(v.y); r.z = interp(v.z); r.w = interp(v.w);
                reinterpret_cast<float4*>(out)[g] = r;
            }
            for (long long i = (n4 << 2) + t0; i < n; i += stride) out[i] = interp(__ldg(x + i));
        } else {
            for (long long i = t0; i < n; i += stride) out[i] = interp(__ldg(x + i));
        }
    });
}

// Four entries per thread and step (16-byte loads when the pointers allow).  Without weights only the integer counts are
// accumulated (native shared-memory atomics) and the weighted sums are taken from them when the bins are flushed;
// with weights the float32 partial sums (compare-and-swap atomics) are flushed into float64 at bounded intervals.
template <bool VEC>
__global__ void __launch_bounds__(256, 6) fill_hist2d_kernel(const float* __restrict__ x, const float* __restrict__ y,
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
    float* s_px = (float*)(s_cnt + slots);      // padded copies of the edges (pad_axis_find, slot form)
    float* s_py = s_px + (nx + 3);
    for (int i = threadIdx.x; i <= nx; i += blockDim.x) s_ex[i] = edges_x[i];
    for (int i = threadIdx.x; i <= ny; i += blockDim.x) s_ey[i] = edges_y[i];
    for (int i = threadIdx.x; i < slots; i += blockDim.x) { s_sumw[i] = 0.f; s_cnt[i] = 0u; }
    pad_axis_fill<true>(s_px, edges_x, nx);
    pad_axis_fill<true>(s_py, edges_y, ny);
    __syncthreads();
    const AxisGuess ax = classify_axis(s_ex, nx), ay = classify_axis(s_ey, ny);
    const bool fsum = acc != nullptr && w != nullptr;          // float partial sums are needed
    const bool icnt = counts != nullptr || (acc != nullptr && w == nullptr);
    auto flush = [&]() {
        __syncthreads();
        for (int i = threadIdx.x; i < slots; i += blockDim.x) {
            if (fsum) { const float v = s_sumw[i]; if (v != 0.f) { atomicAdd(acc + i, (double)v); s_sumw[i] = 0.f; } }
            if (icnt) {
                const unsigned int c = s_cnt[i];
                if (c) {
                    if (counts) atomicAdd(counts + i, (unsigned long long)c);
                    if (acc && !w) atomicAdd(acc + i, (double)c);
                    s_cnt[i] = 0u;
                }
            }
        }
        __syncthreads();
    };
    const float top_x = (float)(nx + 1), top_y = (float)(ny + 1);
    const int row = ny + 2;
    const uint32_t sumw_a = smem_u32(s_sumw), cnt_a = smem_u32(s_cnt);
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    dispatch_axes(ax.mode, ay.mode, [&](auto tx, auto ty) {
        constexpr int AX = decltype(tx)::value, AY = decltype(ty)::value;
        auto slot_of = [&](float xv, float yv) {
            return pad_axis_find<AX, true>(xv, s_ex, s_px, nx, ax, top_x) * row + pad_axis_find<AY, true>(yv, s_ey, s_py, ny, ay, top_y);
        };
        auto put = [&](int s, float wv) {
            if (fsum) red_shared_add_f32_at(sumw_a + 4u * (unsigned)s, wv);
            if (icnt) red_shared_add_u32_at(cnt_a + 4u * (unsigned)s, 1u);
        };
        if (VEC) {
            const long long n4 = n >> 2;
            const long long iters = (n4 + stride - 1) / stride;
            for (long long it = 0; it < iters; ++it) {
                const long long g = t0 + it * stride;
                if (g < n4) {
                    const float4 xv = __ldg(reinterpret_cast<const float4*>(x) + g), yv = __ldg(reinterpret_cast<const float4*>(y) + g);
                    const float4 wv = w ? __ldg(reinterpret_cast<const float4*>(w) + g) : make_float4(1.f, 1.f, 1.f, 1.f);
                    // all four slots before the first update (the updates are opaque to the compiler: an edge load
                    // cannot move across one)
                    const int s0 = slot_of(xv.x, yv.x), s1 = slot_of(xv.y, yv.y), s2 = slot_of(xv.z, yv.z), s3 = slot_of(xv.w, yv.w);
                    put(s0, wv.x); put(s1, wv.y); put(s2, wv.z); put(s3, wv.w);
                }
                if (fsum && (it + 1) % 16 == 0) flush();      // bounded float32 partial sums
            }
            for (long long i = (n4 << 2) + t0; i < n; i += stride) put(slot_of(__ldg(x + i), __ldg(y + i)), w ? __ldg(w + i) : 1.f);
        } else {
            const long long iters = (n + stride - 1) / stride;
            for (long long it = 0; it < iters; ++it) {
                const long long i = t0 + it * stride;
                if (i < n) put(slot_of(__ldg(x + i), __ldg(y + i)), w ? __ldg(w + i) : 1.f);
                if (fsum && (it + 1) % 64 == 0) flush();
            }
        }
    });
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
    if ((size_t)nk * 16 > 200 * 1024) {
        set_error("hepk_lookup_interp: %d knots do not fit 200 KB of shared memory", nk);
        return HEPK_ERR_UNSUPPORTED;
    }
    if (n == 0) return HEPK_OK;
    HEPK_REQUIRE(x && out, "x/out is NULL");
    const size_t smem = (size_t)nk * 16;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(dev::lookup_interp_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    HEPK_CUDA_TRY(cudaFuncSetAttribute(dev::lookup_interp_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    const bool vec = aligned16(x) && aligned16(out);
    auto kern = vec ? dev::lookup_interp_kernel<true> : dev::lookup_interp_kernel<false>;
    kern<<<grid_resident((const void*)kern, smem, vec ? (n + 3) / 4 : n), 256, smem, (cudaStream_t)stream>>>(x, n, xs, ys, nk, out); count_launch();
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
    const size_t smem = ((size_t)(nx + 1) + (size_t)(ny + 1) + 2 * (size_t)slots + (size_t)(nx + 3) + (size_t)(ny + 3)) * 4;
    const bool vec = aligned16(x) && aligned16(y) && (!weights || aligned16(weights));
    auto kern = vec ? dev::fill_hist2d_kernel<true> : dev::fill_hist2d_kernel<false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    if (sumw) HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, (size_t)slots * sizeof(double), st));
    unsigned grid = grid_resident((const void*)kern, smem, (n + 3) / 4);
    kern<<<grid, 256, smem, st>>>(x, y, weights, n, edges_x, nx, edges_y, ny, sumw ? (double*)workspace : nullptr,
                                  (unsigned long long*)counts); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    if (sumw) {
        dev::hist2d_finalize<<<(unsigned)((slots + 255) / 256), 256, 0, st>>>(sumw, (const double*)workspace, (int)slots); count_launch();
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    return HEPK_OK;
}

// ------------------------------------------------------------------------------------------ SURVEY.md 8(f-3)
// hepk_triplet_mass: eight lanes per event, four events per warp.  The selected jets' four-vectors are
// built once per event (one lane per jet, float64) into shared memory; lanes take the (a, b) pairs round-robin and run over c > b,
// so every triplet costs four float64 adds, four multiply-adds and a square root; the best triplet per lane is
// reduced over the warp by (distance, a, b, c).  ALU-bound on long events, launch/latency-bound on short ones.
namespace hepk {
namespace dev {

constexpr int TRIPLET_CAP = 64;      // selected jets of one event held in shared memory (more: recomputed on the fly)
constexpr int TRIPLET_WARPS = 4;
constexpr int TRIPLET_GROUP = 8;     // lanes per event: four events per warp (a typical event has ~10 pairs)
constexpr int TRIPLET_GPW = 32 / TRIPLET_GROUP;

struct Vec4 { double e, x, y, z; };

__device__ __forceinline__ Vec4 four_vector(float pt, float eta, float phi, float m)
{
    const double p = pt, mm = m;
    double s, c;
    sincos((double)phi, &s, &c);
    const double ch = cosh((double)eta);
    Vec4 v;
    v.e = sqrt(p * p * ch * ch + mm * mm);
    v.x = p * c; v.y = p * s; v.z = p * sinh((double)eta);
    return v;
}

__global__ void __launch_bounds__(32 * TRIPLET_WARPS) triplet_kernel(const float* __restrict__ pt, const float* __restrict__ eta,
                                                                      const float* __restrict__ phi, const float* __restrict__ mass,
                                                                      const long long* __restrict__ offsets, long long n_events,
                                                                      long long base, const unsigned char* __restrict__ mask_rows,
                                                                      const unsigned char* __restrict__ mask_content, float target,
                                                                      float* __restrict__ out_mass, int* __restrict__ out_idx)
{
    __shared__ Vec4 s_vec[TRIPLET_WARPS * TRIPLET_GPW][TRIPLET_CAP];
    __shared__ int s_loc[TRIPLET_WARPS * TRIPLET_GPW][TRIPLET_CAP];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int grp = lane / TRIPLET_GROUP, sl = lane % TRIPLET_GROUP;
    Vec4* vec = s_vec[warp * TRIPLET_GPW + grp];
    int* loc = s_loc[warp * TRIPLET_GPW + grp];
    const long long ng = (long long)gridDim.x * TRIPLET_WARPS * TRIPLET_GPW;
    const long long g_first = ((long long)blockIdx.x * TRIPLET_WARPS + warp) * TRIPLET_GPW + grp;
    // all four groups of a warp run the same number of rounds (warp-wide votes and shuffles below)
    const long long rounds = (n_events + ng - 1) / ng;
    for (long long r = 0; r < rounds; ++r) {
        const long long e = g_first + r * ng;
        const bool live = e < n_events;
        const long long g0 = live ? __ldg(offsets + e) : 0, g1 = live ? __ldg(offsets + e + 1) : 0;
        const bool row = live && (!mask_rows || mask_rows[e]);
        // ---- selected jets -> local index list (and four-vectors while they fit), eight jets per step
        int nsel = 0;
        const long long span = row ? g1 - g0 : 0;
        const long long steps = __reduce_max_sync(0xffffffffu, (unsigned)((span + TRIPLET_GROUP - 1) / TRIPLET_GROUP));
        for (long long st = 0; st < steps; ++st) {
            const long long g = g0 + st * TRIPLET_GROUP + sl;
            const bool sel = row && g < g1 && (!mask_content || mask_content[g - base]);
            const unsigned m = (__ballot_sync(0xffffffffu, sel) >> (TRIPLET_GROUP * grp)) & ((1u << TRIPLET_GROUP) - 1u);
            const int at = nsel + __popc(m & ((1u << sl) - 1u));
            if (sel && at < TRIPLET_CAP) {
                const long long i = g - base;
                loc[at] = (int)(g - g0);
                vec[at] = four_vector(__ldg(pt + i), __ldg(eta + i), __ldg(phi + i), __ldg(mass + i));
            }
            nsel += __popc(m);
        }
        __syncwarp();
        const bool cached = nsel <= TRIPLET_CAP;
        // local index and four-vector of the s-th selected jet (slow way when the event does not fit the cache)
        auto local_of = [&](int s) -> int {
            if (cached) return loc[s];
            int seen = 0;
            for (long long g = g0; g < g1; ++g)
                if (!mask_content || mask_content[g - base]) { if (seen == s) return (int)(g - g0); ++seen; }
            return -1;
        };
        auto vec_of = [&](int s) -> Vec4 {
            if (cached) return vec[s];
            const long long i = g0 - base + local_of(s);
            return four_vector(__ldg(pt + i), __ldg(eta + i), __ldg(phi + i), __ldg(mass + i));
        };
        // ---- triplets: a lane of the group takes pairs (a, b) round-robin, runs over c
        double best = CUDART_INF;
        double best_m = 0.0;
        int ba = 0x7fffffff, bb = 0x7fffffff, bc = 0x7fffffff;
        const long long npairs = (long long)nsel * (nsel - 1) / 2;
        for (long long p = sl; p < npairs; p += TRIPLET_GROUP) {
            int a = 0;
            long long q = p;
            while (q >= nsel - 1 - a) { q -= nsel - 1 - a; ++a; }
            const int b = a + 1 + (int)q;
            const Vec4 va = vec_of(a), vb = vec_of(b);
            const double e2 = va.e + vb.e, x2 = va.x + vb.x, y2 = va.y + vb.y, z2 = va.z + vb.z;
            for (int c = b + 1; c < nsel; ++c) {
                const Vec4 vc = vec_of(c);
                const double E = e2 + vc.e, X = x2 + vc.x, Y = y2 + vc.y, Z = z2 + vc.z;
                double m2 = E * E - X * X - Y * Y - Z * Z;
                if (!(m2 > 0.0)) m2 = 0.0;
                const double M = sqrt(m2);
                const double d = fabs(M - (double)target);
                if (d < best) { best = d; best_m = M; ba = a; bb = b; bc = c; }     // visited in (a, b, c) order per lane
            }
        }
        __syncwarp();
        // ---- argmin over the group's lanes by (distance, a, b, c)
#pragma unroll
        for (int o = TRIPLET_GROUP / 2; o >= 1; o >>= 1) {
            const double od = __shfl_xor_sync(0xffffffffu, best, o);
            const double om = __shfl_xor_sync(0xffffffffu, best_m, o);
            const int oa = __shfl_xor_sync(0xffffffffu, ba, o), ob = __shfl_xor_sync(0xffffffffu, bb, o),
                      oc = __shfl_xor_sync(0xffffffffu, bc, o);
            const bool take = od < best || (od == best && (oa < ba || (oa == ba && (ob < bb || (ob == bb && oc < bc)))));
            if (take) { best = od; best_m = om; ba = oa; bb = ob; bc = oc; }
        }
        if (sl == 0 && live) {
            const bool have = nsel >= 3;
            out_mass[e] = have ? (float)best_m : 0.0f;
            if (out_idx) {
                out_idx[3 * e] = have ? local_of(ba) : -1;
                out_idx[3 * e + 1] = have ? local_of(bb) : -1;
                out_idx[3 * e + 2] = have ? local_of(bc) : -1;
            }
        }
        __syncwarp();
    }
}

}  // namespace dev
}  // namespace hepk

extern "C" int32_t hepk_triplet_mass(const float* pt, const float* eta, const float* phi, const float* mass,
                                     const int64_t* offsets, int64_t n_events, int64_t content_base, const uint8_t* mask_rows,
                                     const uint8_t* mask_content, float target, float* out_mass, int32_t* out_idx, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    if (n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(offsets && out_mass, "offsets/out_mass is NULL");
    const long long per_block = dev::TRIPLET_WARPS * dev::TRIPLET_GPW;
    long long blocks = (n_events + per_block - 1) / per_block;
    const long long maxb = (long long)sm_count() * 12;
    if (blocks > maxb) blocks = maxb;
    dev::triplet_kernel<<<(unsigned)blocks, 32 * dev::TRIPLET_WARPS, 0, (cudaStream_t)stream>>>(
        pt, eta, phi, mass, (const long long*)offsets, n_events, content_base, mask_rows, mask_content, target, out_mass, out_idx); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

// ------------------------------------------------------------------------------------------ hepk_validate_offsets
namespace hepk {
namespace dev {
__global__ void validate_offsets_kernel(const long long* __restrict__ off, long long n_events, long long base, long long n_objects,
                                        unsigned long long* __restrict__ n_bad)
{
    unsigned long long bad = 0;
    for (long long e = (long long)blockIdx.x * blockDim.x + threadIdx.x; e < n_events; e += (long long)gridDim.x * blockDim.x)
        if (__ldg(off + e) > __ldg(off + e + 1)) ++bad;
    if (blockIdx.x == 0 && threadIdx.x == 0) {
        if (off[0] < base) ++bad;
        if (off[n_events] - base > n_objects) ++bad;
    }
    bad = __reduce_add_sync(0xffffffffu, (unsigned)bad);
    if ((threadIdx.x & 31) == 0 && bad) atomicAdd(n_bad, bad);
}
}  // namespace dev
}  // namespace hepk

extern "C" int32_t hepk_validate_offsets(const int64_t* offsets, int64_t n_events, int64_t content_base, int64_t n_objects,
                                         int64_t* n_bad, void* stream)
{
    HEPK_REQUIRE(n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(offsets && n_bad, "offsets/n_bad is NULL");
    cudaStream_t st = (cudaStream_t)stream;
    HEPK_CUDA_TRY(cudaMemsetAsync(n_bad, 0, sizeof(int64_t), st));
    dev::validate_offsets_kernel<<<grid_for(n_events), 256, 0, st>>>((const long long*)offsets, n_events, content_base, n_objects,
                                                                    (unsigned long long*)n_bad); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}
