// hepk_hist.cu — weighted histogram fills with the sum of squared weights, and the event weight from a lookup
// (include/hepk.h: hepk_fill_histogram_w2, hepk_fill_histogram_2d_w2, hepk_event_weight_lookup; SURVEY.md 8(f-2),
// PAPER.md:L109, L134).
//
// One fill kernel for one and two dimensions.  Bins are privatised per CTA in shared memory, one ROW per slot
// holding all columns of that slot (sumw, sumw2 value, sumw2 remainder, count), so an entry's updates are
// immediate offsets from one address.  Small histograms (<= FIXED_WORDS words) take fixed-point int32 bins — native
// shared-memory integer atomics, exact sums, any order — when a pre-pass over the weights finds them finite and
// within a factor 8 of each other; every CTA checks all its bins after each step of 1024 entries and moves a bin
// to its 64-bit global accumulator before it can leave the int32 range.  Everything else takes float32 bins
// (compare-and-swap atomics) flushed into float64 accumulators at bounded intervals.
#include <mutex>

#include "hepk_common.cuh"
#include "hepk_hist_lanes.cuh"

namespace hepk {
namespace dev {

enum { HH_WMAX = 0, HH_WMIN = 1, HH_BAD = 2, HH_DONE = 3 /* CTAs of the lane-private fill that have finished */, HH_WORDS = 4 };
constexpr int HIST_FIXED_WORDS = 1024;      // privatised words a CTA can afford to check after every step
constexpr int HIST_FLUSH_AT = 1 << 29;

struct HistParams {
    const float *x, *y, *w;
    long long n;
    const float *edges_x, *edges_y;
    int nx, ny;                 // ny = 0: one dimension
    int slots, WS, col_w2, col_cnt, want_sumw;      // columns: [sumw] [w2 value, w2 remainder] [count]; -1 = absent
    long long* acc;             // [slots][WS] int64 fixed point or float64 bits
    const unsigned int* hdr;    // weight range (HH_*)
    float *sumw, *sumw2;
    long long* counts;
    int fixed_allowed;          // the histogram is small enough for the fixed-point scheme
};

__global__ void hist_weight_range_kernel(const float* __restrict__ w, long long n, unsigned int* __restrict__ hdr)
{
    float m = 0.0f, mn = CUDART_INF_F;
    bool bad = false;
    for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
        const float a = fabsf(__ldg(w + i));
        bad = bad || !(a < CUDART_INF_F);
        m = fmaxf(m, a);
        if (a > 0.0f) mn = fminf(mn, a);
    }
    const unsigned int b = __reduce_max_sync(0xffffffffu, __float_as_uint(m));
    const unsigned int c = __reduce_min_sync(0xffffffffu, __float_as_uint(mn));
    if (__any_sync(0xffffffffu, bad) && (threadIdx.x & 31) == 0) atomicOr(hdr + HH_BAD, 1u);
    if ((threadIdx.x & 31) == 0) {
        if (b) atomicMax(hdr + HH_WMAX, b);
        atomicMin(hdr + HH_WMIN, c);
    }
}

// fixed-point scales 2^k (weights) and 2^k2 (squared weights): |w| 2^k < 2^19; 0: float bins
__device__ __forceinline__ void hist_fill_scales(const HistParams& P, float& sc, float& sc2)
{
    sc = sc2 = 0.0f;
    if (!P.fixed_allowed) return;
    float wm = 1.0f, wn = 1.0f;
    if (P.w) {
        if (P.hdr[HH_BAD]) return;
        wm = __uint_as_float(P.hdr[HH_WMAX]);
        wn = __uint_as_float(P.hdr[HH_WMIN]);
    }
    if (!(wm > 0.0f && wm < CUDART_INF_F && wn > 0.0f && wm <= 8.0f * wn)) return;
    if (!(wm * wm < CUDART_INF_F && wn * wn > 0.0f)) return;
    int e, e2;
    frexpf(wm, &e);
    frexpf(wm * wm, &e2);
    const int k = 19 - e, k2 = 19 - e2;
    if (k <= -100 || k >= 100 || k2 <= -100 || k2 >= 100) return;
    sc = ldexpf(1.0f, k);
    sc2 = ldexpf(1.0f, k2);
}

template <bool VEC>
__global__ void __launch_bounds__(256, 6) hist_fill_kernel(const __grid_constant__ HistParams P)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_ex = (float*)smem_raw;
    float* s_ey = s_ex + (P.nx + 1);
    int* s_bins = (int*)(s_ey + (P.ny > 0 ? P.ny + 1 : 0));
    __shared__ float s_sc[2];
    const int n_words = P.slots * P.WS;
    float* s_px = (float*)(s_bins + n_words);      // padded copies of the edges (pad_axis_find, slot form)
    float* s_py = s_px + (P.nx + 3);
    for (int i = threadIdx.x; i <= P.nx; i += blockDim.x) s_ex[i] = P.edges_x[i];
    if (P.ny > 0) for (int i = threadIdx.x; i <= P.ny; i += blockDim.x) s_ey[i] = P.edges_y[i];
    for (int i = threadIdx.x; i < n_words; i += blockDim.x) s_bins[i] = 0;
    pad_axis_fill<true>(s_px, P.edges_x, P.nx);
    if (P.ny > 0) pad_axis_fill<true>(s_py, P.edges_y, P.ny);
    if (threadIdx.x == 0) hist_fill_scales(P, s_sc[0], s_sc[1]);
    __syncthreads();
    const float sc = s_sc[0], sc2 = s_sc[1];
    const bool fixed = sc != 0.0f;
    // arithmetic bin guess on linear or log2 axes (exact after one +-1 step), binary search otherwise
    const AxisGuess ax = classify_axis(s_ex, P.nx);
    AxisGuess ay;
    ay.mode = 1; ay.lo = 0.f; ay.inv = 0.f;        // (one dimension: the tag of the unused axis)
    if (P.ny > 0) ay = classify_axis(s_ey, P.ny);
    const float top_x = (float)(P.nx + 1), top_y = (float)(P.ny + 1);
    const uint32_t bins_a = smem_u32(s_bins);
    const uint32_t w2_off = 4u * (unsigned)(P.col_w2 >= 0 ? P.col_w2 : 0), cnt_off = 4u * (unsigned)(P.col_cnt >= 0 ? P.col_cnt : 0);

    // move bins into the global accumulators; `all`: everything non-zero, else only integers about to overflow
    auto flush = [&](bool all) {
        for (int i = threadIdx.x; i < n_words; i += blockDim.x) {
            const int v = s_bins[i];
            if (v == 0) continue;
            const bool is_int = fixed || (i % P.WS) == P.col_cnt;
            if (is_int) {
                if (!all && (unsigned)(v + HIST_FLUSH_AT) < 2u * (unsigned)HIST_FLUSH_AT) continue;
                const int y = atomicExch(s_bins + i, 0);
                if (y) atomicAdd((unsigned long long*)P.acc + i, (unsigned long long)(long long)y);
            } else {
                const float y = atomicExch((float*)s_bins + i, 0.0f);
                if (y != 0.0f) atomicAdd((double*)P.acc + i, (double)y);
            }
        }
    };
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    // fixed point: a step adds at most 1024 entries < 2^19 each to a bin, so a check per step keeps |bin| < 2^31;
    // float: bounded partial sums (a flush every 32 steps)
    const int check_every = fixed ? 1 : 32;
    dispatch_axes(ax.mode, ay.mode, [&](auto tx, auto ty) {
        constexpr int AX = decltype(tx)::value, AY = decltype(ty)::value;
        auto slot_of = [&](float xv, float yv) {
            int s = pad_axis_find<AX, true>(xv, s_ex, s_px, P.nx, ax, top_x);
            if (P.ny > 0) s = s * (P.ny + 2) + pad_axis_find<AY, true>(yv, s_ey, s_py, P.ny, ay, top_y);
            return s;
        };
        auto put = [&](int s, float wv) {
            const uint32_t row = bins_a + 4u * (unsigned)(s * P.WS);
            if (fixed) {
                if (P.want_sumw) red_shared_add_u32_at(row, (unsigned int)__float2int_rn(wv * sc));
                if (P.col_w2 >= 0) {
                    const float y2 = wv * wv * sc2;
                    const int qh = __float2int_rn(y2);
                    red_shared_add_u32_at(row + w2_off, (unsigned int)qh);
                    red_shared_add_u32_at(row + w2_off + 4u, (unsigned int)__float2int_rn((y2 - (float)qh) * 1048576.0f));
                }
            } else {
                if (P.want_sumw) red_shared_add_f32_at(row, wv);
                if (P.col_w2 >= 0) red_shared_add_f32_at(row + w2_off, wv * wv);
            }
            if (P.col_cnt >= 0) red_shared_add_u32_at(row + cnt_off, 1u);
        };
        if (VEC) {
            const long long n4 = P.n / 4;
            const long long iters = (n4 + stride - 1) / stride;
            for (long long it = 0; it < iters; ++it) {
                const long long g = t0 + it * stride;
                if (g < n4) {
                    const float4 xv = __ldg((const float4*)P.x + g);
                    const float4 yv = P.ny > 0 ? __ldg((const float4*)P.y + g) : make_float4(0.f, 0.f, 0.f, 0.f);
                    const float4 wv = P.w ? __ldg((const float4*)P.w + g) : make_float4(1.f, 1.f, 1.f, 1.f);
                    // all four slots before the first update (an edge load cannot move across a shared-memory atomic)
                    const int s0 = slot_of(xv.x, yv.x), s1 = slot_of(xv.y, yv.y), s2 = slot_of(xv.z, yv.z), s3 = slot_of(xv.w, yv.w);
                    put(s0, wv.x); put(s1, wv.y); put(s2, wv.z); put(s3, wv.w);
                }
                if ((it + 1) % check_every == 0) flush(!fixed);
            }
            for (long long i = n4 * 4 + t0; i < P.n; i += stride) put(slot_of(P.x[i], P.ny > 0 ? P.y[i] : 0.f), P.w ? P.w[i] : 1.f);
        } else {
            const long long iters = (P.n + stride - 1) / stride;
            for (long long it = 0; it < iters; ++it) {
                const long long i = t0 + it * stride;
                if (i < P.n) put(slot_of(P.x[i], P.ny > 0 ? P.y[i] : 0.f), P.w ? P.w[i] : 1.f);
                if ((it + 1) % (4 * check_every) == 0) flush(!fixed);
            }
        }
    });
    __syncthreads();
    flush(true);
}

// the caller's arrays from the accumulators (one thread per slot)
__global__ void hist_finalize_kernel(const __grid_constant__ HistParams P)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= P.slots) return;
    float sc, sc2;
    hist_fill_scales(P, sc, sc2);
    const long long* row = P.acc + (long long)s * P.WS;
    if (P.want_sumw && P.sumw) {
        const double add = sc != 0.0f ? (double)row[0] / (double)sc : __longlong_as_double(row[0]);
        P.sumw[s] = (float)((double)P.sumw[s] + add);
    }
    if (P.col_w2 >= 0) {
        const double add = sc2 != 0.0f ? ((double)row[P.col_w2] + (double)row[P.col_w2 + 1] * (1.0 / 1048576.0)) / (double)sc2
                                       : __longlong_as_double(row[P.col_w2]);
        P.sumw2[s] = (float)((double)P.sumw2[s] + add);
    }
    if (P.col_cnt >= 0) P.counts[s] += row[P.col_cnt];
}

// w_out = w_in * table[B(x)]: one float32 multiply per event (exact class)
__global__ void __launch_bounds__(256) event_weight_lookup_kernel(const float* __restrict__ w_in, const float* __restrict__ x,
                                                                  long long n, const float* __restrict__ edges, int nb,
                                                                  const float* __restrict__ table, float* __restrict__ w_out)
{
    extern __shared__ __align__(16) unsigned char smem_raw[];
    float* s_e = (float*)smem_raw;
    float* s_t = s_e + (nb + 1);
    for (int i = threadIdx.x; i <= nb; i += blockDim.x) s_e[i] = edges[i];
    for (int i = threadIdx.x; i < nb; i += blockDim.x) s_t[i] = table[i];
    __syncthreads();
    // (HBM bound as it is: the padded-axis form of the guess saves a third of the instructions and no time here, and
    // its longer set-up showed in back-to-back calls of this 21 us kernel)
    const AxisGuess ax = classify_axis(s_e, nb);
    const long long stride = (long long)gridDim.x * blockDim.x;
    const long long t0 = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const bool vec = ((reinterpret_cast<uintptr_t>(x) | reinterpret_cast<uintptr_t>(w_out) | reinterpret_cast<uintptr_t>(w_in)) & 15u) == 0;
    if (vec) {
        const long long n4 = n / 4;
        for (long long g = t0; g < n4; g += stride) {
            const float4 xv = __ldg((const float4*)x + g);
            const float4 wv = w_in ? __ldg((const float4*)w_in + g) : make_float4(1.f, 1.f, 1.f, 1.f);
            float4 o;
            o.x = __fmul_rn(wv.x, s_t[find_bin_guess(xv.x, s_e, nb, ax)]);
            o.y = __fmul_rn(wv.y, s_t[find_bin_guess(xv.y, s_e, nb, ax)]);
            o.z = __fmul_rn(wv.z, s_t[find_bin_guess(xv.z, s_e, nb, ax)]);
            o.w = __fmul_rn(wv.w, s_t[find_bin_guess(xv.w, s_e, nb, ax)]);
            ((float4*)w_out)[g] = o;
        }
        for (long long i = n4 * 4 + t0; i < n; i += stride)
            w_out[i] = __fmul_rn(w_in ? w_in[i] : 1.0f, s_t[find_bin_guess(x[i], s_e, nb, ax)]);
    } else {
        for (long long i = t0; i < n; i += stride)
            w_out[i] = __fmul_rn(w_in ? w_in[i] : 1.0f, s_t[find_bin_guess(x[i], s_e, nb, ax)]);
    }
}

// measurement hook: lane-atomics of red.shared.add.s32 per launch, random addresses in `nbins` words
__global__ void probe_shared_atomics_kernel(int iters, int nbins, unsigned int* out)
{
    extern __shared__ unsigned int h[];
    for (int i = threadIdx.x; i < nbins; i += blockDim.x) h[i] = 0u;
    __syncthreads();
    const uint32_t base = smem_u32(h);
    unsigned int x = threadIdx.x * 2654435761u + blockIdx.x * 97u + 12345u;
    for (int i = 0; i < iters; ++i) {
        x = x * 1664525u + 1013904223u;
        const unsigned int idx = (x >> 8) % (unsigned)nbins;
        asm volatile("red.shared.add.s32 [%0], %1;" ::"r"(base + 4u * idx), "r"(1) : "memory");
    }
    __syncthreads();
    if (threadIdx.x == 0) out[blockIdx.x] = h[0];
}

}  // namespace dev

static unsigned grid_for_items(long long items)
{
    long long g = (items + 255) / 256;
    const long long maxb = (long long)sm_count() * 8;
    if (g > maxb) g = maxb;
    return (unsigned)(g < 1 ? 1 : g);
}

struct HistShape { int slots, ncol, WS, col_w2, col_cnt, want_sumw; };
static HistShape hist_shape(int nx, int ny, bool sumw, bool sumw2, bool counts)
{
    HistShape h;
    h.slots = (nx + 2) * (ny > 0 ? ny + 2 : 1);
    h.want_sumw = sumw ? 1 : 0;
    h.ncol = 1;                                   // column 0 is sumw (kept, unused, when not asked for)
    h.col_w2 = -1; h.col_cnt = -1;
    if (sumw2) { h.col_w2 = h.ncol; h.ncol += 2; }
    if (counts) { h.col_cnt = h.ncol; h.ncol += 1; }
    h.WS = (h.ncol & 1) ? h.ncol : h.ncol + 1;    // odd row length: the rows of a column cover all banks
    return h;
}

static int32_t hist_fill_launch(const char* who, const float* x, const float* y, const float* weights, long long n,
                                const float* edges_x, int nx, const float* edges_y, int ny, float* sumw, float* sumw2,
                                long long* counts, void* workspace, size_t workspace_bytes, cudaStream_t st)
{
    const HistShape h = hist_shape(nx, ny, sumw != nullptr, sumw2 != nullptr, counts != nullptr);
    if (n == 0 || (!sumw && !sumw2 && !counts)) return HEPK_OK;
    const size_t need = dev::HH_WORDS * 4 + (size_t)h.slots * h.WS * 8;
    if (!workspace || workspace_bytes < need) {
        set_error("%s: workspace is NULL or smaller than %zu bytes", who, need);
        return HEPK_ERR_INVALID;
    }
    const size_t smem = ((size_t)(nx + 1) + (ny > 0 ? (size_t)(ny + 1) : 0) + (size_t)h.slots * h.WS + (size_t)(nx + 3) + (size_t)(ny > 0 ? ny + 3 : 0)) * 4;
    if (smem > 200 * 1024) {
        set_error("%s: %d slots x %d columns do not fit 200 KB of shared memory", who, h.slots, h.WS);
        return HEPK_ERR_UNSUPPORTED;
    }
    dev::HistParams P;
    P.x = x; P.y = y; P.w = weights; P.n = n;
    P.edges_x = edges_x; P.edges_y = edges_y; P.nx = nx; P.ny = ny;
    P.slots = h.slots; P.WS = h.WS; P.col_w2 = h.col_w2; P.col_cnt = h.col_cnt; P.want_sumw = h.want_sumw;
    P.hdr = (const unsigned int*)workspace;
    P.acc = (long long*)((char*)workspace + dev::HH_WORDS * 4);
    P.sumw = sumw; P.sumw2 = sumw2; P.counts = counts;
    P.fixed_allowed = h.slots * h.WS <= dev::HIST_FIXED_WORDS ? 1 : 0;
    HEPK_CUDA_TRY(cudaMemsetAsync(workspace, 0, need, st));
    const bool vec = aligned16(x) && (!y || aligned16(y)) && (!weights || aligned16(weights));
    if (ny == 0) {
        // One dimension, few bins: a private copy of the bins per lane (hepk_hist_lanes.cuh) — float32 partial sums of
        // n / (threads of the grid) <= 32768 entries each, merged in float64; no pass over the weights, no atomics.
        const int mode = !weights ? 0 : (sumw2 ? 3 : (counts ? (sumw ? 2 : 0) : 1));
        const size_t head = dev::lane_hist_head_bytes(nx), per_warp = dev::lane_hist_warp_bytes(nx, mode);
        int warps = (size_t)max_smem_optin() > head ? (int)(((size_t)max_smem_optin() - head) / per_warp) : 0;
        if (warps > 8) warps = 8;
        if (warps >= 4 && n >= (1 << 16) && n <= 32768ll * sm_count() * warps * 32) {
            void (*k)(const float*, const float*, long long, const float*, int, dev::LaneHistOut);
            if (mode == 0) k = vec ? dev::fill_hist_lanes_kernel<0, true, true> : dev::fill_hist_lanes_kernel<0, false, true>;
            else if (mode == 1) k = vec ? dev::fill_hist_lanes_kernel<1, true, true> : dev::fill_hist_lanes_kernel<1, false, true>;
            else if (mode == 2) k = vec ? dev::fill_hist_lanes_kernel<2, true, true> : dev::fill_hist_lanes_kernel<2, false, true>;
            else k = vec ? dev::fill_hist_lanes_kernel<3, true, true> : dev::fill_hist_lanes_kernel<3, false, true>;
            P.fixed_allowed = 0;                  // the accumulators hold float64 sums
            dev::LaneHistOut o;
            o.sumw = nullptr; o.counts = nullptr; o.acc = P.acc;
            o.WS = h.WS; o.want_sumw = h.want_sumw; o.col_w2 = h.col_w2; o.col_cnt = h.col_cnt;
            // the last CTA to finish adds the rows to the caller's arrays (what hist_finalize_kernel does for float64 rows)
            o.done = (unsigned int*)workspace + dev::HH_DONE;
            o.fin_sumw = sumw; o.fin_sumw2 = sumw2; o.fin_counts = counts;
            const size_t sm = head + (size_t)warps * per_warp;
            HEPK_CUDA_TRY(cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm));
            k<<<sm_count(), warps * 32, sm, st>>>(x, weights, n, edges_x, nx, o); count_launch();
            HEPK_CUDA_TRY(cudaGetLastError());
            return HEPK_OK;
        }
    }
    if (weights && P.fixed_allowed) {
        static const unsigned int inf_bits = 0x7f800000u;
        HEPK_CUDA_TRY(cudaMemcpyAsync((unsigned int*)workspace + dev::HH_WMIN, &inf_bits, 4, cudaMemcpyHostToDevice, st));
        dev::hist_weight_range_kernel<<<grid_for_items((n + 7) / 8), 256, 0, st>>>(weights, n, (unsigned int*)workspace); count_launch();
        HEPK_CUDA_TRY(cudaGetLastError());
    }
    auto kern = vec ? dev::hist_fill_kernel<true> : dev::hist_fill_kernel<false>;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    int occ = 0;
    if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, kern, 256, smem) != cudaSuccess || occ < 1) occ = 1;
    long long grid = (long long)sm_count() * occ;
    const long long items = (n + 1023) / 1024;
    if (grid > items) grid = items;
    if (grid < 1) grid = 1;
    kern<<<(unsigned)grid, 256, smem, st>>>(P); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    dev::hist_finalize_kernel<<<(unsigned)((h.slots + 255) / 256), 256, 0, st>>>(P); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

}  // namespace hepk

using namespace hepk;

extern "C" size_t hepk_hist_workspace_bytes(int32_t nx, int32_t ny)
{
    if (nx < 1 || ny < 0) return 0;
    const HistShape h = hist_shape(nx, ny, true, true, true);      // the largest shape: every output asked for
    return dev::HH_WORDS * 4 + (size_t)h.slots * h.WS * 8;
}

extern "C" int32_t hepk_fill_histogram_w2(const float* data, const float* weights, int64_t n, const float* edges, int32_t nbins,
                                          float* sumw, float* sumw2, int64_t* counts, void* workspace, size_t workspace_bytes,
                                          void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges && nbins >= 1, "edges is NULL or nbins < 1");
    if (nbins + 2 > 16384) {
        set_error("hepk_fill_histogram_w2: nbins+2 = %d exceeds 16384", nbins + 2);
        return HEPK_ERR_UNSUPPORTED;
    }
    HEPK_REQUIRE(n == 0 || data, "data is NULL");
    return hist_fill_launch("hepk_fill_histogram_w2", data, nullptr, weights, n, edges, nbins, nullptr, 0, sumw, sumw2,
                            (long long*)counts, workspace, workspace_bytes, (cudaStream_t)stream);
}

// ---- the same fill with its scratch in the library (include/hepk.h: hepk_fill_histogram_w2_static) -------------------
// For callers that cannot allocate (code under CUDA graph capture, serving loops, harnesses that forbid cudaMalloc):
// the 64-bit accumulators live in a file-scope device array instead of a caller's workspace.  Every GPU that loads
// the library holds the array until exit.  In host code its NAME is a host-side stand-in, not a device address: the
// address comes from cudaGetSymbolAddress, once per device, with that device current.
namespace hepk {
constexpr int STATIC_MAX_SLOTS = HEPK_STATIC_HIST_MAX_BINS + 2;
constexpr size_t STATIC_SCRATCH_BYTES = ((size_t)dev::HH_WORDS * 4 + (size_t)STATIC_MAX_SLOTS * 5 * 8 + 255) / 256 * 256;
static __device__ __align__(256) unsigned char g_static_hist_scratch[STATIC_SCRATCH_BYTES];

static std::mutex g_static_mutex;
static void* g_static_ptr[64];          // per device: the array's device address (nullptr: not asked for yet)

static int32_t static_hist_scratch(void** out)
{
    int dev = -1;
    HEPK_CUDA_TRY(cudaGetDevice(&dev));
    if (dev < 0 || dev >= 64) {
        set_error("hepk_fill_histogram_w2_static: device %d is beyond the 64 the library keeps track of", dev);
        return HEPK_ERR_UNSUPPORTED;
    }
    std::lock_guard<std::mutex> lock(g_static_mutex);
    if (!g_static_ptr[dev]) {
        void* p = nullptr;
        HEPK_CUDA_TRY(cudaGetSymbolAddress(&p, g_static_hist_scratch));
        g_static_ptr[dev] = p;
    }
    *out = g_static_ptr[dev];
    return HEPK_OK;
}
}  // namespace hepk

extern "C" size_t hepk_static_hist_scratch_bytes(void) { return hepk::STATIC_SCRATCH_BYTES; }

extern "C" int32_t hepk_fill_histogram_w2_static(const float* data, const float* weights, int64_t n, const float* edges,
                                                 int32_t nbins, float* sumw, float* sumw2, int64_t* counts, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges && nbins >= 1, "edges is NULL or nbins < 1");
    if (nbins > HEPK_STATIC_HIST_MAX_BINS) {
        set_error("hepk_fill_histogram_w2_static: nbins = %d exceeds the %d bins the library's own scratch holds "
                  "(use hepk_fill_histogram_w2 with a workspace)", nbins, (int)HEPK_STATIC_HIST_MAX_BINS);
        return HEPK_ERR_UNSUPPORTED;
    }
    HEPK_REQUIRE(n == 0 || data, "data is NULL");
    void* scratch = nullptr;
    const int32_t rc = static_hist_scratch(&scratch);
    if (rc != HEPK_OK) return rc;
    // (hist_fill_launch clears the part of the scratch it uses on the stream before the fill: the array keeps the
    // last call's contents)
    return hist_fill_launch("hepk_fill_histogram_w2_static", data, nullptr, weights, n, edges, nbins, nullptr, 0, sumw, sumw2,
                            (long long*)counts, scratch, STATIC_SCRATCH_BYTES, (cudaStream_t)stream);
}

extern "C" int32_t hepk_fill_histogram_2d_w2(const float* x, const float* y, const float* weights, int64_t n,
                                             const float* edges_x, int32_t nx, const float* edges_y, int32_t ny,
                                             float* sumw, float* sumw2, int64_t* counts, void* workspace, size_t workspace_bytes,
                                             void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges_x && edges_y && nx >= 1 && ny >= 1, "edges are NULL or an axis has no bins");
    if ((long long)(nx + 2) * (ny + 2) > 16384) {
        set_error("hepk_fill_histogram_2d_w2: (nx+2)*(ny+2) = %lld exceeds 16384", (long long)(nx + 2) * (ny + 2));
        return HEPK_ERR_UNSUPPORTED;
    }
    HEPK_REQUIRE(n == 0 || (x && y), "x/y is NULL");
    return hist_fill_launch("hepk_fill_histogram_2d_w2", x, y, weights, n, edges_x, nx, edges_y, ny, sumw, sumw2,
                            (long long*)counts, workspace, workspace_bytes, (cudaStream_t)stream);
}

extern "C" int32_t hepk_event_weight_lookup(const float* w_in, const float* x, int64_t n, const float* edges, int32_t nbins,
                                            const float* table, float* w_out, void* stream)
{
    HEPK_REQUIRE(n >= 0, "n < 0");
    HEPK_REQUIRE(edges && table && nbins >= 1, "edges/table is NULL or nbins < 1");
    if ((size_t)(2 * nbins + 1) * 4 > 200 * 1024) {
        set_error("hepk_event_weight_lookup: %d bins do not fit 200 KB of shared memory", nbins);
        return HEPK_ERR_UNSUPPORTED;
    }
    if (n == 0) return HEPK_OK;
    HEPK_REQUIRE(x && w_out, "x/w_out is NULL");
    const size_t smem = (size_t)(2 * nbins + 1) * 4;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(dev::event_weight_lookup_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
    dev::event_weight_lookup_kernel<<<grid_for_items((n + 3) / 4), 256, smem, (cudaStream_t)stream>>>(w_in, x, n, edges, nbins,
                                                                                                    table, w_out); count_launch();
    HEPK_CUDA_TRY(cudaGetLastError());
    return HEPK_OK;
}

extern "C" int32_t hepk_probe_shared_atomics(int32_t warps_per_sm, int32_t nbins, void* scratch, double* lane_atomics_per_second)
{
    HEPK_REQUIRE(warps_per_sm >= 1 && warps_per_sm <= 32 && nbins >= 32 && nbins <= 32768, "warps 1..32, bins 32..32768");
    HEPK_REQUIRE(scratch && lane_atomics_per_second, "scratch/result is NULL");
    auto kern = dev::probe_shared_atomics_kernel;
    HEPK_CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, nbins * 4));
    const int iters = 20000, grid = sm_count();
    cudaEvent_t a, b;
    HEPK_CUDA_TRY(cudaEventCreate(&a));
    HEPK_CUDA_TRY(cudaEventCreate(&b));
    kern<<<grid, warps_per_sm * 32, nbins * 4>>>(200, nbins, (unsigned int*)scratch); count_launch();
    cudaEventRecord(a);
    kern<<<grid, warps_per_sm * 32, nbins * 4>>>(iters, nbins, (unsigned int*)scratch); count_launch();
    cudaEventRecord(b);
    HEPK_CUDA_TRY(cudaEventSynchronize(b));
    float ms = 0.f;
    cudaEventElapsedTime(&ms, a, b);
    cudaEventDestroy(a); cudaEventDestroy(b);
    *lane_atomics_per_second = (double)iters * warps_per_sm * 32 * grid / ((double)ms * 1e-3);
    return HEPK_OK;
}
