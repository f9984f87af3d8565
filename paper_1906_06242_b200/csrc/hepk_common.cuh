// hepk_common.cuh — shared host/device helpers of libhepk (sm_100a only).
//
// Nothing here is shared with the CPU oracle (oracle/): the two sides have independent sources.
#pragma once

#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include <stdio.h>

#include "../../include/hepk.h"

// ------------------------------------------------------------------------------------------ host side
namespace hepk {

void set_error(const char* fmt, ...);
int32_t cuda_fail(cudaError_t e, const char* what);
int sm_count();                 // SMs of the current device (cached per device)
int max_smem_optin();           // max opt-in dynamic shared memory per CTA
void profile_mark(cudaStream_t st, int which);   // no-op unless hepk_profile_begin() is active (which: 0 before, 1 after)
void count_launch();            // one more kernel of this library enqueued (hepk_kernel_launches)

#define HEPK_CUDA_TRY(call)                                         \
    do {                                                            \
        cudaError_t _e = (call);                                    \
        if (_e != cudaSuccess) return ::hepk::cuda_fail(_e, #call); \
    } while (0)

#define HEPK_REQUIRE(cond, msg)                              \
    do {                                                     \
        if (!(cond)) {                                       \
            ::hepk::set_error("%s: %s", __func__, msg);      \
            return HEPK_ERR_INVALID;                         \
        }                                                    \
    } while (0)

static inline bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }

}  // namespace hepk

// ------------------------------------------------------------------------------------------ device side
namespace hepk {
namespace dev {

// float32 constants of the dphi wrap: PI_F = 0x40490FDB, TWO_PI_F = 0x40C90FDB (R6).
#define HEPK_PI_F 3.14159274101257324f
#define HEPK_TWO_PI_F 6.28318548202514648f

__device__ __forceinline__ uint32_t smem_u32(const void* p)
{
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}

// ---- mbarrier + TMA 1-D bulk copy (cp.async.bulk, SASS UBLKCP) -------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init()
{
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
// generic-proxy accesses to shared memory before this point are ordered before later async-proxy (TMA) accesses
__device__ __forceinline__ void fence_proxy_async_smem()
{
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_%=:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra DONE_%=;\n"
        "bra WAIT_%=;\n"
        "DONE_%=:\n"
        "}\n" ::"r"(smem_u32(bar)),
        "r"(parity)
        : "memory");
}
// global -> shared bulk copy; dst, src 16-byte aligned, bytes a multiple of 16
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

__device__ __forceinline__ void bulk_g2s_addr(uint32_t dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst_smem),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}

// shared-memory reductions in the shared state space (a generic-address atomicAdd on shared memory goes through an
// address-space dispatch first)
__device__ __forceinline__ void red_shared_add_u32(void* p, unsigned int v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(smem_u32(p)), "r"(v) : "memory");
}
__device__ __forceinline__ void red_shared_add_f32(void* p, float v)
{
    asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(smem_u32(p)), "f"(v) : "memory");
}

// the same on a shared-memory byte address (smem_u32 taken once outside the loop: the conversion is three instructions)
__device__ __forceinline__ void red_shared_add_u32_at(uint32_t a, unsigned int v)
{
    asm volatile("red.shared.add.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory");
}
__device__ __forceinline__ void red_shared_add_f32_at(uint32_t a, float v)
{
    asm volatile("red.shared.add.f32 [%0], %1;" ::"r"(a), "f"(v) : "memory");
}

// ---- staging a slice [l0, l1) of a column into shared memory -----------------------------------
// Element l of `col` lands at dst[l - a0], a0 <= l0 chosen so that the 16-byte aligned body of the slice
// can be moved by ONE bulk copy; the ragged head (col not 16-byte aligned near element 0) and the tail
// beyond the last full 16-byte group of the column go through ordinary loads.  Works for any
// sizeof(T)-aligned column pointer.  dst must be 16-byte aligned with room for (l1-l0) + 2*(16/sizeof(T)) elements.
template <typename T>
struct StageGeom {
    static constexpr int A = 16 / (int)sizeof(T);
    long long a0;      // column index mapped to dst[0] (may be negative)
    long long bulk0;   // bulk body [bulk0, bulk1)
    long long bulk1;
    __device__ __forceinline__ StageGeom(const T* col, long long l0, long long l1, long long n_total)
    {
        const int mis = (int)((reinterpret_cast<uintptr_t>(col) / sizeof(T)) % A);
        a0 = l0 - ((l0 + mis) % A);
        long long first = a0 < 0 ? a0 + A : a0;
        long long ceil1 = l1 + ((A - (int)((l1 + mis) % A)) % A);
        long long floorn = n_total - ((n_total + mis) % A);
        long long last = ceil1 < floorn ? ceil1 : floorn;
        bulk0 = first;
        bulk1 = last > first ? last : first;
    }
};

// Issue the copies of one column.  Called by ALL threads of the CTA (uniform arguments).
// Thread `issuer` issues the bulk copy and returns its byte count (others return 0); the scalar head/tail
// elements are copied by the first few threads and become visible at the next __syncthreads().
template <typename T>
__device__ __forceinline__ uint32_t stage_column(T* dst, const T* __restrict__ col, long long l0, long long l1,
                                                 long long n_total, uint64_t* bar, int tid, int issuer,
                                                 long long* a0_out)
{
    StageGeom<T> g(col, l0, l1, n_total);
    *a0_out = g.a0;
    uint32_t bytes = 0;
    if (tid == issuer && g.bulk1 > g.bulk0 && l1 > l0) {
        bytes = (uint32_t)((g.bulk1 - g.bulk0) * (long long)sizeof(T));
        bulk_g2s(dst + (g.bulk0 - g.a0), col + g.bulk0, bytes, bar);
    }
    // scalar head [l0, min(bulk0, l1)) and tail [max(bulk1, l0), l1)
    const long long head_end = g.bulk0 < l1 ? g.bulk0 : l1;
    const long long head_n = head_end > l0 ? head_end - l0 : 0;
    const long long tail_beg = g.bulk1 > l0 ? g.bulk1 : l0;
    const long long tail_n = (l1 > tail_beg && g.bulk0 <= l1) ? l1 - tail_beg : 0;
    if (tid < head_n) dst[l0 + tid - g.a0] = col[l0 + tid];
    else if (tid < head_n + tail_n) dst[tail_beg + (tid - head_n) - g.a0] = col[tail_beg + (tid - head_n)];
    return bytes;
}

// ---- exact-class float32 arithmetic (one IEEE rn operation per node, never contracted) ------------
// dR^2 = deta^2 + dphi^2 with the single-step phi wrap.  |dphi| > PI_F  <=>  the oracle's two-sided test
// (dphi > PI_F or dphi <= -PI_F), except at dphi == -PI_F exactly, where (-PI_F + 2PI_F)^2 == PI_F^2 ==
// (-PI_F)^2 bit for bit; and (|d| - 2PI_F)^2 == (d -/+ 2PI_F)^2 because negation is exact.
__device__ __forceinline__ float dr2_exact(float eta_a, float phi_a, float eta_b, float phi_b)
{
    const float deta = __fsub_rn(eta_a, eta_b);
    const float ad = fabsf(__fsub_rn(phi_a, phi_b));
    // the wrapped magnitude is min(ad, |ad - 2PI_F|): ad > PI_F => |t| <= PI_F < ad (rn is monotone), ad < PI_F =>
    // |t| >= PI_F > ad, and at ad == PI_F both are PI_F; two instructions (|.| is a free operand modifier)
    const float w = fminf(ad, fabsf(__fsub_rn(ad, HEPK_TWO_PI_F)));
    return __fadd_rn(__fmul_rn(deta, deta), __fmul_rn(w, w));
}

// B(v): b with edges[b] <= v < edges[b+1]; clamped (v < edges[0] -> 0; v >= edges[n] or NaN -> n-1).
__device__ __forceinline__ int find_bin_clamped(float v, const float* edges, int n)
{
    if (v < edges[0]) return 0;
    if (!(v < edges[n])) return n - 1;
    int lo = 0, hi = n;
    while (hi - lo > 1) {
        const int mid = (lo + hi) >> 1;
        if (v >= edges[mid]) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- lookup axes without a search --------------------------------------------------------------------
// An axis whose edges are uniform in v (mode 1) or in log2 v (mode 2) to within 0.45 bins lets B(v) be guessed
// arithmetically to within one bin (the log2 approximation is good to ~1e-5 bins) and fixed with one +-1 step
// against the edges, which makes the result exact.  classify_axis is called by ALL threads of the CTA (it uses
// __syncthreads_and) on edges already staged in shared memory.
struct AxisGuess { int mode; float lo, inv; };      // mode 0: binary search

__device__ __forceinline__ AxisGuess classify_axis(const float* s_edges, int n)
{
    const float lo = s_edges[0], hi = s_edges[n];
    const float inv1 = (float)n / (hi - lo);
    const float l0 = __log2f(lo), inv2 = (float)n / (__log2f(hi) - l0);
    bool ok1 = (hi > lo) && (inv1 > 0.0f) && (inv1 < CUDART_INF_F);
    // (mode 2 wants a NORMAL first edge: pad_axis_find's log2 flushes denormal values to zero, which is only right when
    // every denormal value lies below the axis)
    bool ok2 = (lo >= 1.17549435e-38f) && (hi > lo) && (inv2 > 0.0f) && (inv2 < CUDART_INF_F);
    for (int i = threadIdx.x; i <= n; i += blockDim.x) {
        ok1 = ok1 && (fabsf((s_edges[i] - lo) * inv1 - (float)i) <= 0.45f);
        ok2 = ok2 && (fabsf((__log2f(s_edges[i]) - l0) * inv2 - (float)i) <= 0.45f);
    }
    ok1 = __syncthreads_and(ok1);
    ok2 = __syncthreads_and(ok2);
    AxisGuess a;
    a.mode = ok1 ? 1 : (ok2 ? 2 : 0);
    a.lo = ok1 ? lo : l0;
    a.inv = ok1 ? inv1 : inv2;
    return a;
}

__device__ __forceinline__ int find_bin_guess(float v, const float* edges, int n, const AxisGuess& a)
{
    if (a.mode == 0) return find_bin_clamped(v, edges, n);
    const float pos = a.mode == 1 ? v : __log2f(v);
    int g = (int)((pos - a.lo) * a.inv);              // NaN -> 0, +-inf saturate
    g = max(0, min(g, n - 1));
    const float e0 = edges[g], e1 = edges[g + 1];
    g += (v >= e1) ? 1 : 0;
    g -= (v < e0) ? 1 : 0;
    g = max(0, min(g, n - 1));
    return (v != v) ? n - 1 : g;
}

// Slot of an axis (0 underflow, 1 + b, n + 1 overflow / NaN) through the arithmetic bin guess (linear or log2 axis,
// exact after one +-1 step; binary search otherwise).
__device__ __forceinline__ int axis_slot(float v, const float* s_e, int n, const AxisGuess& ax)
{
    const int b = find_bin_guess(v, s_e, n, ax);
    int s = 1 + b;
    s = (v < s_e[0]) ? 0 : s;
    s = !(v < s_e[n]) ? n + 1 : s;
    return s;
}

// ---- padded axes: the +-1 step with no clamps, range tests or NaN selects ------------------------------
// A second copy of the edges whose ends absorb every special case, so that the guess needs one fused multiply-add, a
// float clamp, a conversion, two loads and two compare-and-adjust steps (13 instructions; find_bin_guess / axis_slot
// take 25-30 with their range tests, clamps and NaN selects, and a run-time mode test).
//   SLOTS (histograms):  pad[0] = -inf, pad[1 + i] = edges[i] (i = 0..n), pad[n + 2] = NaN;
//                        slot s in [0, n + 1] is the one with pad[s] <= v < pad[s + 1]   (0 underflow, n + 1 overflow)
//   bins (clamped lookups): pad[0] = -inf, pad[i] = edges[i] (i = 1..n-1), pad[n] = NaN;
//                        bin b in [0, n - 1] is the one with pad[b] <= v < pad[b + 1]     (B(v) of find_bin_clamped)
// No comparison with NaN is true, so the last slot / bin takes everything at or beyond the last edge, and a NaN value
// (guess = top through fminf(NaN, top) = top, no comparison moves it) lands there too, as the readings R5 / R9 ask.
// The guess is floor of the position in slot units, good to +-1 on an axis classify_axis accepted (mode 1 or 2), and
// the step against the REAL edges makes the result exact.  AXIS is the mode, fixed at compile time by the caller;
// AXIS == 0 takes the general functions above on the unpadded edges.
template <bool SLOTS>
__device__ __forceinline__ int pad_axis_words(int n) { return SLOTS ? n + 3 : n + 1; }

template <bool SLOTS>
__device__ __forceinline__ void pad_axis_fill(float* s_pad, const float* __restrict__ edges, int n)     // all threads of the CTA
{
    const int last = SLOTS ? n + 2 : n;
    for (int i = threadIdx.x; i <= last; i += blockDim.x)
        s_pad[i] = i == 0 ? -CUDART_INF_F : (i == last ? CUDART_NAN_F : edges[SLOTS ? i - 1 : i]);
}

// top = (float)(n + 1) for slots, (float)(n - 1) for bins
template <int AXIS, bool SLOTS>
__device__ __forceinline__ int pad_axis_find(float v, const float* s_edges, const float* s_pad, int n, const AxisGuess& a, float top)
{
    if (AXIS == 0) return SLOTS ? axis_slot(v, s_edges, n, a) : find_bin_guess(v, s_edges, n, a);
    const float one = SLOTS ? 1.0f : 0.0f;
    float pos;
    if (AXIS == 1) {
        pos = fmaf(v - a.lo, a.inv, one);
    } else {
        // One MUFU and no branch: lg2.approx.ftz gives -inf for zeros and denormals (clamped to the first slot below, where
        // they belong: the first edge is a normal float), NaN for NaN (-> top, as for any NaN) and NaN for negative values,
        // which belong in the first slot instead: one select.  (__log2f without -ftz is five instructions, and the
        // three-way test on v a branch.)
        float lg;
        asm("lg2.approx.ftz.f32 %0, %1;" : "=f"(lg) : "f"(v));
        pos = fmaf(lg - a.lo, a.inv, one);
        pos = v < 0.0f ? 0.0f : pos;
    }
    int s = (int)fmaxf(fminf(pos, top), 0.0f);
    const float e0 = s_pad[s], e1 = s_pad[s + 1];
    s += (v >= e1) ? 1 : 0;
    s -= (v < e0) ? 1 : 0;
    return s;
}

// Calls f(tag_x, tag_y) with the axis modes as compile-time tags when both axes have an arithmetic guess, and with
// (0, 0) (the general functions, which test the mode at run time) otherwise.  The modes are uniform over the CTA.
template <int N> struct AxisTag { static constexpr int value = N; };
template <class F>
__device__ __forceinline__ void dispatch_axes(int mode_x, int mode_y, F&& f)
{
    if (mode_x == 1 && mode_y == 1) f(AxisTag<1>{}, AxisTag<1>{});
    else if (mode_x == 1 && mode_y == 2) f(AxisTag<1>{}, AxisTag<2>{});
    else if (mode_x == 2 && mode_y == 1) f(AxisTag<2>{}, AxisTag<1>{});
    else if (mode_x == 2 && mode_y == 2) f(AxisTag<2>{}, AxisTag<2>{});
    else f(AxisTag<0>{}, AxisTag<0>{});
}

template <class F>
__device__ __forceinline__ void dispatch_axis(int mode, F&& f)
{
    if (mode == 1) f(AxisTag<1>{});
    else if (mode == 2) f(AxisTag<2>{});
    else f(AxisTag<0>{});
}

// Histogram slot: 0 underflow, 1+b, nbins+1 overflow/NaN.  Arithmetic guess for (near-)uniform axes,
// verified against the edges; anything the guess gets wrong falls back to the binary search, so the
// result is exact for any ascending edges.
__device__ __forceinline__ int hist_slot(float x, const float* edges, int nbins, float lo, float inv_w)
{
    if (x < lo) return 0;
    if (!(x < edges[nbins])) return nbins + 1;
    int g = (int)((x - lo) * inv_w);
    g = g < 0 ? 0 : (g > nbins - 1 ? nbins - 1 : g);
    if (edges[g] <= x) {
        if (x < edges[g + 1]) return 1 + g;
        if (g + 2 <= nbins && x < edges[g + 2]) return 2 + g;
    } else if (g > 0 && edges[g - 1] <= x) {
        return g;
    }
    int a = 0, b = nbins;
    while (b - a > 1) {
        const int mid = (a + b) >> 1;
        if (x >= edges[mid]) a = mid; else b = mid;
    }
    return 1 + a;
}

// ---- tolerance-class float32 pair mass, cancellation-free form ---------------------------------
// M^2 = m1^2 + m2^2 + 2 pt1 pt2 [ ch1 ch2 t + 2 (sinh^2(deta/2) + sin^2(dphi/2)) ],
//   ch_i = cosh(eta_i), x_i = (m_i / (pt_i ch_i))^2, x = x1 + x2 + x1 x2, t = x / (sqrt(1+x) + 1)
// which equals (E1+E2)^2 - |p1+p2|^2 for E = sqrt(pt^2 cosh^2 eta + m^2) with every term >= 0
// (DESIGN.md "pair mass"): E1E2 = pt1 pt2 ch1 ch2 (1+t), cosh(deta) - cos(dphi) = 2 sinh^2 + 2 sin^2.
// dphi is reduced to [-pi, pi] with an error-free subtraction and a two-term 2*pi so that jets
// straddling the +-pi seam keep full relative accuracy.
__device__ __forceinline__ float pair_mass_f32(float pt1, float eta1, float phi1, float m1,
                                               float pt2, float eta2, float phi2, float m2)
{
    const float e1 = expf(eta1), e2 = expf(eta2);
    const float ch1 = 0.5f * (e1 + 1.0f / e1);
    const float ch2 = 0.5f * (e2 + 1.0f / e2);
    // sinh(deta/2) through expm1 (no cancellation for small deta)
    const float hx = 0.5f * fabsf(eta1 - eta2);
    const float em1 = expm1f(hx);
    const float sh = 0.5f * (em1 + em1 / (em1 + 1.0f));
    // dphi = phi1 - phi2 as an unevaluated sum d + dl (TwoSum), wrapped by 2*pi = TWO_PI_F + TWO_PI_LO
    float d = __fsub_rn(phi1, phi2);
    const float bb = __fsub_rn(d, phi1);
    float dl = __fsub_rn(__fsub_rn(phi1, __fsub_rn(d, bb)), __fadd_rn(phi2, bb));
    const float TWO_PI_LO = -1.7484555e-07f;   // 2*pi - TWO_PI_F
    if (d > HEPK_PI_F) { d = __fsub_rn(d, HEPK_TWO_PI_F); dl = __fsub_rn(dl, TWO_PI_LO); }
    else if (d < -HEPK_PI_F) { d = __fadd_rn(d, HEPK_TWO_PI_F); dl = __fadd_rn(dl, TWO_PI_LO); }
    const float sn = sinf(0.5f * (d + dl));
    const float r1 = m1 / (pt1 * ch1), r2 = m2 / (pt2 * ch2);
    const float x1 = r1 * r1, x2 = r2 * r2;
    const float x = x1 + x2 + x1 * x2;
    const float t = x / (sqrtf(1.0f + x) + 1.0f);
    const float bracket = ch1 * ch2 * t + 2.0f * (sh * sh + sn * sn);
    const float msq = m1 * m1 + m2 * m2 + 2.0f * pt1 * pt2 * bracket;
    return sqrtf(fmaxf(msq, 0.0f));
}

// hardware approximations (1-2 ulp each)
__device__ __forceinline__ float ex2_approx(float x)
{
    float r;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rcp_approx(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}


// pair_mass_f32 (hepk_common.cuh) with the transcendental pieces written out for the ranges that occur here (exp
// through ex2.approx, sinh by a Taylor polynomial for h <= 1, sin by an odd polynomial on [-pi/2, pi/2]) and the
// hardware approximations (ex2, rcp, sqrt: 1-2 ulp each) in place of the library calls; tolerance class, every term of M^2 >= 0, ~60 instructions.
__device__ __forceinline__ float pair_mass_lean(float pt1, float eta1, float phi1, float m1,
                                                float pt2, float eta2, float phi2, float m2)
{
    const float LOG2E = 1.44269504088896341f;
    const float e1 = ex2_approx(eta1 * LOG2E), e2 = ex2_approx(eta2 * LOG2E);
    const float ch1 = 0.5f * (e1 + rcp_approx(e1));
    const float ch2 = 0.5f * (e2 + rcp_approx(e2));
    const float h = 0.5f * fabsf(eta1 - eta2);
    const float h2 = h * h;
    float sh_small = fmaf(h2, 1.0f / 39916800.0f, 1.0f / 362880.0f);
    sh_small = fmaf(sh_small, h2, 1.0f / 5040.0f);
    sh_small = fmaf(sh_small, h2, 1.0f / 120.0f);
    sh_small = fmaf(sh_small, h2, 1.0f / 6.0f);
    sh_small = fmaf(sh_small * h2, h, h);
    const float eh = ex2_approx(h * LOG2E);
    const float sh_big = 0.5f * (eh - rcp_approx(eh));
    const float sh = h <= 1.0f ? sh_small : sh_big;
    float d = __fsub_rn(phi1, phi2);
    const float bb = __fsub_rn(d, phi1);
    float dl = __fsub_rn(__fsub_rn(phi1, __fsub_rn(d, bb)), __fadd_rn(phi2, bb));
    const float TWO_PI_LO = -1.7484555e-07f;   // 2*pi - TWO_PI_F
    if (d > HEPK_PI_F) { d = __fsub_rn(d, HEPK_TWO_PI_F); dl = __fsub_rn(dl, TWO_PI_LO); }
    else if (d < -HEPK_PI_F) { d = __fadd_rn(d, HEPK_TWO_PI_F); dl = __fadd_rn(dl, TWO_PI_LO); }
    const float x_ = 0.5f * (d + dl), z = x_ * x_;
    float sn = fmaf(z, 1.0f / 6227020800.0f, -1.0f / 39916800.0f);
    sn = fmaf(sn, z, 1.0f / 362880.0f);
    sn = fmaf(sn, z, -1.0f / 5040.0f);
    sn = fmaf(sn, z, 1.0f / 120.0f);
    sn = fmaf(sn, z, -1.0f / 6.0f);
    sn = fmaf(sn * z, x_, x_);
    const float r1 = m1 * rcp_approx(pt1 * ch1), r2 = m2 * rcp_approx(pt2 * ch2);
    const float x1 = r1 * r1, x2 = r2 * r2;
    const float x = x1 + x2 + x1 * x2;
    const float t = x * rcp_approx(sqrt_approx(1.0f + x) + 1.0f);
    const float bracket = ch1 * ch2 * t + 2.0f * (sh * sh + sn * sn);
    const float msq = m1 * m1 + m2 * m2 + 2.0f * pt1 * pt2 * bracket;
    return sqrt_approx(fmaxf(msq, 0.0f));
}


// The defining form in float64 (include/hepk.h, hepk_pair_invmass).  Used only where the float32 result above
// lands within its own error band of a histogram edge, so that the bin is decided by the float32 rounding of
// the float64 value — the precision the result is defined in (R16).
static __device__ __noinline__ float pair_mass_f64(float pt1, float eta1, float phi1, float m1,
                                            float pt2, float eta2, float phi2, float m2)
{
    const double a1 = pt1, a2 = pt2;
    double s1, c1, s2, c2;
    sincos((double)phi1, &s1, &c1);
    sincos((double)phi2, &s2, &c2);
    const double ch1 = cosh((double)eta1), ch2 = cosh((double)eta2);
    const double e = sqrt(a1 * a1 * ch1 * ch1 + (double)m1 * (double)m1) + sqrt(a2 * a2 * ch2 * ch2 + (double)m2 * (double)m2);
    const double px = a1 * c1 + a2 * c2, py = a1 * s1 + a2 * s2;
    const double pz = a1 * sinh((double)eta1) + a2 * sinh((double)eta2);
    double msq = e * e - px * px - py * py - pz * pz;
    if (!(msq > 0.0)) msq = 0.0;
    return (float)sqrt(msq);
}

// relative half-width of the band around a histogram edge inside which pair_mass_f32 is not trusted to pick the
// bin (its measured worst error is 1.1e-6 relative; R16)
#define HEPK_MASS_GUARD_REL 8e-6f
#define HEPK_MASS_GUARD_ABS 1e-6f

// ---- per-event running state of the reductions (count, sum, min, top-2 with first-index ties) ------
struct Top2 {
    float b1, b2;
    int i1, i2;
    __device__ __forceinline__ void init() { b1 = b2 = -CUDART_INF_F; i1 = i2 = -1; }
    // strict > keeps the smallest index among equal values, for both places
    __device__ __forceinline__ void push(float p, int k)
    {
        if (p > b1) { b2 = b1; i2 = i1; b1 = p; i1 = k; }
        else if (p > b2) { b2 = p; i2 = k; }
    }
    // general data (may hold NaN or -inf): NaN skipped, the first element always taken (oracle's argmax rule)
    __device__ __forceinline__ void push_any(float p, int k)
    {
        if (p != p) return;
        if (i1 < 0 || p > b1) { b2 = b1; i2 = i1; b1 = p; i1 = k; }
        else if (i2 < 0 || p > b2) { b2 = p; i2 = k; }
    }
};

}  // namespace dev
}  // namespace hepk
