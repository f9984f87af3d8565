// hepk_stream.cu — hepk_analysis_chain_host: the chain on HOST-resident arrays, streamed to the device in
// batches of events (Fig. 1: "the cache is loaded in batches of a few GB of contiguous
// 1-dimensional arrays").  Per batch: host->device copies of the offsets slices and column slices, the fused
// chain kernel, device->host copies of the per-event outputs.  With overlap, two buffer sets on two streams
// let the copies of batch b+1 run under the kernels of batch b.
#include <string.h>

#include <vector>

#include "hepk_common.cuh"

namespace hepk {

struct SlotLayout {
    size_t joff, moff, eoff;
    size_t jcol[4], mcol[3], ecol[3];
    size_t weights, evw_x;
    size_t out_i[2], out_f[5], out_mask;
    size_t hist_sumw, hist_sumw2, hist_counts, chain_ws;
    size_t bytes;
};

struct HostPlan {
    long long B, n_batches, maxJ, maxM, maxE;
    long long spv, n_sumw, n_sumw2, n_cnt;
    size_t chain_ws_bytes;
    size_t shared_bytes;          // calib + axis edges + event-weight lookup
    size_t cal_pt, cal_eta, cal_tab, axis[HEPK_N_OBS], evw_edges, evw_table;
    SlotLayout slot;
};

static size_t up256(size_t x) { return (x + 255) / 256 * 256; }

static bool make_plan(const hepk_chain_desc* d, long long B, HostPlan* p)
{
    memset(p, 0, sizeof(*p));
    if (B < 1) B = 1;
    if (B > d->n_events && d->n_events > 0) B = d->n_events;
    p->B = B;
    p->n_batches = (d->n_events + B - 1) / B;
    const bool has_el = d->electrons.offsets != nullptr;
    for (long long b = 0; b < p->n_batches; ++b) {
        const long long e0 = b * B, e1 = (e0 + B < d->n_events) ? e0 + B : d->n_events;
        const long long nj = d->jets.offsets[e1] - d->jets.offsets[e0];
        const long long nm = d->muons.offsets[e1] - d->muons.offsets[e0];
        const long long ne = has_el ? d->electrons.offsets[e1] - d->electrons.offsets[e0] : 0;
        if (nj < 0 || nm < 0 || ne < 0) return false;
        if (nj > p->maxJ) p->maxJ = nj;
        if (nm > p->maxM) p->maxM = nm;
        if (ne > p->maxE) p->maxE = ne;
    }
    long long spv = 0;
    for (int o = 0; o < HEPK_N_OBS; ++o)
        if (d->axis_edges[o]) spv += d->axis_nbins[o] + 2;
    p->spv = spv;
    p->n_sumw = d->hist_sumw ? spv * d->n_variants * d->n_wvar : 0;
    p->n_sumw2 = d->hist_sumw2 ? spv * d->n_variants * d->n_wvar : 0;
    p->n_cnt = d->hist_counts ? spv * d->n_variants : 0;
    p->chain_ws_bytes = hepk_chain_workspace_bytes(d);      // depends on which histogram outputs are non-NULL only

    size_t o = 0;
    auto take = [&](size_t bytes) { size_t r = o; o += up256(bytes); return r; };
    if (d->calib_table) {
        p->cal_pt = take((size_t)(d->calib_npt + 1) * 4);
        p->cal_eta = take((size_t)(d->calib_neta + 1) * 4);
        p->cal_tab = take((size_t)d->calib_npt * d->calib_neta * 4);
    }
    for (int ob = 0; ob < HEPK_N_OBS; ++ob)
        if (d->axis_edges[ob]) p->axis[ob] = take((size_t)(d->axis_nbins[ob] + 1) * 4);
    if (d->evw_table) {
        p->evw_edges = take((size_t)(d->evw_nbins + 1) * 4);
        p->evw_table = take((size_t)d->evw_nbins * 4);
    }
    p->shared_bytes = o;

    SlotLayout& s = p->slot;
    o = 0;
    const int V = d->n_variants, W = d->n_wvar;
    s.joff = take((size_t)(B + 1) * 8);
    s.moff = take((size_t)(B + 1) * 8);
    s.eoff = take(has_el ? (size_t)(B + 1) * 8 : 0);
    for (int c = 0; c < 4; ++c) s.jcol[c] = take((size_t)p->maxJ * 4);
    for (int c = 0; c < 3; ++c) s.mcol[c] = take((size_t)p->maxM * 4);
    for (int c = 0; c < 3; ++c) s.ecol[c] = take((size_t)p->maxE * 4);
    s.weights = take(d->weights ? (size_t)W * B * 4 : 0);
    s.evw_x = take(d->evw_table ? (size_t)B * 4 : 0);
    for (int c = 0; c < 2; ++c) s.out_i[c] = take((size_t)V * B * 4);
    for (int c = 0; c < 5; ++c) s.out_f[c] = take((size_t)V * B * 4);
    s.out_mask = take(d->out_jet_mask ? (size_t)V * p->maxJ : 0);
    s.hist_sumw = take((size_t)p->n_sumw * 4);
    s.hist_sumw2 = take((size_t)p->n_sumw2 * 4);
    s.hist_counts = take((size_t)p->n_cnt * 8);
    s.chain_ws = take(p->chain_ws_bytes);
    s.bytes = o;
    return true;
}

// Two copy/compute streams owned by ONE call (created on the current device, destroyed before it returns), so
// concurrent calls from several host threads or on several devices share nothing.
struct CallStreams {
    cudaStream_t s[2] = {nullptr, nullptr};
    bool own = false;
    ~CallStreams()
    {
        if (!own) return;
        for (int i = 0; i < 2; ++i)
            if (s[i]) { cudaStreamSynchronize(s[i]); cudaStreamDestroy(s[i]); }   // drains work in flight on an error return
    }
};

}  // namespace hepk

using namespace hepk;

extern "C" size_t hepk_chain_host_workspace_bytes(const hepk_chain_desc* d, int64_t batch_events)
{
    if (!d || d->n_events <= 0 || !d->jets.offsets || !d->muons.offsets || d->n_variants < 1 || d->n_wvar < 1) return 0;
    HostPlan p;
    if (!make_plan(d, batch_events, &p)) return 0;
    return p.shared_bytes + 2 * p.slot.bytes + 256;
}

extern "C" int32_t hepk_analysis_chain_host(const hepk_chain_desc* d, int64_t batch_events, int32_t overlap,
                                            void* workspace, size_t workspace_bytes, void* stream)
{
    HEPK_REQUIRE(d != nullptr, "descriptor is NULL");
    HEPK_REQUIRE(d->n_events >= 0, "n_events < 0");
    HEPK_REQUIRE(batch_events >= 1, "batch_events < 1");
    HEPK_REQUIRE(d->n_variants >= 1 && d->n_variants <= HEPK_MAX_VARIANTS, "n_variants out of range");
    HEPK_REQUIRE(d->n_wvar >= 1 && d->n_wvar <= HEPK_MAX_WVAR, "n_wvar out of range");
    if (d->n_events == 0) return HEPK_OK;
    HEPK_REQUIRE(d->jets.offsets && d->muons.offsets, "jets/muons offsets are NULL");
    HostPlan p;
    HEPK_REQUIRE(make_plan(d, batch_events, &p), "offsets are not monotone");
    const int n_slots = overlap ? 2 : 1;
    HEPK_REQUIRE(workspace != nullptr, "workspace is NULL");
    HEPK_REQUIRE(workspace_bytes >= p.shared_bytes + n_slots * p.slot.bytes, "workspace too small");
    HEPK_REQUIRE(((uintptr_t)workspace & 255) == 0, "workspace must be 256-byte aligned");

    cudaStream_t user = (cudaStream_t)stream;
    CallStreams cs;
    cudaStream_t st[2] = {user, user};
    if (overlap) {
        cs.own = true;
        for (int i = 0; i < 2; ++i) HEPK_CUDA_TRY(cudaStreamCreateWithFlags(&cs.s[i], cudaStreamNonBlocking));
        st[0] = cs.s[0]; st[1] = cs.s[1];
        HEPK_CUDA_TRY(cudaStreamSynchronize(user));     // earlier work of the caller's stream is complete
    }
    // on an error return after work was enqueued on the caller's stream, wait for it before handing the buffers back
    struct Drain { cudaStream_t q; bool armed; ~Drain() { if (armed) cudaStreamSynchronize(q); } } drain{user, true};
    unsigned char* base = (unsigned char*)workspace;
    unsigned char* slot_base[2] = {base + p.shared_bytes, base + p.shared_bytes + p.slot.bytes};
    const bool has_el = d->electrons.offsets != nullptr;
    const int V = d->n_variants, W = d->n_wvar;
    const long long N = d->n_events;
    const long long w_stride = d->weights_stride > 0 ? d->weights_stride : N;      // host rows
    const long long o_stride = d->out_stride > 0 ? d->out_stride : N;

    // tables shared by every batch
    hepk_chain_desc tmpl = *d;
    if (d->calib_table) {
        HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.cal_pt, d->calib_pt_edges, (size_t)(d->calib_npt + 1) * 4, cudaMemcpyHostToDevice, st[0]));
        HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.cal_eta, d->calib_eta_edges, (size_t)(d->calib_neta + 1) * 4, cudaMemcpyHostToDevice, st[0]));
        HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.cal_tab, d->calib_table, (size_t)d->calib_npt * d->calib_neta * 4, cudaMemcpyHostToDevice, st[0]));
        tmpl.calib_pt_edges = (const float*)(base + p.cal_pt);
        tmpl.calib_eta_edges = (const float*)(base + p.cal_eta);
        tmpl.calib_table = (const float*)(base + p.cal_tab);
    }
    for (int ob = 0; ob < HEPK_N_OBS; ++ob)
        if (d->axis_edges[ob]) {
            HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.axis[ob], d->axis_edges[ob], (size_t)(d->axis_nbins[ob] + 1) * 4, cudaMemcpyHostToDevice, st[0]));
            tmpl.axis_edges[ob] = (const float*)(base + p.axis[ob]);
        }
    if (d->evw_table) {
        HEPK_REQUIRE(d->evw_x && d->evw_edges && d->evw_nbins >= 1, "event-weight lookup: x, edges or bins missing");
        HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.evw_edges, d->evw_edges, (size_t)(d->evw_nbins + 1) * 4, cudaMemcpyHostToDevice, st[0]));
        HEPK_CUDA_TRY(cudaMemcpyAsync(base + p.evw_table, d->evw_table, (size_t)d->evw_nbins * 4, cudaMemcpyHostToDevice, st[0]));
        tmpl.evw_edges = (const float*)(base + p.evw_edges);
        tmpl.evw_table = (const float*)(base + p.evw_table);
    }
    for (int s = 0; s < n_slots; ++s) {
        if (p.n_sumw) HEPK_CUDA_TRY(cudaMemsetAsync(slot_base[s] + p.slot.hist_sumw, 0, (size_t)p.n_sumw * 4, st[0]));
        if (p.n_sumw2) HEPK_CUDA_TRY(cudaMemsetAsync(slot_base[s] + p.slot.hist_sumw2, 0, (size_t)p.n_sumw2 * 4, st[0]));
        if (p.n_cnt) HEPK_CUDA_TRY(cudaMemsetAsync(slot_base[s] + p.slot.hist_counts, 0, (size_t)p.n_cnt * 8, st[0]));
    }
    if (overlap) HEPK_CUDA_TRY(cudaStreamSynchronize(st[0]));   // tables visible to both streams

    int* const out_i_host[2] = {d->out_njet, d->out_argmax};
    float* const out_f_host[5] = {d->out_ht, d->out_maxpt, d->out_minpt, d->out_mjj, d->out_subpt};

    for (long long b = 0; b < p.n_batches; ++b) {
        const int s = (int)(b % n_slots);
        cudaStream_t q = st[s];
        unsigned char* sb = slot_base[s];
        const long long e0 = b * p.B, e1 = (e0 + p.B < N) ? e0 + p.B : N, nb = e1 - e0;
        hepk_chain_desc bd = tmpl;
        bd.n_events = nb;
        bd.weights_stride = 0; bd.out_stride = 0;      // the staged batch is contiguous
        auto stage_coll = [&](const hepk_collection& hc, hepk_collection& dc, size_t off_o, const size_t* col_o, int ncol) -> cudaError_t {
            const long long g0 = hc.offsets[e0], g1 = hc.offsets[e1], n = g1 - g0;
            cudaError_t e = cudaMemcpyAsync(sb + off_o, hc.offsets + e0, (size_t)(nb + 1) * 8, cudaMemcpyHostToDevice, q);
            if (e != cudaSuccess) return e;
            dc.offsets = (const int64_t*)(sb + off_o);
            dc.content_base = g0;
            dc.n_objects = n;
            const float* src[4] = {hc.pt, hc.eta, hc.phi, hc.mass};
            const float** dst[4] = {&dc.pt, &dc.eta, &dc.phi, &dc.mass};
            for (int c = 0; c < ncol; ++c) {
                *dst[c] = (const float*)(sb + col_o[c]);
                if (n > 0) {
                    e = cudaMemcpyAsync(sb + col_o[c], src[c] + (g0 - hc.content_base), (size_t)n * 4, cudaMemcpyHostToDevice, q);
                    if (e != cudaSuccess) return e;
                }
            }
            if (ncol < 4) dc.mass = nullptr;
            return cudaSuccess;
        };
        HEPK_CUDA_TRY(stage_coll(d->jets, bd.jets, p.slot.joff, p.slot.jcol, 4));
        HEPK_CUDA_TRY(stage_coll(d->muons, bd.muons, p.slot.moff, p.slot.mcol, 3));
        if (has_el) HEPK_CUDA_TRY(stage_coll(d->electrons, bd.electrons, p.slot.eoff, p.slot.ecol, 3));
        if (d->weights) {
            for (int w = 0; w < W; ++w)
                HEPK_CUDA_TRY(cudaMemcpyAsync(sb + p.slot.weights + (size_t)w * nb * 4, d->weights + (size_t)w * w_stride + e0,
                                              (size_t)nb * 4, cudaMemcpyHostToDevice, q));
            bd.weights = (const float*)(sb + p.slot.weights);
        }
        if (d->evw_table) {
            HEPK_CUDA_TRY(cudaMemcpyAsync(sb + p.slot.evw_x, d->evw_x + e0, (size_t)nb * 4, cudaMemcpyHostToDevice, q));
            bd.evw_x = (const float*)(sb + p.slot.evw_x);
        }
        int** out_i_dev[2] = {&bd.out_njet, &bd.out_argmax};
        float** out_f_dev[5] = {&bd.out_ht, &bd.out_maxpt, &bd.out_minpt, &bd.out_mjj, &bd.out_subpt};
        for (int c = 0; c < 2; ++c) *out_i_dev[c] = out_i_host[c] ? (int*)(sb + p.slot.out_i[c]) : nullptr;
        for (int c = 0; c < 5; ++c) *out_f_dev[c] = out_f_host[c] ? (float*)(sb + p.slot.out_f[c]) : nullptr;
        bd.out_jet_mask = d->out_jet_mask ? (uint8_t*)(sb + p.slot.out_mask) : nullptr;
        bd.hist_sumw = p.n_sumw ? (float*)(sb + p.slot.hist_sumw) : nullptr;
        bd.hist_sumw2 = p.n_sumw2 ? (float*)(sb + p.slot.hist_sumw2) : nullptr;
        bd.hist_counts = p.n_cnt ? (int64_t*)(sb + p.slot.hist_counts) : nullptr;

        const int32_t rc = hepk_analysis_chain(&bd, sb + p.slot.chain_ws, p.chain_ws_bytes, q);
        if (rc != HEPK_OK) return rc;

        // per-event outputs: device [V][nb] -> host [V][N] at column e0, ONE strided copy per output and batch
        for (int c = 0; c < 2; ++c)
            if (out_i_host[c])
                HEPK_CUDA_TRY(cudaMemcpy2DAsync(out_i_host[c] + e0, (size_t)o_stride * 4, sb + p.slot.out_i[c], (size_t)nb * 4,
                                                (size_t)nb * 4, (size_t)V, cudaMemcpyDeviceToHost, q));
        for (int c = 0; c < 5; ++c)
            if (out_f_host[c])
                HEPK_CUDA_TRY(cudaMemcpy2DAsync(out_f_host[c] + e0, (size_t)o_stride * 4, sb + p.slot.out_f[c], (size_t)nb * 4,
                                                (size_t)nb * 4, (size_t)V, cudaMemcpyDeviceToHost, q));
        for (int v = 0; v < V; ++v) {
            if (d->out_jet_mask && bd.jets.n_objects > 0)
                HEPK_CUDA_TRY(cudaMemcpyAsync(d->out_jet_mask + (size_t)v * d->jets.n_objects + (bd.jets.content_base - d->jets.content_base),
                                              sb + p.slot.out_mask + (size_t)v * bd.jets.n_objects, (size_t)bd.jets.n_objects,
                                              cudaMemcpyDeviceToHost, q));
        }
    }
    // histograms: one copy back per buffer set, added on the host in float64
    const long long n_max = p.n_sumw > p.n_sumw2 ? p.n_sumw : p.n_sumw2;
    std::vector<float> hs((size_t)n_max);
    std::vector<long long> hc((size_t)p.n_cnt);
    std::vector<double> acc((size_t)p.n_sumw, 0.0), acc2((size_t)p.n_sumw2, 0.0);
    for (int s = 0; s < n_slots; ++s) {
        HEPK_CUDA_TRY(cudaStreamSynchronize(st[s]));
        if (p.n_sumw) {
            HEPK_CUDA_TRY(cudaMemcpy(hs.data(), slot_base[s] + p.slot.hist_sumw, (size_t)p.n_sumw * 4, cudaMemcpyDeviceToHost));
            for (long long i = 0; i < p.n_sumw; ++i) acc[i] += (double)hs[i];
        }
        if (p.n_sumw2) {
            HEPK_CUDA_TRY(cudaMemcpy(hs.data(), slot_base[s] + p.slot.hist_sumw2, (size_t)p.n_sumw2 * 4, cudaMemcpyDeviceToHost));
            for (long long i = 0; i < p.n_sumw2; ++i) acc2[i] += (double)hs[i];
        }
        if (p.n_cnt) {
            HEPK_CUDA_TRY(cudaMemcpy(hc.data(), slot_base[s] + p.slot.hist_counts, (size_t)p.n_cnt * 8, cudaMemcpyDeviceToHost));
            for (long long i = 0; i < p.n_cnt; ++i) d->hist_counts[i] += hc[i];
        }
    }
    for (long long i = 0; i < p.n_sumw; ++i) d->hist_sumw[i] = (float)((double)d->hist_sumw[i] + acc[i]);
    for (long long i = 0; i < p.n_sumw2; ++i) d->hist_sumw2[i] = (float)((double)d->hist_sumw2[i] + acc2[i]);
    drain.armed = false;
    return HEPK_OK;
}
