// C ABI, part 2: A1 event upload / binning and the events handle.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <new>

#include "cdc_internal.cuh"

namespace {

void free_events(cdc_events *ev)
{
    if (!ev) return;
    // stream-ordered: the memory returns to the pool after the work already queued on the upload stream
    // work queued on another stream (scan / best track are asynchronous on a caller-chosen stream) must have finished
    // before the memory goes back to the pool
    if (ev->last_stream && ev->last_stream != ev->alloc_stream) cudaStreamSynchronize(ev->last_stream);
    if (ev->slab) cudaFreeAsync(ev->slab, ev->alloc_stream);
    if (ev->big_slab) cudaFreeAsync(ev->big_slab, ev->alloc_stream);
    if (ev->axes.d) cudaFreeAsync(ev->axes.d, ev->alloc_stream);
    if (ev->ev_k0) cudaEventDestroy(ev->ev_k0);
    if (ev->ev_k1) cudaEventDestroy(ev->ev_k1);
    delete ev;
}

struct Carver {                 // pass 1 (base == nullptr) sizes the slab, pass 2 hands out the pieces
    char *base = nullptr;
    size_t off = 0;
    template <typename T>
    void take(T *&p, size_t n)
    {
        const size_t bytes = (std::max<size_t>(n, 1) * sizeof(T) + 255) & ~(size_t)255;
        if (base) p = reinterpret_cast<T *>(base + off);
        off += bytes;
    }
};

void carve(cdc_events *ev, Carver &c)
{
    const size_t E = (size_t)ev->n_events, W = (size_t)ev->W, H = (size_t)ev->total_hits, P = ev->pool_cap;
    c.take(ev->d_offsets, E + 1); c.take(ev->d_wire_id, H); c.take(ev->d_drift, H);
    c.take(ev->d_drift_tab, E * W); c.take(ev->d_bits, E * ev->n_bit_words); c.take(ev->d_err, 1);
    c.take(ev->d_counters, CNT_N); c.take(ev->d_ev_maxS, E); c.take(ev->d_ev_best, E); c.take(ev->d_peak_key, E);
    c.take(ev->d_wire_label, E * W); c.take(ev->d_wire_best, E * W); c.take(ev->d_grids, E);
    c.take(ev->d_pool, P); c.take(ev->d_pool_S64, P); c.take(ev->d_pool_chi2, P); c.take(ev->d_pool_nmatch, P);
    c.take(ev->d_pool_slot, P); c.take(ev->d_rec, (size_t)kRecSlots * kRecCap); c.take(ev->d_rec_count, kRecSlots);
    c.take(ev->d_slot_counter, 1); c.take(ev->d_ev_slot, E);
}

}  // namespace

#define EV_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { free_events(ev); \
    cdc_set_error(std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    return e_ == cudaErrorMemoryAllocation ? CDC_ERR_NOMEM : CDC_ERR_CUDA; } } while (0)

extern "C" int32_t cdc_event_upload(const cdc_geometry *g, int32_t n_events, const int32_t *h_hit_offsets,
                                    const int32_t *wire_id, const float *drift_mm, int32_t hits_on_device,
                                    void *stream, cdc_events **out)
{
    return cdc_guard("cdc_event_upload", [&]() -> int32_t {
    if (!g || !h_hit_offsets || !out) CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: null argument");
    *out = nullptr;
    if (n_events < 1 || n_events > 65535) CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: n_events must be in [1, 65535]");
    if (h_hit_offsets[0] != 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: hit_offsets[0] must be 0");
    int32_t max_hits = 0;
    for (int e = 0; e < n_events; ++e) {
        const int32_t c = h_hit_offsets[e + 1] - h_hit_offsets[e];
        if (c < 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: hit_offsets must be non-decreasing");
        max_hits = std::max(max_hits, c);
    }
    const int32_t total = h_hit_offsets[n_events];
    if (total > 0 && (!wire_id || !drift_mm)) CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: null hit arrays");
    cudaStream_t s = (cudaStream_t)stream;
    cdc_events *ev = new (std::nothrow) cdc_events;
    if (!ev) CDC_FAIL(CDC_ERR_NOMEM, "cdc_event_upload: host allocation failed");
    ev->geom = g; ev->n_events = n_events; ev->total_hits = total; ev->W = g->W; ev->n_bit_words = (g->W + 31) / 32;
    ev->max_hits_per_event = max_hits;
    ev->offsets.assign(h_hit_offsets, h_hit_offsets + n_events + 1);
    ev->pool_cap = std::max<uint32_t>(1u << 16, 64u * (uint32_t)n_events);
    ev->alloc_stream = s;
    Carver sizing;
    carve(ev, sizing);
    EV_CUDA(cudaMallocAsync(&ev->slab, sizing.off, s));
    Carver placing;
    placing.base = static_cast<char *>(ev->slab);
    carve(ev, placing);
    EV_CUDA(cudaMemsetAsync(ev->d_counters, 0, sizeof(unsigned long long) * CNT_N, s));
    EV_CUDA(cudaMemcpyAsync(ev->d_offsets, h_hit_offsets, sizeof(int32_t) * (size_t)(n_events + 1), cudaMemcpyHostToDevice, s));
    if (total > 0) {
        const cudaMemcpyKind k = hits_on_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice;
        EV_CUDA(cudaMemcpyAsync(ev->d_wire_id, wire_id, sizeof(int32_t) * (size_t)total, k, s));
        EV_CUDA(cudaMemcpyAsync(ev->d_drift, drift_mm, sizeof(float) * (size_t)total, k, s));
    }
    EV_CUDA(launch_bin_events(n_events, g->W, ev->n_bit_words, max_hits, ev->d_offsets, ev->d_wire_id, ev->d_drift,
                              ev->d_drift_tab, ev->d_bits, ev->d_err, s));
    int32_t err = 0;
    EV_CUDA(cudaMemcpyAsync(&err, ev->d_err, sizeof(int32_t), cudaMemcpyDeviceToHost, s));
    EV_CUDA(cudaStreamSynchronize(s));
    if (err & 1) { free_events(ev); CDC_FAIL(CDC_ERR_RANGE, "cdc_event_upload: wire id out of range"); }
    if (err & 2) { free_events(ev); CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: drift distance outside [0, 8] mm or non-finite"); }
    if (err & 4) { free_events(ev); CDC_FAIL(CDC_ERR_INVALID, "cdc_event_upload: duplicate wire id within an event"); }
    *out = ev;
    return CDC_OK;
    });
}

extern "C" int32_t cdc_events_destroy(cdc_events *ev)
{
    return cdc_guard("cdc_events_destroy", [&]() -> int32_t {
    free_events(ev);
    return CDC_OK;
    });
}

extern "C" int32_t cdc_events_tables(const cdc_events *ev, float *h_drift_of_wire, uint32_t *h_hit_bits)
{
    return cdc_guard("cdc_events_tables", [&]() -> int32_t {
    if (!ev) CDC_FAIL(CDC_ERR_INVALID, "cdc_events_tables: null events");
    if (h_drift_of_wire)
        CDC_CUDA(cudaMemcpy(h_drift_of_wire, ev->d_drift_tab, sizeof(float) * (size_t)ev->n_events * ev->W, cudaMemcpyDeviceToHost));
    if (h_hit_bits)
        CDC_CUDA(cudaMemcpy(h_hit_bits, ev->d_bits, sizeof(uint32_t) * (size_t)ev->n_events * ev->n_bit_words, cudaMemcpyDeviceToHost));
    return CDC_OK;
    });
}
