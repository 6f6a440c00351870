// C ABI, part 4: the whole path with host buffers in and out (the end-to-end call).
#include <string.h>

#include <algorithm>
#include <vector>

#include "cdc_internal.cuh"

namespace {

struct Scratch {                       // device buffers of one call, freed on every exit path
    float *zref = nullptr;
    double *ranges = nullptr, *chi2 = nullptr;
    int32_t *peak = nullptr, *labels = nullptr;
    uint64_t *key = nullptr;
    int64_t *seed = nullptr;
    uint32_t *nmatch = nullptr;
    cdc_events *ev = nullptr;
    cudaStream_t s = nullptr;
    template <typename T>
    cudaError_t get(T **p, size_t n) { return cudaMallocAsync((void **)p, sizeof(T) * n, s); }   // stream-ordered pool:
    ~Scratch()                                                                                  // no device sync
    {
        void *all[] = {zref, ranges, chi2, peak, labels, key, seed, nmatch};
        for (void *p : all)
            if (p) cudaFreeAsync(p, s);
        if (ev) cdc_events_destroy(ev);
    }
};

}  // namespace

extern "C" int32_t cdc_find_tracks_host(const cdc_geometry *g, int32_t n_events, const int32_t *h_hit_offsets,
                                        const int32_t *h_wire_id, const float *h_drift_mm, const cdc_grid_spec *h_grids,
                                        const cdc_scan_params *params, const cdc_hough_params *hp,
                                        const float *h_zref_mm, int32_t hough_sets_axes, int64_t *h_best_seed, uint32_t *h_best_n_match,
                                        double *h_best_chi2, uint64_t *h_best_key, int32_t *h_labels,
                                        double *h_ranges, void *stream)
{
    return cdc_guard("cdc_find_tracks_host", [&]() -> int32_t {
    if (!g || !h_hit_offsets || !h_grids || !params || !h_best_seed || !h_best_n_match || !h_best_chi2 || !h_best_key)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_find_tracks_host: null argument");
    if (hp && !h_zref_mm) CDC_FAIL(CDC_ERR_INVALID, "cdc_find_tracks_host: Hough ranges need h_zref_mm");
    cudaStream_t s = (cudaStream_t)stream;
    Scratch S;
    S.s = s;
    int32_t rc = cdc_event_upload(g, n_events, h_hit_offsets, h_wire_id, h_drift_mm, 0, stream, &S.ev);
    if (rc != CDC_OK) return rc;
    const size_t E = (size_t)n_events, H = std::max<size_t>((size_t)h_hit_offsets[n_events], 1);
    CDC_CUDA(S.get(&S.key, E));
    CDC_CUDA(S.get(&S.seed, E));
    CDC_CUDA(S.get(&S.nmatch, E));
    CDC_CUDA(S.get(&S.chi2, E));
    CDC_CUDA(S.get(&S.labels, H));
    std::vector<cdc_grid_spec> grids(h_grids, h_grids + n_events);
    if (hp) {
        CDC_CUDA(S.get(&S.zref, E));
        CDC_CUDA(S.get(&S.ranges, 6 * E));
        CDC_CUDA(S.get(&S.peak, 4 * E));
        CDC_CUDA(cudaMemcpyAsync(S.zref, h_zref_mm, sizeof(float) * E, cudaMemcpyHostToDevice, s));
        rc = cdc_hough_seed_ranges(g, S.ev, hp, params->charge, S.zref, S.ranges, S.peak, nullptr, stream);
        if (rc != CDC_OK) return rc;
        std::vector<double> rg(6 * E);
        CDC_CUDA(cudaMemcpyAsync(rg.data(), S.ranges, sizeof(double) * 6 * E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));
        const int axis_of[3] = {0, 2, 3};                 // Hough gives theta, px, py
        for (size_t e = 0; hough_sets_axes && e < E; ++e)
            for (int k = 0; k < 3; ++k) {
                const int a = axis_of[k];
                const double lo = rg[6 * e + 2 * k], hi = rg[6 * e + 2 * k + 1];
                grids[e].lo[a] = lo;
                grids[e].step[a] = grids[e].n[a] > 1 ? (hi - lo) / (double)(grids[e].n[a] - 1) : 0.0;
            }
        if (h_ranges) memcpy(h_ranges, rg.data(), sizeof(double) * 6 * E);
    }
    rc = cdc_seed_scan(g, S.ev, grids.data(), params, nullptr, nullptr, nullptr, S.key, stream);
    if (rc != CDC_OK) return rc;
    rc = cdc_best_track(g, S.ev, grids.data(), params, S.key, S.seed, S.nmatch, S.chi2, S.labels, stream);
    if (rc != CDC_OK) return rc;
    CDC_CUDA(cudaMemcpyAsync(h_best_key, S.key, sizeof(uint64_t) * E, cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaMemcpyAsync(h_best_seed, S.seed, sizeof(int64_t) * E, cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaMemcpyAsync(h_best_n_match, S.nmatch, sizeof(uint32_t) * E, cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaMemcpyAsync(h_best_chi2, S.chi2, sizeof(double) * E, cudaMemcpyDeviceToHost, s));
    if (h_labels && h_hit_offsets[n_events] > 0)
        CDC_CUDA(cudaMemcpyAsync(h_labels, S.labels, sizeof(int32_t) * (size_t)h_hit_offsets[n_events], cudaMemcpyDeviceToHost, s));
    cdc_scan_stats st;
    rc = cdc_scan_get_stats(S.ev, &st, stream);           // synchronises
    if (rc != CDC_OK) return rc;
    return CDC_OK;
    });
}
