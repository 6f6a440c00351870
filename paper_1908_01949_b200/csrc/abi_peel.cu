// C ABI, part 7: cdc_peel_turns -- the event reconstruction loop of PAPER.md:83 without the fit (reading C18).
// Scanning, re-scoring, labelling, hit removal and the extrapolation to the next entrance run in kernels (scan.cu,
// best.cu, peel.cu); once per partition the host reads a few numbers per event back, applies the stop rules and
// turns the extrapolated state into the next grid (atan2 from the host libm, as the cos / sin of the theta nodes:
// reading C11).
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "peel.cuh"

namespace {

struct Dev {                          // device scratch of one call, freed on every exit path
    std::vector<void *> p;
    cudaStream_t s;
    explicit Dev(cudaStream_t st) : s(st) {}
    template <typename T>
    cudaError_t get(T **out, size_t n)
    {
        void *q = nullptr;
        cudaError_t e = cudaMallocAsync(&q, std::max<size_t>(n, 1) * sizeof(T), s);
        if (e == cudaSuccess) p.push_back(q);
        *out = static_cast<T *>(q);
        return e;
    }
    ~Dev() { for (void *q : p) cudaFreeAsync(q, s); }
};

struct RestoreBits {                  // the events' fired-wire bitmap is put back on every exit path
    uint32_t *dst = nullptr;
    const uint32_t *saved = nullptr;
    size_t bytes = 0;
    cudaStream_t s = nullptr;
    ~RestoreBits()
    {
        if (dst && saved) { cudaMemcpyAsync(dst, saved, bytes, cudaMemcpyDeviceToDevice, s); cudaStreamSynchronize(s); }
    }
};

}  // namespace

extern "C" int32_t cdc_peel_turns(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids0,
                                  const cdc_scan_params *p, const cdc_peel_params *pp, int32_t *h_n_partitions,
                                  int32_t *h_status, double *h_seeds, uint32_t *h_n_match, double *h_chi2,
                                  double *h_centres_or_null, int32_t *d_partition, void *stream)
{
    return cdc_guard("cdc_peel_turns", [&]() -> int32_t {
    if (!g || !ev || !h_grids0 || !p || !pp || !h_n_partitions || !h_status || !h_seeds || !h_n_match || !h_chi2)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: events belong to another geometry");
    const int P = pp->max_partitions, E = ev->n_events;
    if (P < 1 || P > 8) CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: need 1 <= max_partitions <= 8");
    for (int e = 0; e < ev->n_events; ++e)
        for (int a = 0; a < 5; ++a)
            if (h_grids0[e].first[a] != 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: grid node offsets (first) must be 0");
    if (pp->min_hits < 0 || pp->min_classified < 0 || pp->extrap_max_steps < 1)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: need min_hits >= 0, min_classified >= 0, extrap_max_steps >= 1");
    for (int a = 0; a < 5; ++a) {
        if (pp->n[a] < 1 || pp->n[a] > CDC_MAX_AXIS) CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: n must be in [1, 4096]");
        if (!(pp->half_width[a] >= 0.0) || !isfinite(pp->half_width[a]))
            CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: half_width must be finite and >= 0");
    }
    if (!(pp->extrap_tol_mm >= 0.0) || !isfinite(pp->extrap_tol_mm))
        CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: extrap_tol_mm must be finite and >= 0");
    if (pp->extrap_tol_mm > 0.0 && (!(pp->extrap_h_max_mm >= p->h_mm) || !isfinite(pp->extrap_h_max_mm)))
        CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: adaptive extrapolation needs h <= extrap_h_max_mm < inf");
    if (ev->total_hits > 0 && !d_partition) CDC_FAIL(CDC_ERR_INVALID, "cdc_peel_turns: null d_partition");
    cudaStream_t s = (cudaStream_t)stream;
    Dev D(s);
    uint64_t *d_key = nullptr; int64_t *d_best = nullptr; uint32_t *d_nm = nullptr; double *d_c2 = nullptr;
    int32_t *d_labels = nullptr, *d_active = nullptr, *d_counts = nullptr, *d_ok = nullptr; double *d_next = nullptr;
    uint32_t *d_saved = nullptr;
    const size_t n_bits = (size_t)E * ev->n_bit_words;
    CDC_CUDA(D.get(&d_key, (size_t)E)); CDC_CUDA(D.get(&d_best, (size_t)E)); CDC_CUDA(D.get(&d_nm, (size_t)E));
    CDC_CUDA(D.get(&d_c2, (size_t)E)); CDC_CUDA(D.get(&d_labels, (size_t)ev->total_hits));
    CDC_CUDA(D.get(&d_active, (size_t)E)); CDC_CUDA(D.get(&d_counts, 2 * (size_t)E)); CDC_CUDA(D.get(&d_ok, (size_t)E));
    CDC_CUDA(D.get(&d_next, 6 * (size_t)E)); CDC_CUDA(D.get(&d_saved, n_bits));
    CDC_CUDA(cudaMemcpyAsync(d_saved, ev->d_bits, sizeof(uint32_t) * n_bits, cudaMemcpyDeviceToDevice, s));
    RestoreBits restore;
    restore.dst = ev->d_bits; restore.saved = d_saved; restore.bytes = sizeof(uint32_t) * n_bits; restore.s = s;
    if (ev->total_hits > 0) CDC_CUDA(cudaMemsetAsync(d_partition, 0xFF, sizeof(int32_t) * (size_t)ev->total_hits, s));

    std::vector<cdc_grid_spec> grids(h_grids0, h_grids0 + E);
    std::vector<int32_t> active(E), counts(2 * (size_t)E), ok(E);
    std::vector<int64_t> best(E);
    std::vector<uint32_t> nm(E);
    std::vector<double> c2(E), next(6 * (size_t)E);
    memset(h_seeds, 0, sizeof(double) * (size_t)E * P * 5);
    memset(h_n_match, 0, sizeof(uint32_t) * (size_t)E * P);
    memset(h_chi2, 0, sizeof(double) * (size_t)E * P);
    if (h_centres_or_null) memset(h_centres_or_null, 0, sizeof(double) * (size_t)E * P * 5);
    int n_active = 0;
    for (int e = 0; e < E; ++e) {
        h_n_partitions[e] = 0;
        const int hits = ev->offsets[e + 1] - ev->offsets[e];
        active[e] = hits >= pp->min_hits ? 1 : 0;                         // stop rule 1 before the first scan
        h_status[e] = active[e] ? 3 : 1;
        n_active += active[e];
    }

    PeelLaunch L;
    L.g = g->g64; L.n_events = E; L.W = ev->W; L.n_bit_words = ev->n_bit_words; L.max_hits_per_event = ev->max_hits_per_event;
    L.d_offsets = ev->d_offsets; L.d_wire_id = ev->d_wire_id; L.d_bits = ev->d_bits;
    L.h = p->h_mm; L.eloss = p->eloss_MeV_per_mm; L.kq = CDC_KAPPA * (double)p->charge; L.extrap_max_steps = pp->extrap_max_steps;
    L.extrap_tol = pp->extrap_tol_mm; L.extrap_h_max = pp->extrap_h_max_mm;
    L.d_labels = d_labels; L.d_best_seed = d_best; L.d_active = d_active; L.d_partition = d_partition;
    L.d_counts = d_counts; L.d_next = d_next; L.d_next_ok = d_ok;

    for (int k = 0; k < P && n_active > 0; ++k) {
        for (int e = 0; e < E; ++e)
            if (!active[e])                                               // a finished event: one seed, result ignored
                for (int a = 0; a < 5; ++a) { grids[e].n[a] = 1; grids[e].step[a] = 0.0; }
        int32_t rc = cdc_seed_scan(g, ev, grids.data(), p, nullptr, nullptr, nullptr, d_key, stream);
        if (rc != CDC_OK) return rc;
        rc = cdc_best_track(g, ev, grids.data(), p, d_key, d_best, d_nm, d_c2, d_labels, stream);
        if (rc != CDC_OK) return rc;
        CDC_CUDA(cudaMemcpyAsync(d_active, active.data(), sizeof(int32_t) * (size_t)E, cudaMemcpyHostToDevice, s));
        L.d_grids = ev->d_grids; L.d_axes = ev->axes.d; L.axis_stride = ev->axes.stride;
        CDC_CUDA(peel_partition(L, k, pp->min_classified, s));
        CDC_CUDA(cudaMemcpyAsync(best.data(), d_best, sizeof(int64_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(nm.data(), d_nm, sizeof(uint32_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(c2.data(), d_c2, sizeof(double) * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(counts.data(), d_counts, sizeof(int32_t) * 2 * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(next.data(), d_next, sizeof(double) * 6 * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(ok.data(), d_ok, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));
        for (int e = 0; e < E; ++e) {
            if (!active[e]) continue;
            if (best[e] < 0) CDC_FAIL(CDC_ERR_RANGE, "cdc_peel_turns: the candidate pool of a scan overflowed");
            auto stop = [&](int why) { h_status[e] = why; active[e] = 0; n_active -= 1; };
            if (counts[2 * (size_t)e] < pp->min_classified) { stop(2); continue; }
            int64_t t = best[e];
            const size_t row = (size_t)e * P + k;
            for (int a = 4; a >= 0; --a) {                               // seed values: node i of axis a, pz fastest
                const int64_t i = t % grids[e].n[a];
                t /= grids[e].n[a];
                h_seeds[row * 5 + a] = grids[e].lo[a] + (double)i * grids[e].step[a];
            }
            h_n_match[row] = nm[e]; h_chi2[row] = c2[e];
            h_n_partitions[e] = k + 1;
            if (counts[2 * (size_t)e + 1] - counts[2 * (size_t)e] < pp->min_hits) { stop(1); continue; }
            if (k + 1 == P) { stop(3); continue; }
            if (!ok[e]) { stop(4); continue; }
            const double *nx = next.data() + 6 * (size_t)e;
            const double c[5] = {atan2(nx[1], nx[0]), nx[2], nx[3], nx[4], nx[5]};
            for (int a = 0; a < 5; ++a) {                                // reading C18, step 7
                grids[e].n[a] = pp->n[a];
                if (pp->n[a] > 1) {
                    grids[e].lo[a] = c[a] - pp->half_width[a];
                    grids[e].step[a] = 2.0 * pp->half_width[a] / (double)(pp->n[a] - 1);
                } else { grids[e].lo[a] = c[a]; grids[e].step[a] = 0.0; }
                if (h_centres_or_null) h_centres_or_null[((size_t)e * P + k + 1) * 5 + a] = c[a];
            }
        }
    }
    return CDC_OK;
    });
}
