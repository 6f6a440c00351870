// C ABI, part 5: cdc_refine_tracks -- the coarse-to-fine refinement loop around the seed scan (reading
// C17).  The host only builds the sub-grid descriptions of the next iteration from the selected lattice points (the
// cos / sin of the theta nodes come from the same libm as everywhere else, reading C11); scanning, exact re-scoring
// and selection run in kernels (scan.cu, refine.cu).
#include <math.h>
#include <string.h>

#include <algorithm>
#include <vector>

#include "refine.cuh"

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

}  // namespace

extern "C" int32_t cdc_refine_tracks(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                                     const cdc_scan_params *p, const cdc_refine_params *rp, double *h_best_seed,
                                     double *h_best_S, uint32_t *h_best_n_match, double *h_best_chi2, int64_t *h_best_q,
                                     int32_t *h_labels_or_null, double *h_trace_S_or_null, int64_t *h_trace_q_or_null,
                                     void *stream)
{
    return cdc_guard("cdc_refine_tracks", [&]() -> int32_t {
    if (!g || !ev || !h_grids || !p || !rp || !h_best_seed || !h_best_S || !h_best_n_match || !h_best_chi2 || !h_best_q)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_refine_tracks: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_refine_tracks: events belong to another geometry");
    const int K = rp->n_parents, T = rp->n_iterations, E = ev->n_events;
    if (K < 1 || K > 8 || T < 0 || T > 20) CDC_FAIL(CDC_ERR_INVALID, "cdc_refine_tracks: need 1 <= n_parents <= 8, 0 <= n_iterations <= 20");
    for (int e = 0; e < ev->n_events; ++e)
        for (int a = 0; a < 5; ++a)
            if (h_grids[e].first[a] != 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_refine_tracks: grid node offsets (first) must be 0");
    cudaStream_t s = (cudaStream_t)stream;
    Dev D(s);
    int64_t total = 0;
    for (int e = 0; e < E; ++e) {
        int64_t prod = 1;
        for (int a = 0; a < 5; ++a) prod *= std::max(h_grids[e].n[a], 1);
        total += prod;
    }
    if (total > (1LL << 30)) CDC_FAIL(CDC_ERR_RANGE, "cdc_refine_tracks: more than 2^30 seeds in the initial grids");
    // ---- iteration 0: fp32 scan of the initial grids, scores materialised
    uint32_t *d_nm = nullptr; float *d_c2 = nullptr; uint64_t *d_key = nullptr;
    CDC_CUDA(D.get(&d_nm, (size_t)total)); CDC_CUDA(D.get(&d_c2, (size_t)total)); CDC_CUDA(D.get(&d_key, (size_t)E));
    int32_t rc = cdc_seed_scan(g, ev, h_grids, p, d_nm, d_c2, nullptr, d_key, stream);
    if (rc != CDC_OK) return rc;

    RefineLaunch L;
    L.g = g->g64; L.n_events = E; L.K = K; L.cap = std::max(2048, K * 243);
    L.d_grids0 = ev->d_grids; L.d_n_match = d_nm; L.d_chi2 = d_c2;
    L.max_seeds_per_event = 0;
    for (const GridDev &G : ev->h_grids) L.max_seeds_per_event = std::max<int64_t>(L.max_seeds_per_event, G.n_seeds);
    L.margin = (float)(p->rescore_margin > 0.0 ? p->rescore_margin : 0.05);
    L.d_drift_tab = ev->d_drift_tab; L.d_bits = ev->d_bits; L.d_offsets = ev->d_offsets; L.d_wire_id = ev->d_wire_id;
    L.W = ev->W; L.n_bit_words = ev->n_bit_words; L.max_hits_per_event = ev->max_hits_per_event;
    L.h = p->h_mm; L.window = p->window_mm; L.eloss = p->eloss_MeV_per_mm; L.max_steps = p->max_steps; L.charge = p->charge;
    L.lookup_every64 = cdc_lookup_every64(g, p->h_mm, p->window_mm);
    L.d_wire_label = ev->d_wire_label; L.d_wire_best = ev->d_wire_best;
    CDC_CUDA(D.get(&L.d_cand_idx, (size_t)E * L.cap)); CDC_CUDA(D.get(&L.d_count, (size_t)E));
    CDC_CUDA(D.get(&L.d_S64, (size_t)E * L.cap)); CDC_CUDA(D.get(&L.d_chi2_64, (size_t)E * L.cap));
    CDC_CUDA(D.get(&L.d_nm64, (size_t)E * L.cap));
    unsigned long long *d_prev = nullptr, *d_cur = nullptr;
    CDC_CUDA(D.get(&d_prev, (size_t)E)); CDC_CUDA(D.get(&d_cur, (size_t)E));
    RefineParent *d_par[2] = {nullptr, nullptr};
    CDC_CUDA(D.get(&d_par[0], (size_t)E * K)); CDC_CUDA(D.get(&d_par[1], (size_t)E * K));
    int32_t *d_npar = nullptr, *d_labels = nullptr;
    CDC_CUDA(D.get(&d_npar, (size_t)E)); CDC_CUDA(D.get(&d_labels, (size_t)std::max(ev->total_hits, 1)));
    GridDev *d_sub = nullptr; double *d_sub_axes = nullptr;
    CDC_CUDA(D.get(&d_sub, (size_t)E * K)); CDC_CUDA(D.get(&d_sub_axes, (size_t)E * K * 6 * 3));

    // K-th largest fp32 key per event: K passes of "largest key below the previous one"
    CDC_CUDA(cudaMemsetAsync(d_prev, 0xFF, sizeof(unsigned long long) * (size_t)E, s));
    for (int k = 0; k < K; ++k) {
        CDC_CUDA(refine_kth_pass(L, d_prev, d_cur, s));
        std::swap(d_prev, d_cur);
    }
    CDC_CUDA(refine_candidates(L, d_prev, s));
    const long long two_T = 1LL << T;
    CDC_CUDA(refine_eval_select(L, 0, two_T, ev->d_grids, ev->axes.d, ev->axes.stride, nullptr, d_par[0], d_npar, s));
    std::vector<int32_t> h_count(E), h_npar(E);
    CDC_CUDA(cudaMemcpyAsync(h_count.data(), L.d_count, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
    std::vector<RefineParent> par((size_t)E * K), par_prev;
    CDC_CUDA(cudaMemcpyAsync(par.data(), d_par[0], sizeof(RefineParent) * par.size(), cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaMemcpyAsync(h_npar.data(), d_npar, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaStreamSynchronize(s));
    for (int e = 0; e < E; ++e)
        if (h_count[e] > L.cap) CDC_FAIL(CDC_ERR_RANGE, "cdc_refine_tracks: too many seeds tie with the K-th best of the initial grid");
    auto trace = [&](int t) {
        for (int e = 0; e < E; ++e)
            for (int k = 0; k < K; ++k) {
                const bool ok = k < h_npar[e];
                if (h_trace_S_or_null) h_trace_S_or_null[((size_t)e * (T + 1) + t) * K + k] = ok ? par[(size_t)e * K + k].S : -1.0;
                if (h_trace_q_or_null)
                    for (int a = 0; a < 5; ++a)
                        h_trace_q_or_null[(((size_t)e * (T + 1) + t) * K + k) * 5 + a] = ok ? par[(size_t)e * K + k].q[a] : 0;
            }
    };
    trace(0);

    // ---- iterations 1..T: 3^5 nodes around every parent at half the previous pitch, all in fp64
    std::vector<GridDev> sub((size_t)E * K);
    std::vector<double> axes((size_t)E * K * 6 * 3, 0.0);
    std::vector<double> sub_lo((size_t)E * K * 5), sub_step((size_t)E * K * 5);
    int cur = 0;
    for (int t = 1; t <= T; ++t) {
        const long long d = 1LL << (T - t);
        for (int e = 0; e < E; ++e) {
            const cdc_grid_spec &G0 = h_grids[e];
            for (int k = 0; k < K; ++k) {
                const size_t gi = (size_t)e * K + k;
                GridDev &S = sub[gi];
                for (int a = 0; a < 5; ++a) S.n[a] = 3;
                S.n_seeds = 243; S.out_offset = 0;
                if (k >= h_npar[e]) continue;
                double *tab = axes.data() + gi * 18;
                for (int a = 0; a < 5; ++a) {
                    const double s_fine = G0.step[a] / (double)two_T;
                    const double lo = G0.lo[a] + (double)(par[gi].q[a] - d) * s_fine;   // reading C17
                    const double step = (double)d * s_fine;
                    sub_lo[gi * 5 + a] = lo; sub_step[gi * 5 + a] = step;
                    for (int i = 0; i < 3; ++i) {
                        const double v = lo + (double)i * step;
                        if (a == 0) { tab[i] = g->R0 * cos(v); tab[3 + i] = g->R0 * sin(v); }     // reading C4
                        else tab[(size_t)(a + 1) * 3 + i] = v;
                    }
                }
            }
        }
        CDC_CUDA(cudaMemcpyAsync(d_sub, sub.data(), sizeof(GridDev) * sub.size(), cudaMemcpyHostToDevice, s));
        CDC_CUDA(cudaMemcpyAsync(d_sub_axes, axes.data(), sizeof(double) * axes.size(), cudaMemcpyHostToDevice, s));
        CDC_CUDA(cudaMemcpyAsync(L.d_count, h_npar.data(), sizeof(int32_t) * (size_t)E, cudaMemcpyHostToDevice, s));
        CDC_CUDA(refine_eval_select(L, 1, d, d_sub, d_sub_axes, 3, d_par[cur], d_par[cur ^ 1], d_npar, s));
        cur ^= 1;
        par_prev = par;
        CDC_CUDA(cudaMemcpyAsync(par.data(), d_par[cur], sizeof(RefineParent) * par.size(), cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaMemcpyAsync(h_npar.data(), d_npar, sizeof(int32_t) * (size_t)E, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));            // also makes the pageable staging vectors reusable
        trace(t);
    }

    // ---- result: first parent of the last iteration; its value is the node its sub-grid handed to the scan
    for (int e = 0; e < E; ++e) {
        if (h_npar[e] < 1) CDC_FAIL(CDC_ERR_NOT_READY, "cdc_refine_tracks: an event has no seed at all");
        const RefineParent &B = par[(size_t)e * K];
        h_best_S[e] = B.S; h_best_n_match[e] = (uint32_t)B.n_match; h_best_chi2[e] = B.chi2;
        int t = B.idx;
        int off[5];
        for (int a = 4; a >= 0; --a) {
            const int na = T == 0 ? h_grids[e].n[a] : 3;
            off[a] = t % na; t /= na;
        }
        for (int a = 0; a < 5; ++a) {
            h_best_q[(size_t)e * 5 + a] = B.q[a];
            if (T == 0) h_best_seed[(size_t)e * 5 + a] = h_grids[e].lo[a] + (double)off[a] * h_grids[e].step[a];
            else {
                const size_t gi = (size_t)e * K + B.rank;
                h_best_seed[(size_t)e * 5 + a] = sub_lo[gi * 5 + a] + (double)off[a] * sub_step[gi * 5 + a];
            }
        }
    }
    if (h_labels_or_null && ev->total_hits > 0) {
        if (T == 0) CDC_CUDA(refine_labels(L, 0, ev->d_grids, ev->axes.d, ev->axes.stride, d_par[cur], d_labels, s));
        else CDC_CUDA(refine_labels(L, 1, d_sub, d_sub_axes, 3, d_par[cur], d_labels, s));
        CDC_CUDA(cudaMemcpyAsync(h_labels_or_null, d_labels, sizeof(int32_t) * (size_t)ev->total_hits, cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));
    }
    return CDC_OK;
    });
}
