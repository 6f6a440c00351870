// C ABI, part 3: A2 Hough ranges, A3-A7 seed scan, A8-A9 best track.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <mutex>

#include "cdc_internal.cuh"

namespace {

constexpr double kDefaultMargin = 0.05;

// One pinned host buffer per process for the small per-scan tables (axis nodes, grid records).  acquire() waits
// for the previous copy out of it (an event), so consecutive scans on any stream never overwrite live data.
struct Staging {
    std::mutex mu;
    char *p = nullptr;
    size_t cap = 0;
    cudaEvent_t done = nullptr;
    int32_t acquire(size_t bytes, char **out)
    {
        mu.lock();
        if (!done) { cudaError_t e = cudaEventCreateWithFlags(&done, cudaEventDisableTiming); if (e != cudaSuccess) { mu.unlock(); CDC_FAIL(CDC_ERR_CUDA, "staging event"); } }
        else cudaEventSynchronize(done);
        if (cap < bytes) {
            if (p) cudaFreeHost(p);
            p = nullptr; cap = 0;
            const size_t want = std::max<size_t>(bytes, 1 << 16);
            if (cudaMallocHost((void **)&p, want) != cudaSuccess) { mu.unlock(); CDC_FAIL(CDC_ERR_NOMEM, "pinned staging allocation failed"); }
            cap = want;
        }
        *out = p;
        return CDC_OK;       // still locked: release() unlocks
    }
    cudaError_t release(cudaStream_t s)
    {
        cudaError_t e = cudaEventRecord(done, s);
        mu.unlock();
        return e;
    }
} g_staging;

int32_t check_params(const cdc_scan_params *p, const char *who)
{
    if (!p) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": null params");
    if (!(p->h_mm > 0.0) || !(p->h_mm <= 4.0)) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": need 0 < h <= 4 mm");
    if (p->max_steps < 1) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": max_steps < 1");
    if (!(p->window_mm > 0.0)) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": window <= 0");
    if (!(p->eloss_MeV_per_mm >= 0.0)) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": negative energy loss");
    if (p->charge != 1 && p->charge != -1) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": charge must be +-1");
    if (p->kernel_variant < 0 || p->kernel_variant > 3) CDC_FAIL(CDC_ERR_INVALID, std::string(who) + ": kernel_variant must be 0, 1, 2 or 3");
    return CDC_OK;
}

// A3 host part: validate the grids, build the fp64 axis tables and the per-event grid records
int32_t prepare_grids(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *grids, cudaStream_t s)
{
    const int E = ev->n_events;
    int32_t stride = 1;
    ev->h_grids.resize(E);
    int64_t off = 0;
    for (int e = 0; e < E; ++e) {
        int64_t prod = 1;
        for (int a = 0; a < 5; ++a) {
            const int32_t n = grids[e].n[a];
            if (n < 1 || n > CDC_MAX_AXIS) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: grid n must be in [1, 4096]");
            if (!isfinite(grids[e].lo[a]) || !isfinite(grids[e].step[a]))
                CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: non-finite grid lo / step");
            if (grids[e].first[a] < 0) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: negative grid node offset (first)");
            prod *= n;
            if (prod > 2147483647LL) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: more than 2^31 - 1 seeds in a grid");
            stride = std::max(stride, n);
            ev->h_grids[e].n[a] = n;
        }
        ev->h_grids[e].n_seeds = (int32_t)prod;
        ev->h_grids[e].out_offset = off;
        off += prod;
    }
    if (ev->axes.stride < stride) {
        if (ev->axes.d) CDC_CUDA(cudaFreeAsync(ev->axes.d, s));
        ev->axes.d = nullptr; ev->axes.stride = 0;
        CDC_CUDA(cudaMallocAsync((void **)&ev->axes.d, sizeof(double) * (size_t)E * 6 * stride, s));
        ev->axes.stride = stride;
    }
    stride = ev->axes.stride;
    const size_t n_tab = (size_t)E * 6 * stride;
    // process-wide pinned staging: the copies are truly asynchronous; wait only if the previous user's copy
    // out of the staging buffer has not finished yet
    const size_t grid_off = (sizeof(double) * n_tab + 255) & ~(size_t)255;
    char *stage = nullptr;
    {
        const int32_t rc = g_staging.acquire(grid_off + sizeof(GridDev) * (size_t)E, &stage);
        if (rc != CDC_OK) return rc;
    }
    double *tab = reinterpret_cast<double *>(stage);
    GridDev *h_grids_pinned = reinterpret_cast<GridDev *>(stage + grid_off);
    for (int e = 0; e < E; ++e) {
        double *t = tab + (size_t)e * 6 * stride;
        const cdc_grid_spec &G = grids[e];
        for (int i = 0; i < G.n[0]; ++i) {            // reading C4: r0 = (R0 cos(theta), R0 sin(theta), z)
            const double th = G.lo[0] + (double)(G.first[0] + i) * G.step[0];
            t[i] = g->R0 * cos(th);
            t[stride + i] = g->R0 * sin(th);
        }
        for (int a = 1; a < 5; ++a)
            for (int i = 0; i < G.n[a]; ++i) t[(size_t)(a + 1) * stride + i] = G.lo[a] + (double)(G.first[a] + i) * G.step[a];
        h_grids_pinned[e] = ev->h_grids[e];
    }
    const cudaError_t c1 = cudaMemcpyAsync(ev->axes.d, tab, sizeof(double) * n_tab, cudaMemcpyHostToDevice, s);
    const cudaError_t c2 = cudaMemcpyAsync(ev->d_grids, h_grids_pinned, sizeof(GridDev) * (size_t)E, cudaMemcpyHostToDevice, s);
    const cudaError_t c3 = g_staging.release(s);          // always unlocks
    CDC_CUDA(c1); CDC_CUDA(c2); CDC_CUDA(c3);
    return CDC_OK;
}

// everything of a scan launch that follows from the geometry, the scanned grids and the parameters (the per-call
// output pointers are set by the caller)
int32_t fill_scan_launch(const cdc_geometry *g, const cdc_events *ev, const cdc_scan_params *p, ScanLaunch &L)
{
    L.gd = g->gd; L.fd = g->fd; L.n_events = ev->n_events; L.d_grids = ev->d_grids; L.d_axes = ev->axes.d;
    L.axis_stride = ev->axes.stride; L.d_drift_tab = ev->d_drift_tab; L.d_bits = ev->d_bits;
    L.h = (float)p->h_mm; L.h64 = p->h_mm; L.lambda = (float)(p->window_mm * p->window_mm);
    L.eloss_h = (float)(p->eloss_MeV_per_mm * p->h_mm);
    L.max_steps = p->max_steps; L.charge = p->charge;
    L.margin = (float)(p->rescore_margin > 0.0 ? p->rescore_margin : kDefaultMargin);
    L.d_n_match = nullptr; L.d_chi2 = nullptr; L.d_debug = nullptr; L.d_best_key = nullptr;
    L.d_pool = ev->d_pool; L.pool_cap = ev->pool_cap; L.d_counters = ev->d_counters;
    // lookup cadence K: the 2 x 2 candidate set is taken around c = r_n + (K h / 2) T_n, the middle of the next K steps.
    // A wire that can own a match in interval n + i lies within `reach` of vertex n + i, which lies within K h / 2 (+ the
    // sagitta of that arc) of c; every wire outside the set is at least `excl` away from c (reading C8).
    {
        const double dmax = 8.0 + p->window_mm + 0.05;           // largest matching D: drift <= 8 mm (upload check)
        const double reach = sqrt(dmax * dmax + p->h_mm * p->h_mm) + 0.1;
        if (reach > g->excl) CDC_FAIL(CDC_ERR_RANGE, "cdc_seed_scan: window + step too large for the 2 x 2 wire lookup");
        const double sag = 0.15;                                 // (K h / 2)^2 / (2 R) for R >= 150 mm, K h / 2 <= 6.7 mm
        int K = (int)floor(2.0 * (g->excl - reach - sag) / p->h_mm);
        K = std::max(1, std::min(K, 16));
        double ahead = 0.5 * K * p->h_mm;
        if (ahead + reach + sag > g->excl) { K = 1; ahead = 0.0; }
        L.lookup_every = K; L.lookahead = (float)ahead;
        // the straight-line prediction of the centre needs a track radius well above K h (the kernel checks
        // |a| B_max < 1 / 20 mm per seed); tighter curls look up around r_n itself, every K0 steps
        const int K0 = std::max(1, std::min(1 + (int)floor((g->excl - reach) / p->h_mm), 16));
        L.lookup_every_tight = K0;
        // vertex n + i lies i h along the arc: (i h - ahead) along the tangent from c and at most kappa (i h)^2 / 2 off
        // it, so it stays within ahead + sag of c for every i <= K iff kappa <= 2 sqrt(sag^2 + 2 sag ahead) / (K h)^2
        // (kappa = |a| B_max, the track's curvature bound); never above the old fixed 1 / 20 mm
        {
            const double Kh = K * p->h_mm;
            L.tight_curv = (float)(ahead > 0.0 ? std::min(0.05, 0.98 * 2.0 * sqrt(sag * sag + 2.0 * sag * ahead) / (Kh * Kh)) : 0.05);
        }
        // the two-seed kernel looks wires up around the midpoint of its two seeds, at most sep_cap (as a wire sees it)
        // from either seed's own centre: every bound that speaks of "the lookup centre" is widened by it
        const bool pair = p->kernel_variant == 1 && !(g->field.kind != 0 && p->eloss_MeV_per_mm > 0.0);
        const double sep_cap = pair ? 1.5 : 0.0;
        L.sep_cap = (float)sep_cap;
        L.k_margin = (float)(0.9999 * (g->excl - reach - sag) - 0.01);
        L.k_margin0 = (float)(0.9999 * (g->excl - reach) - 0.01);
        {
            double se = 0.0;
            for (int j = 0; j < g->n_layers; ++j) se = std::max(se, fabs(sin(g->stereo[j])));
            L.sin_eps = (float)(1.0001 * se);
        }
        const double grow = reach + 0.2 + sep_cap + std::max(ahead + sag, (K0 - 1) * p->h_mm);
        const double ulo = std::max(g->r[0] - grow, 0.0), uhi = g->r[g->n_layers - 1] + grow;
        L.u2_lo = (float)(ulo * ulo); L.u2_hi = (float)(uhi * uhi);
        L.back = (float)(std::max(ahead + 0.2, (K0 - 1) * p->h_mm) + sep_cap);
        L.uz = g->uz; L.inv_uz = (float)(1.0 / (double)g->uz);
        // a held wire lies within the 2 x 2 set of the last lookup vertex (two layer pitches x two cells) and
        // the track has moved at most K h since: |delta| <= diag + K h; it stays held while the track crosses
        // that neighbourhood, at most ~(diag + K h) / min|T_perp| of path -- bounded here by 4 diag
        const double diag = hypot(2.0 * g->pitch, 2.0 * g->cell_max);
        // the kernel's curvature bounds allow |a| = kappa / p to grow by 5 % between two lookups; p > 1 MeV/c on a live
        // track, so the momentum lost over one lookup period must stay below 0.04 MeV/c
        if (p->eloss_MeV_per_mm * (std::max(K, K0) * p->h_mm + 1.0) > 0.04)
            CDC_FAIL(CDC_ERR_RANGE, "cdc_seed_scan: energy loss too large for the lookup cadence (eloss * K h must stay below 0.04 MeV/c)");
        L.delta_max = (float)(diag + std::max(K, K0) * p->h_mm + 1.0 + sep_cap);
        L.b_max = (float)(1.001 * g->b_max);
        L.hold_path = (float)(4.0 * diag + 2.0 * std::max(K, K0) * p->h_mm + 2.0 * sep_cap);
    }
    L.max_seeds_per_event = 0;
    L.max_pairs_per_event = 0;
    for (const GridDev &G : ev->h_grids) {
        L.max_seeds_per_event = std::max<int64_t>(L.max_seeds_per_event, G.n_seeds);
        L.max_pairs_per_event = std::max<int64_t>(L.max_pairs_per_event, ((int64_t)G.n_seeds / G.n[1]) * ((G.n[1] + 1) / 2));
    }
    L.variant = p->kernel_variant;
    return CDC_OK;
}

}  // namespace

int32_t cdc_lookup_every64(const cdc_geometry *g, double h_mm, double window_mm)
{
    const double dmax = 8.0 + window_mm + 0.05;
    const double reach = sqrt(dmax * dmax + h_mm * h_mm) + 0.1;
    const double excl3 = 1.5 * (g->excl + 0.2) - 0.3;           // 1.5 layer pitches / 1.5 cells (g->excl is one of them)
    if (reach > excl3) return 1;
    return std::max(1, std::min(1 + (int)floor((excl3 - reach) / h_mm), 16));
}

// ------------------------------------------------------------------------------------------------ A2
extern "C" int32_t cdc_hough_dims(const cdc_hough_params *hp, int32_t *dims3)
{
    return cdc_guard("cdc_hough_dims", [&]() -> int32_t {
    if (!hp || !dims3) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_dims: null argument");
    if (!(hp->bin_xy_mm > 0) || !(hp->bin_R_mm > 0) || !(hp->R_hi_mm > hp->R_lo_mm) || !(hp->half_xy_mm > 0) || !(hp->tol_mm > 0))
        CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_dims: bad Hough parameters");
    dims3[0] = (int32_t)floor((hp->R_hi_mm - hp->R_lo_mm) / hp->bin_R_mm + 0.5);
    dims3[1] = (int32_t)floor(2.0 * hp->half_xy_mm / hp->bin_xy_mm + 0.5);
    dims3[2] = dims3[1];
    if (dims3[0] < 1 || dims3[1] < 1 || (int64_t)dims3[0] * dims3[1] * dims3[2] > 0x7FFFFFFFLL || dims3[0] > 256)
        CDC_FAIL(CDC_ERR_RANGE, "cdc_hough_dims: accumulator too large (nR <= 256, bins < 2^31)");
    return CDC_OK;
    });
}

extern "C" int32_t cdc_hough_seed_ranges(const cdc_geometry *g, const cdc_events *ev, const cdc_hough_params *hp,
                                         int32_t charge, const float *d_zref_mm, double *d_ranges, int32_t *d_peak,
                                         uint32_t *d_accum_or_null, void *stream)
{
    return cdc_guard("cdc_hough_seed_ranges", [&]() -> int32_t {
    if (!g || !ev || !hp || !d_zref_mm || !d_ranges || !d_peak) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges: events belong to another geometry");
    if (charge != 1 && charge != -1) CDC_FAIL(CDC_ERR_INVALID, "cdc_hough_seed_ranges: charge must be +-1");
    int32_t dims[3];
    const int32_t rc = cdc_hough_dims(hp, dims);
    if (rc != CDC_OK) return rc;
    HoughLaunch L;
    L.n_events = ev->n_events; L.nR = dims[0]; L.ncy = dims[1]; L.ncx = dims[2];
    L.bin_xy = (float)hp->bin_xy_mm; L.bin_R = (float)hp->bin_R_mm; L.tol = (float)hp->tol_mm; L.R_lo = (float)hp->R_lo_mm;
    L.half_xy = (float)hp->half_xy_mm; L.origin = (float)hp->origin_mm;
    L.bin_xy64 = hp->bin_xy_mm; L.bin_R64 = hp->bin_R_mm; L.R_lo64 = hp->R_lo_mm; L.half_xy64 = hp->half_xy_mm;
    L.R0 = g->R0; L.half_theta = hp->half_theta_rad; L.half_pt = hp->half_pt_MeV; L.bz = g->field.bz_T; L.charge = charge;
    L.d_wire5 = g->d_wire5; L.d_offsets = ev->d_offsets; L.d_wire_id = ev->d_wire_id; L.d_zref = d_zref_mm;
    L.d_ranges = d_ranges; L.d_peak = d_peak; L.d_accum = d_accum_or_null; L.d_peak_key = ev->d_peak_key;
    CDC_CUDA(launch_hough(L, (cudaStream_t)stream));
    return CDC_OK;
    });
}

// ------------------------------------------------------------------------------------------------ A3-A7
extern "C" int32_t cdc_seed_scan(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                                 const cdc_scan_params *p, uint32_t *d_n_match, float *d_chi2,
                                 cdc_seed_debug *d_debug, uint64_t *d_best_key, void *stream)
{
    return cdc_guard("cdc_seed_scan", [&]() -> int32_t {
    if (!g || !ev || !h_grids || !d_best_key) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan: events belong to another geometry");
    int32_t rc = check_params(p, "cdc_seed_scan");
    if (rc != CDC_OK) return rc;
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = prepare_grids(g, ev, h_grids, s)) != CDC_OK) return rc;
    CDC_CUDA(cudaMemsetAsync(d_best_key, 0, sizeof(uint64_t) * (size_t)ev->n_events, s));
    CDC_CUDA(cudaMemsetAsync(ev->d_counters, 0, sizeof(unsigned long long) * CNT_N, s));
    ScanLaunch L;
    if ((rc = fill_scan_launch(g, ev, p, L)) != CDC_OK) return rc;
    L.d_n_match = d_n_match; L.d_chi2 = d_chi2; L.d_debug = d_debug; L.d_best_key = d_best_key;
    if (!ev->ev_k0) { CDC_CUDA(cudaEventCreate(&ev->ev_k0)); CDC_CUDA(cudaEventCreate(&ev->ev_k1)); }
    CDC_CUDA(launch_seed_scan(L, s, ev->ev_k0, ev->ev_k1));
    ev->scanned = true; ev->adaptive_scanned = false;
    ev->last_stream = s;
    return CDC_OK;
    });
}

// ------------------------------------------------------------------------------------------------ SURVEY 8(f) #4
extern "C" int32_t cdc_seed_scan_adaptive(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                                          const cdc_scan_params *p, double tol_mm, double h_max_mm, uint32_t *d_n_match,
                                          float *d_chi2, cdc_seed_debug *d_debug, int32_t *d_levels, uint64_t *d_best_key,
                                          void *stream)
{
    return cdc_guard("cdc_seed_scan_adaptive", [&]() -> int32_t {
    if (!g || !ev || !h_grids || !d_best_key) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_adaptive: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_adaptive: events belong to another geometry");
    int32_t rc = check_params(p, "cdc_seed_scan_adaptive");
    if (rc != CDC_OK) return rc;
    if (!(tol_mm > 0.0) || !isfinite(tol_mm) || !(h_max_mm >= p->h_mm) || !isfinite(h_max_mm))
        CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_adaptive: need tol > 0 and h_max >= h");
    int J = 0;
    while (J < 6 && p->h_mm * (double)(2 << J) <= h_max_mm) ++J;            // levels 0 .. J, h 2^J <= h_max
    const double H = p->h_mm * (double)(1 << J);
    // the 2 x 2 set around a step's START vertex must hold every wire that can own a match in that step
    const double dmax = 8.0 + p->window_mm + 0.05;
    const double reach = sqrt(dmax * dmax + H * H) + 0.1;
    if (reach > g->excl) CDC_FAIL(CDC_ERR_RANGE, "cdc_seed_scan_adaptive: window + longest step too large for the 2 x 2 wire lookup (h_max <= ~12 mm)");
    cudaStream_t s = (cudaStream_t)stream;
    if ((rc = prepare_grids(g, ev, h_grids, s)) != CDC_OK) return rc;
    CDC_CUDA(cudaMemsetAsync(d_best_key, 0, sizeof(uint64_t) * (size_t)ev->n_events, s));
    CDC_CUDA(cudaMemsetAsync(ev->d_counters, 0, sizeof(unsigned long long) * CNT_N, s));
    ScanLaunch L;
    if ((rc = fill_scan_launch(g, ev, p, L)) != CDC_OK) return rc;
    L.d_n_match = d_n_match; L.d_chi2 = d_chi2; L.d_debug = d_debug; L.d_best_key = d_best_key;
    const double grow = reach + 0.2;
    const double ulo = std::max(g->r[0] - grow, 0.0), uhi = g->r[g->n_layers - 1] + grow;
    L.u2_lo = (float)(ulo * ulo); L.u2_hi = (float)(uhi * uhi);
    if (!ev->ev_k0) { CDC_CUDA(cudaEventCreate(&ev->ev_k0)); CDC_CUDA(cudaEventCreate(&ev->ev_k1)); }
    CDC_CUDA(launch_seed_scan_adaptive(L, tol_mm, J, d_levels, s, ev->ev_k0, ev->ev_k1));
    ev->scanned = false;                       // no candidate pool was filled: cdc_best_track does not apply to this variant
    ev->adaptive_scanned = true;
    ev->last_stream = s;
    return CDC_OK;
    });
}

extern "C" int32_t cdc_scan_get_stats(const cdc_events *ev, cdc_scan_stats *out, void *stream)
{
    return cdc_guard("cdc_scan_get_stats", [&]() -> int32_t {
    if (!ev || !out) CDC_FAIL(CDC_ERR_INVALID, "cdc_scan_get_stats: null argument");
    if (!ev->scanned && !ev->adaptive_scanned) CDC_FAIL(CDC_ERR_NOT_READY, "cdc_scan_get_stats: no scan has run on these events");
    unsigned long long c[CNT_N];
    CDC_CUDA(cudaMemcpyAsync(c, ev->d_counters, sizeof(c), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
    CDC_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
    out->n_seeds = 0;
    for (const GridDev &G : ev->h_grids) out->n_seeds += (uint64_t)G.n_seeds;
    out->n_steps = c[CNT_STEPS]; out->n_gas_steps = c[CNT_GAS]; out->n_approach_tests = c[CNT_TESTS];
    out->n_pool = c[CNT_POOL]; out->pool_cap = ev->pool_cap;
    out->n_lookups = c[CNT_LOOKUP]; out->n_g1 = c[CNT_G1]; out->n_approaches = c[CNT_APPROACH];
    float ms = 0.f;
    CDC_CUDA(cudaEventSynchronize(ev->ev_k1));
    CDC_CUDA(cudaEventElapsedTime(&ms, ev->ev_k0, ev->ev_k1));
    out->kernel_ms = (double)ms;
    return CDC_OK;
    });
}

// ------------------------------------------------------------------------------------------------ A8-A9
extern "C" int32_t cdc_best_track(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                                  const cdc_scan_params *p, const uint64_t *d_best_key, int64_t *d_best_seed,
                                  uint32_t *d_best_n_match, double *d_best_chi2, int32_t *d_labels, void *stream)
{
    return cdc_guard("cdc_best_track", [&]() -> int32_t {
    if (!g || !ev || !h_grids || !d_best_key || !d_best_seed || !d_best_n_match || !d_best_chi2)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_best_track: null argument");
    if (ev->geom != g) CDC_FAIL(CDC_ERR_INVALID, "cdc_best_track: events belong to another geometry");
    if (!ev->scanned) CDC_FAIL(CDC_ERR_NOT_READY, "cdc_best_track: call cdc_seed_scan first");
    int32_t rc = check_params(p, "cdc_best_track");
    if (rc != CDC_OK) return rc;
    for (int e = 0; e < ev->n_events; ++e)
        for (int a = 0; a < 5; ++a)
            if (h_grids[e].n[a] != ev->h_grids[e].n[a]) CDC_FAIL(CDC_ERR_INVALID, "cdc_best_track: grids differ from the scanned ones");
    cudaStream_t s = (cudaStream_t)stream;
    ev->last_stream = s;
    // how many candidates did the scan append?  (one 8-byte read-back; the launches below are sized by it)
    unsigned long long n_pool = 0;
    CDC_CUDA(cudaMemcpyAsync(&n_pool, ev->d_counters + CNT_POOL, sizeof(n_pool), cudaMemcpyDeviceToHost, s));
    CDC_CUDA(cudaStreamSynchronize(s));
    PoolEntry *pool = ev->d_pool;
    double *pS64 = ev->d_pool_S64, *pchi2 = ev->d_pool_chi2;
    int32_t *pnm = ev->d_pool_nmatch, *pslot = ev->d_pool_slot;
    uint32_t cap = ev->pool_cap;
    if (n_pool > (unsigned long long)ev->pool_cap) {
        // Overflow: the pool was filled against the RUNNING maximum, in launch order, so what it holds is arbitrary.
        // Collect again against the FINAL maximum: the scan is repeated with best_key left as it is (every seed now sees
        // the final maximum as the running one) and a pool as large as the first pass's count, an upper bound of what
        // the second can append (the final threshold is the highest).  Bounded by the true number of near-ties.
        if (n_pool > (1ull << 26))
            CDC_FAIL(CDC_ERR_RANGE, "cdc_best_track: more than 2^26 seeds within the re-score margin of the running maximum");
        if ((unsigned long long)ev->big_cap < n_pool) {
            if (ev->big_slab) CDC_CUDA(cudaFreeAsync(ev->big_slab, s));
            ev->big_slab = nullptr; ev->big_cap = 0;
            const size_t n = (size_t)n_pool, a = 256;
            const size_t o1 = (n * sizeof(PoolEntry) + a - 1) / a * a, o2 = o1 + (n * 8 + a - 1) / a * a, o3 = o2 + (n * 8 + a - 1) / a * a,
                         o4 = o3 + (n * 4 + a - 1) / a * a, o5 = o4 + (n * 4 + a - 1) / a * a;
            CDC_CUDA(cudaMallocAsync(&ev->big_slab, o5, s));
            char *b = static_cast<char *>(ev->big_slab);
            ev->d_bpool = reinterpret_cast<PoolEntry *>(b); ev->d_bS64 = reinterpret_cast<double *>(b + o1);
            ev->d_bchi2 = reinterpret_cast<double *>(b + o2); ev->d_bnmatch = reinterpret_cast<int32_t *>(b + o3);
            ev->d_bslot = reinterpret_cast<int32_t *>(b + o4);
            ev->big_cap = (uint32_t)n_pool;
        }
        unsigned long long saved[CNT_N];
        CDC_CUDA(cudaMemcpyAsync(saved, ev->d_counters, sizeof(saved), cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));
        CDC_CUDA(cudaMemsetAsync(ev->d_counters + CNT_POOL, 0, sizeof(unsigned long long), s));
        ScanLaunch SL;
        if ((rc = fill_scan_launch(g, ev, p, SL)) != CDC_OK) return rc;
        SL.d_best_key = const_cast<uint64_t *>(d_best_key);          // atomicMax with values that cannot exceed it: unchanged
        SL.d_pool = ev->d_bpool; SL.pool_cap = ev->big_cap;
        CDC_CUDA(launch_seed_scan(SL, s, nullptr, nullptr));
        CDC_CUDA(cudaMemcpyAsync(&n_pool, ev->d_counters + CNT_POOL, sizeof(n_pool), cudaMemcpyDeviceToHost, s));
        CDC_CUDA(cudaStreamSynchronize(s));
        saved[CNT_POOL] = n_pool;                                     // the scan's work counters stay those of the first pass
        CDC_CUDA(cudaMemcpyAsync(ev->d_counters, saved, sizeof(saved), cudaMemcpyHostToDevice, s));
        CDC_CUDA(cudaStreamSynchronize(s));
        if (n_pool > (unsigned long long)ev->big_cap) CDC_FAIL(CDC_ERR_RANGE, "cdc_best_track: candidate pool overflow in the second pass");
        pool = ev->d_bpool; pS64 = ev->d_bS64; pchi2 = ev->d_bchi2; pnm = ev->d_bnmatch; pslot = ev->d_bslot; cap = ev->big_cap;
    }
    ev->last_pool_count = n_pool;
    BestLaunch L;
    L.g = g->g64; L.n_events = ev->n_events; L.d_grids = ev->d_grids; L.d_axes = ev->axes.d; L.axis_stride = ev->axes.stride;
    L.d_offsets = ev->d_offsets; L.d_wire_id = ev->d_wire_id; L.d_drift = ev->d_drift; L.d_drift_tab = ev->d_drift_tab;
    L.d_bits = ev->d_bits; L.W = ev->W; L.n_bit_words = ev->n_bit_words; L.max_hits_per_event = ev->max_hits_per_event;
    L.h = p->h_mm; L.window = p->window_mm; L.eloss = p->eloss_MeV_per_mm; L.max_steps = p->max_steps; L.charge = p->charge;
    L.lookup_every64 = cdc_lookup_every64(g, p->h_mm, p->window_mm);
    L.margin = (float)(p->rescore_margin > 0.0 ? p->rescore_margin : kDefaultMargin);
    L.d_best_key = d_best_key; L.d_pool = pool; L.pool_cap = cap; L.n_entries = (uint32_t)n_pool; L.d_counters = ev->d_counters;
    L.d_pool_S64 = pS64; L.d_pool_chi2 = pchi2; L.d_pool_nmatch = pnm;
    L.d_ev_maxS = ev->d_ev_maxS; L.d_ev_best = ev->d_ev_best; L.d_wire_label = ev->d_wire_label; L.d_wire_best = ev->d_wire_best;
    L.d_rec = ev->d_rec; L.d_rec_count = ev->d_rec_count; L.d_pool_slot = pslot; L.d_slot_counter = ev->d_slot_counter;
    L.d_ev_slot = ev->d_ev_slot;
    L.d_best_seed = d_best_seed; L.d_best_n_match = d_best_n_match; L.d_best_chi2 = d_best_chi2; L.d_labels = d_labels;
    CDC_CUDA(launch_best_track(L, (cudaStream_t)stream));
    return CDC_OK;
    });
}

extern "C" int32_t cdc_fp32_peak_probe(int32_t iters, double *h_flops_per_s, double *h_ms, void *stream)
{
    return cdc_guard("cdc_fp32_peak_probe", [&]() -> int32_t {
    if (iters < 1) CDC_FAIL(CDC_ERR_INVALID, "cdc_fp32_peak_probe: iters < 1");
    CDC_CUDA(run_fp32_peak_probe(iters, h_flops_per_s, h_ms, (cudaStream_t)stream));
    return CDC_OK;
    });
}

extern "C" int32_t cdc_fp32_issue_probe(int32_t mode, int32_t iters, double *h_ms, double *h_warp_instructions, double *h_flops,
                                        void *stream)
{
    return cdc_guard("cdc_fp32_issue_probe", [&]() -> int32_t {
    if (iters < 1 || mode < 0 || mode > 7) CDC_FAIL(CDC_ERR_INVALID, "cdc_fp32_issue_probe: need iters >= 1, 0 <= mode <= 7");
    CDC_CUDA(run_fp32_issue_probe(mode, iters, h_ms, h_warp_instructions, h_flops, (cudaStream_t)stream));
    return CDC_OK;
    });
}
