// Internal declarations shared by the translation units of libcdc_seedscan.so.
// Nothing here is visible through the C ABI (include/cdc_seedscan.h).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include <new>
#include <stdexcept>
#include <string>
#include <vector>

#include "../../include/cdc_seedscan.h"

#define CDC_MAX_LAYERS 32
#define CDC_KAPPA 0.299792458   // curvature [1/mm] = kappa q B[T] / p[MeV/c]  (reading C1)
#define CDC_MAX_AXIS 4096

// ---- device-side tables (A0) -------------------------------------------------------------------
struct LayerDev {            // 32 B, one per sense layer, read through shared memory in the scan
    float r;                 // waist radius
    float shift_k;           // sigma_j tan|eps| / r_j : azimuth shift of the wire at height z is atan(z * shift_k)
    float phi0;
    float kscale;            // n_j / 2 pi
    float uz;                // cos(eps) as stored in the canonical wire table
    float inv_uz;
    int32_t n;
    int32_t offset;
};

struct FieldDev {
    int32_t kind;
    float bz;                // uniform field
    int32_t nr, nz;
    float r0, z0, inv_dr, inv_dz;
    float cr, cz;            // -r0 / dr - 1/2, -z0 / dz - 1/2: fma(rho, inv_dr, cr) = cell coordinate - 1/2
    int32_t n_cells;         // (nr - 1) (nz - 1)
    float grad_max;          // bound of |dB/dx| over the table (T/mm; +inf if B_r != 0 on the axis): see scan.cu, field reuse
    const float2 *tab;       // [nz][nr] (B_r, B_z) nodes (fp64 path)
    const float4 *cells;     // [nr-1][nz-1][2] (z fastest): bilinear coefficients about the cell centre (c0, c_z, c_r, c_rz) of B_r, then of B_z
};

struct GeomDev {
    int32_t n_layers, n_wires_total, n_bit_words;
    float r_first, inv_pitch, tan_abs;       // layer lookup: j = (u - r_first) * inv_pitch, u^2 = rho^2 - (z tan)^2
    float u2_lo, u2_hi;                      // lookup is skipped outside this band of u^2
    float R0sq, z_half, r_out_sq;
    const float4 *wire4;                     // (w0x, w0y, ux, uy)
    const LayerDev *layers;                  // device copy
};

// fp64 view for the exact re-score (A8/A9)
struct Geom64 {
    int32_t n_layers, n_wires_total;
    double R0, z_half, r_out;
    const float *wire5;                      // canonical [W][5]
    const LayerDev *layers;
    float r_first, inv_pitch, tan_abs;
    int32_t field_kind;
    double bz;
    int32_t nr, nz;
    double r0, z0, dr, dz;
    const float *tab;                        // [nz][nr][2]
};

struct cdc_geometry {
    int32_t n_layers = 0, W = 0;
    std::vector<double> r, phi0, stereo;
    std::vector<int32_t> n_wires, offset;
    std::vector<float> wire5;
    double z_half = 0, R0 = 0, r_out = 0;
    double b_max = 0;                        // largest |B| of the field description
    double grad_max = 0;                     // bound of the gradient of B over the table (T/mm), 0 for the uniform field
    double cell_max = 0;                     // largest cell width (arc at the end plate)
    double pitch = 0, excl = 0;              // layer pitch; distance below which a wire is surely in the 2 x 2 set
    float uz = 1.f;
    cdc_field_desc field{};                  // h_br_bz replaced by field_tab.data()
    std::vector<float> field_tab;
    // device
    float4 *d_wire4 = nullptr;
    float *d_wire5 = nullptr;
    float2 *d_field = nullptr;
    float4 *d_cells = nullptr;
    LayerDev *d_layers = nullptr;
    GeomDev gd{};
    FieldDev fd{};
    Geom64 g64{};
};

struct PoolEntry {           // one rescoring candidate (reading C11)
    uint32_t event;
    uint32_t index;          // linear seed index within the event's grid
    float S32;
    uint32_t pad;
};

struct ApproachRec {         // one matched approach of a re-scored seed (reading C12)
    int32_t wire, turn;
    double absd;
};
constexpr int kRecSlots = 256;
constexpr int kRecCap = 2048;

struct AxisTables {          // per event, device: seed-axis node values in fp64 (A3)
    // layout [n_events][6][stride]: R0 cos(theta), R0 sin(theta), z, px, py, pz
    double *d = nullptr;
    int32_t stride = 0;
};

struct GridDev {             // per event, passed in a device array
    int32_t n[5];
    int32_t n_seeds;
    int64_t out_offset;      // offset of this event's seeds in the concatenated per-seed outputs
};

struct cdc_events {
    const cdc_geometry *geom = nullptr;
    int32_t n_events = 0, total_hits = 0, W = 0, n_bit_words = 0;
    std::vector<int32_t> offsets;
    int32_t *d_offsets = nullptr, *d_wire_id = nullptr;
    float *d_drift = nullptr;
    float *d_drift_tab = nullptr;            // [n_events][W]
    uint32_t *d_bits = nullptr;              // [n_events][n_bit_words]
    int32_t *d_err = nullptr;                // validation flags
    // scan scratch
    AxisTables axes;
    GridDev *d_grids = nullptr;
    std::vector<GridDev> h_grids;
    PoolEntry *d_pool = nullptr;
    uint32_t pool_cap = 0;
    unsigned long long *d_counters = nullptr;   // [8]: steps, gas steps, approach tests, pool count, ...
    bool scanned = false;
    bool adaptive_scanned = false;           // the last scan was cdc_seed_scan_adaptive (counters: steps, path units)
    cudaEvent_t ev_k0 = nullptr, ev_k1 = nullptr;   // bracket of the scan kernel
    // best-track scratch
    double *d_pool_S64 = nullptr, *d_pool_chi2 = nullptr;
    int32_t *d_pool_nmatch = nullptr;
    unsigned long long *d_ev_maxS = nullptr;    // per event: bits of the fp64 maximum
    unsigned long long *d_ev_best = nullptr;    // per event: lowest index attaining it
    int32_t *d_wire_label = nullptr;            // [n_events][W] turn label per wire (labels)
    double *d_wire_best = nullptr;              // [n_events][W] smallest |resid| so far
    unsigned long long *d_peak_key = nullptr;   // Hough scratch [n_events]
    int32_t max_hits_per_event = 0;
    // matched-approach records of the re-scored candidates (A9 replays the best seed's list)
    ApproachRec *d_rec = nullptr;               // [kRecSlots][kRecCap]
    int32_t *d_rec_count = nullptr;             // [kRecSlots]
    int32_t *d_pool_slot = nullptr;             // [pool_cap] record slot of a pool entry, -1 = none
    int32_t *d_slot_counter = nullptr;
    int32_t *d_ev_slot = nullptr;               // per event: record slot of the best seed, -1 = re-propagate
    // overflow pool (cdc_best_track): when the scan appended more candidates than pool_cap, the near-ties of the FINAL
    // maximum are collected again into a pool sized for them
    void *big_slab = nullptr;
    uint32_t big_cap = 0;
    PoolEntry *d_bpool = nullptr;
    double *d_bS64 = nullptr, *d_bchi2 = nullptr;
    int32_t *d_bnmatch = nullptr, *d_bslot = nullptr;
    unsigned long long last_pool_count = 0;     // entries the last cdc_best_track re-scored from (after any second pass)
    cudaStream_t last_stream = nullptr;         // stream of the last asynchronous call on this batch
    // one stream-ordered allocation holds every device buffer above
    void *slab = nullptr;
    cudaStream_t alloc_stream = nullptr;
};

enum { CNT_STEPS = 0, CNT_GAS = 1, CNT_TESTS = 2, CNT_POOL = 3, CNT_LOOKUP = 4, CNT_G1 = 5, CNT_APPROACH = 6, CNT_N = 8 };

void cdc_count_launch(int n = 1);

// ---- error plumbing ------------------------------------------------------------------------------
void cdc_set_error(const std::string &msg);
#define CDC_FAIL(code, msg) do { cdc_set_error(msg); return (code); } while (0)
#define CDC_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { \
    cdc_set_error(std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    return (e_ == cudaErrorMemoryAllocation) ? CDC_ERR_NOMEM : CDC_ERR_CUDA; } } while (0)

// ---- no exception crosses the C boundary (include/cdc_seedscan.h): every int32_t entry point runs inside this
template <typename F>
inline int32_t cdc_guard(const char *who, F &&body) noexcept
{
    try {
        return body();
    } catch (const std::bad_alloc &) {
        try { cdc_set_error(std::string(who) + ": out of host memory"); } catch (...) {}
        return CDC_ERR_NOMEM;
    } catch (const std::exception &e) {
        try { cdc_set_error(std::string(who) + ": " + e.what()); } catch (...) {}
        return CDC_ERR_INVALID;
    } catch (...) {
        return CDC_ERR_INVALID;
    }
}

// ---- launchers implemented in the kernel translation units ---------------------------------------
struct ScanLaunch {
    GeomDev gd;
    FieldDev fd;
    int32_t n_events;
    const GridDev *d_grids;
    const double *d_axes;
    int32_t axis_stride;
    const float *d_drift_tab;
    const uint32_t *d_bits;
    float h, lambda, eloss_h;        // eloss_h = eloss per step (MeV)
    double h64;
    int32_t max_steps, charge;
    float margin;
    uint32_t *d_n_match;
    float *d_chi2;
    cdc_seed_debug *d_debug;
    uint64_t *d_best_key;
    PoolEntry *d_pool;
    uint32_t pool_cap;
    unsigned long long *d_counters;
    int64_t max_seeds_per_event;
    int64_t max_pairs_per_event;     // two-seeds-per-thread kernel: ceil(n_z / 2) * n_theta * n_px * n_py * n_pz
    int32_t variant;                 // 0: one seed per thread (scan.cu); 1: two seeds per thread (scan_pair.cu)
    float u2_lo, u2_hi, uz, inv_uz;  // lookup band (widened for the lookup cadence), cos(eps)
    int32_t lookup_every;            // K: steps per layer/cell lookup
    float lookahead;                 // the lookup is centred on r_n + lookahead * T_n (the middle of the next K steps)
    int32_t lookup_every_tight;      // K for tightly curling seeds: lookup centred on r_n itself
    float back;                      // how far inside the band's lower edge a held wire can still be scored from
    float tight_curv;                // |a| B_max at and above which a seed counts as tightly curling (host: sagitta margin)
    float delta_max, b_max, hold_path;   // largest |delta| of a held wire, largest |B|, longest path a wire stays held
    float k_margin, k_margin0, sin_eps, sep_cap;  // two-seed kernel: excl - reach - sag, excl - reach (rounded down), sin|stereo|,
                                         // largest half-separation (as a wire sees it) served by one shared lookup
};
cudaError_t launch_seed_scan(const ScanLaunch &L, cudaStream_t s, cudaEvent_t k0, cudaEvent_t k1);
cudaError_t launch_seed_scan_adaptive(const ScanLaunch &L, double tol, int J, int32_t *d_levels, cudaStream_t s, cudaEvent_t k0,
                                      cudaEvent_t k1);

cudaError_t launch_bin_events(int32_t n_events, int32_t W, int32_t n_bit_words, int32_t max_hits_per_event,
                              const int32_t *d_offsets, const int32_t *d_wire_id, const float *d_drift,
                              float *d_drift_tab, uint32_t *d_bits, int32_t *d_err, cudaStream_t s);

struct HoughLaunch {
    int32_t n_events, nR, ncy, ncx;
    float bin_xy, bin_R, tol, R_lo, half_xy, origin;
    double bin_xy64, bin_R64, R_lo64, half_xy64, R0, half_theta, half_pt, bz;
    int32_t charge;
    const float *d_wire5;
    const int32_t *d_offsets, *d_wire_id;
    const float *d_zref;
    double *d_ranges;
    int32_t *d_peak;
    uint32_t *d_accum;
    unsigned long long *d_peak_key;     // scratch [n_events]
};
cudaError_t launch_hough(const HoughLaunch &L, cudaStream_t s);

struct BestLaunch {
    Geom64 g;
    int32_t n_events;
    const GridDev *d_grids;
    const double *d_axes;
    int32_t axis_stride;
    const int32_t *d_offsets, *d_wire_id;
    const float *d_drift, *d_drift_tab;
    const uint32_t *d_bits;
    int32_t W, n_bit_words, max_hits_per_event;
    double h, window, eloss;
    int32_t max_steps, charge, lookup_every64;
    float margin;
    const uint64_t *d_best_key;
    const PoolEntry *d_pool;
    uint32_t pool_cap;
    uint32_t n_entries;                      // pool entries to re-score (host copy of the counter, <= pool_cap)
    const unsigned long long *d_counters;
    double *d_pool_S64, *d_pool_chi2;
    int32_t *d_pool_nmatch;
    unsigned long long *d_ev_maxS, *d_ev_best;
    int32_t *d_wire_label;
    double *d_wire_best;
    ApproachRec *d_rec;
    int32_t *d_rec_count, *d_pool_slot, *d_slot_counter, *d_ev_slot;
    int64_t *d_best_seed;
    uint32_t *d_best_n_match;
    double *d_best_chi2;
    int32_t *d_labels;
};
cudaError_t launch_best_track(const BestLaunch &L, cudaStream_t s);

// K64: how many intervals the 3 x 3 candidate set of the fp64 evaluation stays a superset (reading C8)
int32_t cdc_lookup_every64(const cdc_geometry *g, double h_mm, double window_mm);

cudaError_t run_fp32_peak_probe(int32_t iters, double *flops_per_s, double *ms, cudaStream_t s);
cudaError_t run_fp32_issue_probe(int32_t mode, int32_t iters, double *ms_out, double *warp_inst, double *flops, cudaStream_t s);
