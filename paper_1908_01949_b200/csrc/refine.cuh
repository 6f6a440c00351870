// Declarations shared by refine.cu (kernels, -fmad=false) and abi_refine.cu (host driver of cdc_refine_tracks).
#pragma once
#include "cdc_internal.cuh"

struct RefineParent {        // one selected seed of an iteration
    long long q[5];          // lattice point on the finest pitch
    double S, chi2;
    int32_t n_match, rank, idx, pad;   // sub-grid it was scanned in (0 in iteration 0) and linear index there
};

struct RefineLaunch {
    Geom64 g;
    int32_t n_events, K, cap;
    const GridDev *d_grids0;         // initial grids (device records of the events handle)
    const uint32_t *d_n_match;       // per-seed fp32 scan outputs of the initial grids
    const float *d_chi2;
    int64_t max_seeds_per_event;
    float margin;
    const float *d_drift_tab;
    const uint32_t *d_bits;
    const int32_t *d_offsets, *d_wire_id;
    int32_t W, n_bit_words, max_hits_per_event;
    double h, window, eloss;
    int32_t max_steps, charge, lookup_every64;
    uint32_t *d_cand_idx;            // [E][cap]
    int32_t *d_count;                // [E]: candidates (iteration 0) or parents (iterations >= 1)
    double *d_S64, *d_chi2_64;       // [E][cap]
    int32_t *d_nm64;
    int32_t *d_wire_label;
    double *d_wire_best;
};

cudaError_t refine_kth_pass(const RefineLaunch &L, const unsigned long long *d_prev, unsigned long long *d_cur, cudaStream_t s);
cudaError_t refine_candidates(const RefineLaunch &L, const unsigned long long *d_kth, cudaStream_t s);
cudaError_t refine_eval_select(const RefineLaunch &L, int mode, long long scale, const GridDev *d_grids, const double *d_axes,
                               int stride, const RefineParent *d_prev, RefineParent *d_out, int32_t *d_n_out, cudaStream_t s);
cudaError_t refine_labels(const RefineLaunch &L, int mode, const GridDev *d_grids, const double *d_axes, int stride,
                          const RefineParent *d_best, int32_t *d_labels, cudaStream_t s);
