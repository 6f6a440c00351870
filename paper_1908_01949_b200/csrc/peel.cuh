// Declarations shared by peel.cu (kernels, -fmad=false) and abi_peel.cu (host driver of cdc_peel_turns).
#pragma once
#include "cdc_internal.cuh"

struct PeelLaunch {
    Geom64 g;
    int32_t n_events, W, n_bit_words, max_hits_per_event;
    const int32_t *d_offsets, *d_wire_id;
    uint32_t *d_bits;                 // [E][n_bit_words] fired-wire bitmap of the unclassified hits (modified)
    const GridDev *d_grids;           // grids of the partition just scanned
    const double *d_axes;
    int32_t axis_stride;
    double h, eloss, kq;
    int32_t extrap_max_steps;
    double extrap_tol, extrap_h_max;  // tol > 0: adaptive extrapolation (reading C19)
    const int32_t *d_labels;          // hit -> turn labels of the partition's best seed
    const int64_t *d_best_seed;       // its linear index per event (-1: none)
    const int32_t *d_active;          // [E] 1 = the event is still being peeled
    int32_t *d_partition;             // [total_hits]
    int32_t *d_counts;                // [E][2]: hits of this partition, unclassified hits before it
    double *d_next;                   // [E][6]: x, y, z, px, py, pz at the next entrance
    int32_t *d_next_ok;               // [E]
};

// counts, then (where the partition is kept) marks its hits and clears their wires; extrapolates the best seed
cudaError_t peel_partition(const PeelLaunch &L, int k, int min_classified, cudaStream_t s);
