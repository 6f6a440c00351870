// Kernel arguments of the seed-scan kernels (scan.cu: one seed per thread; scan_pair.cu: two seeds per thread;
// scan_refill.cu: one seed per thread at a time, two in a row).
#pragma once
#include "cdc_internal.cuh"

constexpr int kBlock = 128;
constexpr int kMaxBitWords = 256;          // 8192 wires

struct ScanArgs {
    GeomDev gd;
    FieldDev fd;
    const GridDev *grids;
    const double *axes;
    int32_t axis_stride;
    const float *drift_tab;
    const uint32_t *bits;
    float h, h_half, h2_8, h2_2, h_6, h2_6;
    double kq;                 // kappa * charge
    float kq_rel;              // kq / fl32(kq) - 1: the systematic part of a = fl32(kq) / p (energy-loss path)
    double h6_64;              // h / 6 in fp64 (for the systematic-rounding correction)
    float lambda, inv_lambda, eloss_h, window;
    float u2_lo, u2_hi;        // lookup band in u^2, widened by (K - 1) h
    float uz, inv_uz;          // cos(eps) of the canonical wire table (one |stereo| for all layers)
    float delta_max, b_max, hold_path;   // bounds behind g_dead (see consider())
    int32_t max_steps, lookup_every, lookup_every_tight;
    float lookahead, tight_curv;
    // two-seed kernel: K = min(lookup_every, floor((k_margin - sep) * two_inv_h)), k_margin = excl - reach - sag;
    // around the seeds' own positions (tight curls, or K < 1): K0 = min(lookup_every_tight, 1 + floor((k_margin0 - sep) * inv_h))
    // (sep = half the two seeds' separation as a wire sees it; above sep_cap the pair does one lookup per seed)
    float k_margin, k_margin0, two_inv_h, inv_h, sin_eps, sep_cap;
    // field reuse (tabulated field): B at a step's start vertex is taken from the previous step's 4th-stage point where
    // reuse_c |a| (|a| reuse_b2 + grad_max) <= reuse_eps (scan.cu)
    float reuse_c, reuse_b2, reuse_eps;
    float margin;
    uint32_t *n_match;
    float *chi2;
    cdc_seed_debug *debug;
    unsigned long long *best_key;
    PoolEntry *pool;
    uint32_t pool_cap;
    unsigned long long *counters;
};

cudaError_t launch_seed_scan_pair(const ScanArgs &A, const ScanLaunch &L, bool eloss, bool track, cudaStream_t s);
cudaError_t launch_seed_scan_refill(const ScanArgs &A, const ScanLaunch &L, bool eloss, bool track, cudaStream_t s);
