/*
 * cdc_seedscan.h -- C ABI of the B200-native brute-force seed scan for a cylindrical drift chamber
 * (hot path of arXiv 1908.01949, "GPU Tracking in the COMET Phase-I Cylindrical Drift Chamber").
 *
 * Citations: PAPER.md:N = line N of the paper text; BJ = BASELINE.json; "reading Cn" = DESIGN.md section 3.
 *
 * Conventions
 *   - plain C, no exceptions cross the boundary.  Every call returns int32_t: CDC_OK or a negative
 *     cdc_status.  cdc_last_error() gives a thread-local message for the last failing call.
 *   - units: mm, MeV/c, tesla, radians.
 *   - pointer names say where the memory lives: h_* = host, d_* = device (cuda:current device).
 *     All d_* buffers are CALLER-OWNED (the Python binding passes torch tensors' data_ptr()); the
 *     library never frees them and never keeps them after the call returns (it keeps its own copies
 *     inside the opaque handles).  Handles are created and destroyed by the library.
 *   - `stream` is a cudaStream_t passed as void* (NULL = the legacy default stream).  Calls enqueue
 *     work on it and return without synchronising, except where stated ("synchronises").
 *   - the seed's linear index, which is also the tie-break order of the argmax, is fixed:
 *       index = ((((i_theta * n_z + i_z) * n_px + i_px) * n_py + i_py) * n_pz + i_pz
 *     with axis order (theta0, z0, px0, py0, pz0) (five scanned parameters at R0 = 50 cm).
 */
#ifndef CDC_SEEDSCAN_H
#define CDC_SEEDSCAN_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
    CDC_OK = 0,
    CDC_ERR_INVALID = -1,     /* invalid argument (null pointer, n < 1, h <= 0, duplicate wire id, bad drift ...) */
    CDC_ERR_RANGE = -2,       /* out of range / table overflow (wire id, field table too small, pool overflow) */
    CDC_ERR_CUDA = -3,        /* a CUDA runtime call or kernel launch failed */
    CDC_ERR_NOMEM = -4,       /* host or device allocation failed */
    CDC_ERR_NOT_READY = -5    /* call order violated (cdc_best_track before cdc_seed_scan) */
} cdc_status;

typedef struct cdc_geometry cdc_geometry;   /* immutable after create: wire tables + field (A0) */
typedef struct cdc_events cdc_events;       /* one batch of events: hits, per-wire tables, scan scratch (A1) */

/* Detector description ("eighteen layers with stereo configuration"; numbers from BJ configs[0];
 * reading C2).  Layer j: waist radius r_mm[j] (radius of the wire at z = 0), n_wires[j] wires at azimuth
 * phi0_rad[j] + 2 pi k / n_wires[j], signed stereo angle stereo_rad[j].  Wire (j, k) is the line
 *   w0 = (r cos phi, r sin phi, 0),  u = (-sin(eps) sin phi, sin(eps) cos phi, cos(eps)),  |z| <= z_half_mm.
 * The fast lookup requires equally spaced layers and equal |stereo| (else CDC_ERR_INVALID).
 * h_wire: optional canonical per-wire table [W][5] = (w0x, w0y, ux, uy, uz) in fp32 (W = sum n_wires); when
 * NULL the library builds it from the layer description in fp64 and rounds once to fp32.  Copied. */
typedef struct {
    int32_t n_layers;
    const double *r_mm;
    const int32_t *n_wires;
    const double *phi0_rad;
    const double *stereo_rad;
    const float *h_wire;
    double z_half_mm, R0_mm, r_out_mm;      /* 750, 500, 827 */
} cdc_geometry_desc;

/* Magnetic field ("1T"; PAPER.md:73 the field is uploaded to the GPU; BJ configs[3]; reading C3).
 * kind 0: uniform (0, 0, bz_T).  kind 1: axisymmetric table, h_br_bz[iz][ir][2] = (B_r, B_z) fp32 at
 * r = r0_mm + ir dr_mm, z = z0_mm + iz dz_mm, bilinear in (rho, z), cell index clamped to the table.  Copied. */
typedef struct {
    int32_t kind;
    double bz_T;
    int32_t nr, nz;
    double r0_mm, z0_mm, dr_mm, dz_mm;
    const float *h_br_bz;
} cdc_field_desc;

/* 5-D seed grid of one event: axis a (theta, z, px, py, pz) has n[a] nodes lo[a] + (first[a] + i) step[a], i = 0 ..
 * n[a] - 1.  first[a] (>= 0, normally 0) lets a slab of a larger grid be scanned with node values that are
 * bit-identical to the larger grid's (one event split over several GPUs along theta); the linear
 * seed index is local to the slab.  cdc_refine_tracks and cdc_peel_turns require first = 0. */
typedef struct {
    double lo[5], step[5];
    int32_t n[5];
    int32_t first[5];
} cdc_grid_spec;

/* Propagation and scoring parameters (BJ configs[0]: fixed 2 mm step, <= 1500 steps, 1 mm window).
 * window_mm: a hit matches iff (D - drift)^2 < lambda = window_mm^2  (Eq. (1), reading C9/C10).
 * eloss_MeV_per_mm: constant momentum loss per mm of in-gas path (BJ configs[2], reading C6); the scan accepts up to
 *   ~3e-3 MeV/mm at h = 2 mm (CDC_ERR_RANGE above: its curvature bounds assume < 0.04 MeV/c lost per lookup period).
 * rescore_margin: seeds whose fp32 score is within this of the event's fp32 maximum are re-evaluated in
 * fp64 by cdc_best_track (reading C11); <= 0 selects the default 0.05.
 * kernel_variant: 0 = the production kernel (one seed per thread; (x, y) components as packed fp32 pairs);
 *   1 = two z0-neighbour seeds per thread, every quantity a packed pair of the two seeds (csrc/scan_pair.cu): measured
 *   slower on B200 (profiles/r2_pair_kernel.md), kept as the comparison point; per-seed n_match,
 *   step counts, best seed and labels are identical, tests/test_gpu_pair.py checks it;
 *   2 = lane refill (csrc/scan_refill.cu): a thread runs two seeds in a row, the short track of one 32-seed chunk and
 *   the long track of the next, and a per-step warp vote ends the warp: every lane stays live (32.0 of 32 in the step
 *   against 29.3 / 30.8) but the second seeds are out of step with their z0 neighbours and the lookup and live-wire
 *   code pay more than the step saves: measured slower (profiles/r2_refill_kernel.md), kept as the comparison point;
 *   per-seed n_match, chi2, positions, best seed and labels are bit-identical, tests/test_gpu_refill.py checks it;
 *   3 = the production kernel with the field reuse off (tabulated field: B is evaluated at every step's start vertex
 *   instead of being carried over from the previous step's 4th-stage point where that is provably below fp32
 *   resolution, reading C22): the A / B switch for that one decision (tests/test_gpu_edges.py,
 *   `bench.py --kernel-variant 3`); identical to 0 in the uniform field. */
typedef struct {
    double h_mm;
    int32_t max_steps;
    double window_mm;
    double eloss_MeV_per_mm;
    int32_t charge;                          /* -1 for e-  */
    double rescore_margin;
    int32_t kernel_variant;
} cdc_scan_params;

/* Hough circle vote (Fig. 4; parametrisation is reading C13): accumulator over circle
 * centres (cx, cy) in [-half_xy, half_xy) and radii R in [R_lo, R_hi); a hit votes for a bin iff
 * | |c - x_hit| - R | < tol at the bin centre; bins with | |c| - R | > origin + tol are ineligible. */
typedef struct {
    double bin_xy_mm, bin_R_mm, tol_mm, R_lo_mm, R_hi_mm, half_xy_mm, origin_mm;   /* 4, 4, 6, 240, 364, 460, 100 */
    double half_theta_rad, half_pt_MeV;                                            /* 0.03, 7.5 */
} cdc_hough_params;

/* Optional per-seed diagnostics of cdc_seed_scan (parity tests): state after the last step. */
typedef struct {
    int32_t n_steps, turns, m_gas, pad;
    double x, y, z;
} cdc_seed_debug;

/* Counters of the last cdc_seed_scan on an event batch (for throughput / roofline accounting). */
typedef struct {
    uint64_t n_seeds;          /* seeds propagated */
    uint64_t n_steps;          /* RKN steps taken, summed over seeds */
    uint64_t n_gas_steps;      /* of which started in the gas volume (rho >= R0); counted only with energy loss or the
                                  debug output (otherwise 0: the production kernel does not track the flag) */
    uint64_t n_approach_tests; /* live candidate wires examined (g evaluated) */
    uint64_t n_pool;           /* candidate-pool entries appended (reading C11) */
    uint64_t pool_cap;
    uint64_t n_lookups;        /* in-gas steps that fell inside the wire band and ran the layer/cell lookup */
    uint64_t n_g1;             /* candidates whose far-end g was evaluated (g_n <= 0) */
    uint64_t n_approaches;     /* owned approaches (g_n <= 0 < g_{n+1}) scored against the window */
    double kernel_ms;          /* device time of the propagate-and-score kernel alone (CUDA events on `stream`) */
} cdc_scan_stats;

const char *cdc_last_error(void);

/* A0: geometry and field tables -> device.  Synchronises.  Errors: INVALID (null, n_layers not in [1, 32],
 * unequal layer pitch / |stereo|), RANGE (field table does not cover rho <= r_out + 2h_max(=8 mm), |z| <= z_half + 8). */
int32_t cdc_geometry_create(const cdc_geometry_desc *geom, const cdc_field_desc *field, cdc_geometry **out);
int32_t cdc_geometry_destroy(cdc_geometry *g);
/* Copy the canonical fp32 wire table [W][5] to host memory (W returned through n_wires_total if non-null). */
int32_t cdc_geometry_wire_table(const cdc_geometry *g, float *h_wire_or_null, int32_t *n_wires_total);

/* A1: hits of a batch of events -> library-owned device copies, a dense per-wire drift table
 * (sentinel -1 = no hit) and a per-wire hit bitmask per event (hits uploaded to the GPU;
 * BJ north_star: "hits binned by (layer, phi-cell) so each step's lookup is O(1)").
 * h_hit_offsets: host, n_events + 1 prefix offsets into wire_id / drift_mm.  wire_id / drift_mm live on the
 * host (hits_on_device = 0) or on the device (1).  Hits need not be sorted.  Synchronises (validation result).
 * Errors: RANGE wire id outside [0, W); INVALID duplicate wire id within an event, drift outside [0, 8] mm (the cell half-width, BJ configs[0]) or non-finite. */
int32_t cdc_event_upload(const cdc_geometry *g, int32_t n_events, const int32_t *h_hit_offsets,
                         const int32_t *wire_id, const float *drift_mm, int32_t hits_on_device,
                         void *stream, cdc_events **out);
int32_t cdc_events_destroy(cdc_events *ev);
/* Copy the A1 tables to host memory: h_drift_of_wire [n_events][W] f32, h_hit_bits [n_events][ceil(W/32)] u32
 * (either may be NULL).  Synchronises. */
int32_t cdc_events_tables(const cdc_events *ev, float *h_drift_of_wire, uint32_t *h_hit_bits);

/* A2: Hough pre-vote.  d_zref_mm[e]: z at which the stereo wires' (x, y) are taken.
 * Outputs per event: d_ranges[e][3][2] = (lo, hi) of theta0, px0, py0 (f64); d_peak[e][4] = (iR, icy, icx, votes)
 * with ties to the lowest linear bin index; d_accum_or_null[e][nR][ncy][ncx] u32 (full accumulator, optional).
 * The field's bz_T and params->charge fix the sense of rotation. */
int32_t cdc_hough_dims(const cdc_hough_params *hp, int32_t *dims3 /* nR, ncy, ncx */);
int32_t cdc_hough_seed_ranges(const cdc_geometry *g, const cdc_events *ev, const cdc_hough_params *hp,
                              int32_t charge, const float *d_zref_mm, double *d_ranges, int32_t *d_peak,
                              uint32_t *d_accum_or_null, void *stream);

/* A2 without any allocation: the same Hough vote (same kernels, same results bit for bit) for callers that cannot
 * allocate -- code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc.  It calls no
 * cudaMalloc / cudaFree or allocating library routine, and needs no cdc_events handle (whose creation allocates): the
 * hits are plain device arrays, d_hit_offsets [n_events + 1] (ascending, hits of event e are [offsets[e], offsets[e + 1]))
 * and d_wire_id [offsets[n_events]], every id in [0, W) -- NOT checked here, an id outside reads outside the wire
 * table.  g: a geometry created earlier (at set-up) on the current device.  Outputs as cdc_hough_seed_ranges (device,
 * caller-owned; every element of d_accum_or_null is written).  The only scratch, one packed peak key per event, is a
 * static device array of CDC_HOUGH_NOALLOC_MAX_EVENTS entries (32 KB on every GPU that loads the library, until exit):
 * n_events beyond that is CDC_ERR_RANGE.  The first call on a device looks the array's address up (a call with
 * n_events = 0 does only that and launches nothing: make it at set-up, before a capture).  EVERY call shares the array:
 * each call clears the keys it uses on `stream` before the vote, but calls that overlap on the GPU (different streams,
 * no ordering between them) race on it -- order them.  Asynchronous. */
#define CDC_HOUGH_NOALLOC_MAX_EVENTS 4096
int32_t cdc_hough_seed_ranges_noalloc(const cdc_geometry *g, int32_t n_events, const int32_t *d_hit_offsets,
                                      const int32_t *d_wire_id, const cdc_hough_params *hp, int32_t charge,
                                      const float *d_zref_mm, double *d_ranges, int32_t *d_peak,
                                      uint32_t *d_accum_or_null, void *stream);

/* A3-A7: the seed scan.  Every seed of every event's grid is propagated by Nystroem-RK4 (PAPER.md:55,
 * reading C5) in fp32 with compensated state, wires near each step are looked up (reading C8), owned
 * approaches to fired wires are scored (readings C9/C10), and the per-event maximum of
 * S = n_match - chi2 / lambda is reduced into d_best_key[e] = (bits(S_fp32) << 32) | (0xFFFFFFFF - index).
 * h_grids: host, one spec per event (product of n <= 2^31 - 1, each n <= 4096).
 * d_n_match_or_null / d_chi2_or_null: per-seed outputs, events concatenated in grid order (sum of n_seeds).
 * d_debug_or_null: cdc_seed_debug per seed.  Seeds close to the running maximum are appended to the
 * library-owned candidate pool of `ev` for cdc_best_track.  Asynchronous. */
int32_t cdc_seed_scan(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                      const cdc_scan_params *params, uint32_t *d_n_match_or_null, float *d_chi2_or_null,
                      cdc_seed_debug *d_debug_or_null, uint64_t *d_best_key, void *stream);
/* the seed scan with the ADAPTIVE step of the propagator the paper cites ("the RKN method
 * was used for the track parameter propagation [5]"; [5] = Lund et al.; reading C19 applied to the scan).
 * Step lengths h 2^j with h 2^j <= h_max_mm; a trial whose error estimate H^2 max|k1 - k2 - k3 + k4| exceeds tol_mm is
 * repeated one level down (never below h), an accepted step with estimate <= tol / 32 raises the level of the next
 * trial.  params->max_steps caps the PATH in units of h; the in-gas count and the energy loss are in those units.
 * Outputs per seed (device, caller-owned): d_n_match u32, d_chi2 f32 (either may be NULL), d_debug_or_null (n_steps =
 * accepted steps, m_gas = in-gas path units, pad = path units, final position), d_levels_or_null i32 [seeds][8]
 * (accepted steps per level 0..6; [7] = hash of the level sequence, hash = hash * 31 + (level + 1)); d_best_key per
 * event: the fused fp32 arg max, packed as cdc_seed_scan packs it.  The step-size decisions are taken in fp32: a seed
 * whose estimate comes within ~2 % of a threshold can take another sequence than an fp64 evaluation (DESIGN.md
 * section 15).  No candidate pool is filled: cdc_best_track does not apply.  h_max is limited by the 2 x 2 wire lookup
 * (CDC_ERR_RANGE above ~12 mm).  Asynchronous. */
int32_t cdc_seed_scan_adaptive(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                               const cdc_scan_params *params, double tol_mm, double h_max_mm, uint32_t *d_n_match_or_null,
                               float *d_chi2_or_null, cdc_seed_debug *d_debug_or_null, int32_t *d_levels_or_null,
                               uint64_t *d_best_key, void *stream);
/* Counters of the last scan.  Synchronises `stream`. */
int32_t cdc_scan_get_stats(const cdc_events *ev, cdc_scan_stats *h_out, void *stream);

/* A8-A9: exact best seed and hit -> turn labels ("lowest E", "hits with d^2 < lambda are
 * classified"; readings C11/C12).  Pool candidates within rescore_margin of the fp32 maximum are re-evaluated
 * in IEEE fp64 without FMA contraction; the maximum of S (ties: lowest index) is the best seed; its matched
 * approaches label each hit with a turn index, or -1.  Per event: d_best_seed i64, d_best_n_match u32,
 * d_best_chi2 f64; d_labels i32 per hit (events concatenated in upload order).  Must follow cdc_seed_scan on
 * the same stream with the same grids / params.  Synchronises `stream` once (an 8-byte read-back of the number of
 * candidates, which sizes the launches).  The candidate pool cannot silently lose the best seed: if the scan appended
 * more candidates than the pool holds (many near-ties, e.g. a plateau of identical seeds), the near-ties of the FINAL
 * fp32 maximum are collected again by a second pass of the scan into a pool sized for them (up to 2^26 entries;
 * beyond that CDC_ERR_RANGE).  cdc_scan_get_stats().n_pool is then the second pass's count. */
int32_t cdc_best_track(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                       const cdc_scan_params *params, const uint64_t *d_best_key, int64_t *d_best_seed,
                       uint32_t *d_best_n_match, double *d_best_chi2, int32_t *d_labels, void *stream);

/* The whole path with host buffers in and out (upload, optional Hough vote, scan, best track, read-back): the
 * end-to-end call.  If hp is non-NULL the Hough vote runs (h_zref_mm required) and its ranges are returned in
 * h_ranges_or_null [n_events][3][2]; if hough_sets_axes is also non-zero the (theta, px, py) axes of every grid are
 * replaced by n[a] nodes spanning those ranges (BJ configs[2]: "Hough pre-vote narrows the ranges"), otherwise the grids
 * are scanned as given.  Outputs (host): h_best_seed, h_best_n_match, h_best_chi2, h_best_key per event; h_labels per
 * hit.  Synchronises. */
int32_t cdc_find_tracks_host(const cdc_geometry *g, int32_t n_events, const int32_t *h_hit_offsets,
                             const int32_t *h_wire_id, const float *h_drift_mm, const cdc_grid_spec *h_grids,
                             const cdc_scan_params *params, const cdc_hough_params *hp_or_null,
                             const float *h_zref_mm_or_null, int32_t hough_sets_axes, int64_t *h_best_seed,
                             uint32_t *h_best_n_match, double *h_best_chi2, uint64_t *h_best_key, int32_t *h_labels,
                             double *h_ranges_or_null, void *stream);

/* Coarse-to-fine refinement around the seed scan ("we took the several candidate seeds with the lowest
 * E, and make other seed sets around them with finer granularity ... repeated ten times"; reading C17):
 * iteration 0 scans h_grids; iteration t = 1..n_iterations scans the 3^5 nodes q_parent + {-d, 0, +d}^5, d = 2^(T-t),
 * around each of the n_parents best seeds so far, on the integer lattice of the finest pitch step / 2^T
 * (value = lo + q * step / 2^T); parents are ordered by (S descending, sub-grid rank, index), duplicates skipped.
 * Outputs (host, per event): best seed values [E][5], S, n_match, chi2, lattice point q [E][5]; labels per hit
 * (optional); the parents of every iteration (optional): S [E][T+1][K] (-1 = none) and q [E][T+1][K][5].
 * Scores, selection and labels are fp64 (bit-equal to a plain IEEE evaluation).  Synchronises. */
typedef struct {
    int32_t n_parents;        /* K, 1..8 */
    int32_t n_iterations;     /* T, 0..20 (the paper: ten) */
} cdc_refine_params;
int32_t cdc_refine_tracks(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids,
                          const cdc_scan_params *params, const cdc_refine_params *rp, double *h_best_seed,
                          double *h_best_S, uint32_t *h_best_n_match, double *h_best_chi2, int64_t *h_best_q,
                          int32_t *h_labels_or_null, double *h_trace_S_or_null, int64_t *h_trace_q_or_null,
                          void *stream);

/* Classification efficiency and purity per turn partition (Eq. (2), (3)) of hit -> turn labels against
 * truth labels (-1 = noise), per event of `ev` (hits in upload order): d_confusion [E][n][n] (truth i classified as j),
 * d_c_true [E][n], d_noise_into [E][n] (noise hits classified into a partition; not part of Eq. (3)'s sum),
 * d_efficiency, d_purity [E][n] f64 (-1 where the denominator is 0).  n_turns <= 8.  Asynchronous. */
int32_t cdc_classification_quality(const cdc_events *ev, int32_t n_turns, const int32_t *d_labels,
                                   const int32_t *d_truth_turn, int32_t *d_confusion, int32_t *d_c_true,
                                   int32_t *d_noise_into, double *d_efficiency, double *d_purity, void *stream);
/* N_c ("the number of hits commonly found from the both direction"): hits that scan A labels turn_a and
 * scan B labels turn_b (a turn of -1 = any turn >= 0), per event.  A backward scan is an ordinary cdc_seed_scan with
 * params->charge = -q and a grid around the exit-side seed with the momentum reversed.  Asynchronous. */
int32_t cdc_common_hits(const cdc_events *ev, const int32_t *d_labels_a, const int32_t *d_labels_b,
                        int32_t turn_a, int32_t turn_b, int32_t *d_n_common, void *stream);

/* Turn-partition peeling: the event reconstruction loop of PAPER.md:83 (section 2.3, Fig. 7) without the Kalman fit
 * (reading C18).  Per event, for partition k = 0, 1, ...:
 *   scan the partition's grid over the still unclassified hits (cdc_seed_scan + cdc_best_track); the partition's hits
 *   are those the best seed's track matches in its FIRST passage through the gas (turn label 0; "classified
 *   as the hits of the turn partition being investigated"); they are removed from the event; the best seed is
 *   extrapolated with the same fp64 RKN steps to its next outward crossing of rho = R0, and the neighbouring
 *   partition's grid is n[] nodes per axis centred on that state, +- half_width[] (theta rad, z mm, px, py, pz MeV/c;
 *   node i = (c - hw) + i * 2 hw / (n - 1), or c alone when n = 1).
 * Stop reasons (h_status): 1 = fewer than min_hits unclassified hits remain (the paper: ten), 2 = the partition has
 * fewer than min_classified hits (it is discarded), 3 = max_partitions recorded, 4 = the track ended (end plate, outer
 * wall, extrap_max_steps, p <= 1 MeV/c) before the next entrance.  params->charge / reversed exit-side seeds make the
 * extrapolation the paper's backward one (see cdc_common_hits).
 * h_grids0: partition 0's grid per event.  Host outputs: h_n_partitions [E], h_status [E], h_seeds [E][P][5] (best
 * seed values), h_n_match [E][P], h_chi2 [E][P], h_centres_or_null [E][P][5] (grid centre of partition k >= 1; row 0
 * is zero); P = max_partitions <= 8; rows k >= h_n_partitions[e] are zero.  d_partition [total_hits] (device, upload
 * order): partition index of every hit, or -1.  The events' hit tables are restored before the call returns.
 * Synchronises once per partition (the host turns the extrapolated state into the next grid: atan2 and the cos / sin
 * of the theta nodes come from the host libm, reading C11).  CDC_ERR_RANGE if a scan's candidate pool overflowed. */
typedef struct {
    int32_t max_partitions;   /* P, 1..8 */
    int32_t min_hits;         /* >= 0; the paper: 10 */
    int32_t min_classified;   /* >= 0 */
    int32_t extrap_max_steps; /* >= 1 */
    int32_t n[5];             /* nodes per axis of the grids of partitions 1.. (1..4096 each) */
    int32_t pad_;
    double half_width[5];
    double extrap_tol_mm;     /* 0: the extrapolation uses the scan's fixed step h.  > 0: adaptive step (reading C19): */
    double extrap_h_max_mm;   /*    step lengths h 2^j in [h, extrap_h_max_mm], controlled by the local error estimate
                               *    h^2 max|k1 - k2 - k3 + k4| of the paper's propagator reference [5]:
                               *    halved on err > tol, doubled after err <= tol / 32; the crossing of rho = R0 is always
                               *    taken on a chord of length h */
} cdc_peel_params;
int32_t cdc_peel_turns(const cdc_geometry *g, cdc_events *ev, const cdc_grid_spec *h_grids0,
                       const cdc_scan_params *params, const cdc_peel_params *pp, int32_t *h_n_partitions,
                       int32_t *h_status, double *h_seeds, uint32_t *h_n_match, double *h_chi2,
                       double *h_centres_or_null, int32_t *d_partition, void *stream);

/* MEASURED COMPARISON POINT, not the product path: the paper's own thread mapping (v1, PAPER.md:73,
 * Fig. 6) -- one block per seed, one thread per fired wire, every thread repeating the RKN propagation -- re-created on
 * sm_100a with the same arithmetic and scoring rule as cdc_seed_scan.  Evaluates the n_seeds seeds d_seed_index[] (linear
 * indices into h_grid) of one event; outputs d_n_match / d_chi2 [n_seeds].  No energy loss.  Asynchronous after an
 * internal table copy. */
int32_t cdc_seed_scan_paper_mapping(const cdc_geometry *g, cdc_events *ev, int32_t event, const cdc_grid_spec *h_grid,
                                    const cdc_scan_params *params, const int64_t *d_seed_index, int32_t n_seeds,
                                    uint32_t *d_n_match, float *d_chi2, void *stream);

/* MEASURED COMPARISON POINT, not the product path: the paper's second mapping ("kernel function
 * separation").  Kernel 1: one thread per seed propagates it and records every vertex (32 bytes x
 * n_seeds x (max_steps + 1) of device memory, CDC_ERR_RANGE above 16 GiB); kernel 2: one block per seed, one thread per
 * fired wire, walks the record and takes the approaches between recorded vertices.  Same arguments and outputs as
 * cdc_seed_scan_paper_mapping, bit-equal results; h_ms2_or_null (host, 2 doubles): device time of the two kernels in
 * ms (the call then synchronises).  No energy loss. */
int32_t cdc_seed_scan_paper_mapping_v2(const cdc_geometry *g, cdc_events *ev, int32_t event, const cdc_grid_spec *h_grid,
                                       const cdc_scan_params *params, const int64_t *d_seed_index, int32_t n_seeds,
                                       uint32_t *d_n_match, float *d_chi2, double *h_ms2_or_null, void *stream);

/* Number of kernels this library has launched in this process so far (bench.py's gpu_launches). */
uint64_t cdc_kernel_launch_count(void);

/* Register-only FFMA chain: the empirical FP32 peak used as the roofline denominator.  Runs `iters`
 * dependent-chain iterations on every SM, returns achieved FLOP/s (2 per FFMA).  Synchronises. */
int32_t cdc_fp32_peak_probe(int32_t iters, double *h_flops_per_s, double *h_ms, void *stream);

/* Issue rates of sm_100a's packed fp32 instructions (PTX fma/add/mul.rn.f32x2 -> SASS FFMA2/FADD2/FMUL2) against the
 * scalar ones, alone and interleaved with integer-pipe work: register-only chains on every SM.  mode: 0 FFMA, 1 FFMA2,
 * 2 FADD, 3 FADD2, 4 FMUL2, 5 FFMA2 + LOP3, 6 FFMA + LOP3, 7 FFMA2 + FFMA.  Returns the kernel time, the warp
 * instructions and the flops it executed (the measurement behind the packed pairs of the scan kernel, DESIGN.md
 * section 7; `python bench.py --issue-probe`).  Synchronises. */
int32_t cdc_fp32_issue_probe(int32_t mode, int32_t iters, double *h_ms, double *h_warp_instructions, double *h_flops,
                             void *stream);

#ifdef __cplusplus
}
#endif
#endif /* CDC_SEEDSCAN_H */
