// Coarse-to-fine refinement of the seed scan ("we took the several candidate seeds with
// the lowest E, and make other seed sets around them with finer granularity ... repeated ten times"; reading C17).
//
// Iteration 0 is the ordinary fp32 scan of the initial grid with its per-seed scores materialised; the K best are
// found exactly: K passes of a packed-key maximum give the K-th largest fp32 score, every seed within `margin` of it
// is re-evaluated in fp64 (one warp per seed, eval64.cuh), and the K best fp64 scores win.  Iterations 1..T evaluate
// the K x 3^5 sub-grid nodes directly in fp64 (a few thousand warps) and select again.  Selection order:
// (S descending, rank of the sub-grid, linear index), skipping lattice points already taken.
// Compiled with -fmad=false (see eval64.cuh).
#include "eval64.cuh"
#include "refine.cuh"

namespace {

constexpr int kSub = 3, kSubSeeds = 243;

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, v, o);
        v = other > v ? other : v;
    }
    return v;
}

__device__ __forceinline__ unsigned long long seed_key(uint32_t nm, float chi2, float inv_lambda, uint32_t idx)
{
    const float S = fmaxf(fmaf(-chi2, inv_lambda, (float)nm), 0.0f);      // as the scan kernel packs it
    return ((unsigned long long)__float_as_uint(S) << 32) | (0xFFFFFFFFu - idx);
}

// one pass: per event, the largest key strictly below prev[e]
__global__ void kth_key_kernel(const GridDev *grids, const uint32_t *n_match, const float *chi2, float inv_lambda,
                               const unsigned long long *prev, unsigned long long *cur)
{
    const int e = blockIdx.y;
    const GridDev G = grids[e];
    const unsigned long long bound = prev[e];
    unsigned long long best = 0ull;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < G.n_seeds; i += (int64_t)gridDim.x * blockDim.x) {
        const unsigned long long k = seed_key(n_match[G.out_offset + i], chi2[G.out_offset + i], inv_lambda, (uint32_t)i);
        if (k < bound && k > best) best = k;
    }
    best = warp_max_u64(best);
    if ((threadIdx.x & 31) == 0 && best) atomicMax(cur + e, best);
}

// seeds whose fp32 score is within margin of the K-th largest -> candidate list of the event
__global__ void cand_kernel(const GridDev *grids, const uint32_t *n_match, const float *chi2, float inv_lambda,
                            const unsigned long long *kth, float margin, uint32_t *cand_idx, int32_t *cand_count, int32_t cap)
{
    const int e = blockIdx.y;
    const GridDev G = grids[e];
    const float thr = __uint_as_float((uint32_t)(kth[e] >> 32)) - margin;
    for (int64_t i = (int64_t)blockIdx.x * blockDim.x + threadIdx.x; i < G.n_seeds; i += (int64_t)gridDim.x * blockDim.x) {
        const float S = fmaxf(fmaf(-chi2[G.out_offset + i], inv_lambda, (float)n_match[G.out_offset + i]), 0.0f);
        if (S >= thr) {
            const int pos = atomicAdd(cand_count + e, 1);
            if (pos < cap) cand_idx[(size_t)e * cap + pos] = (uint32_t)i;
        }
    }
}

// one warp per entry: fp64 score.  mode 0: entry j of event e is seed cand_idx[e][j] of the initial grid e;
// mode 1: entry j is node j % 243 of sub-grid e * K + j / 243 (hits of event e).
__global__ void __launch_bounds__(128) eval_entries_kernel(const BestArgs A, int mode, int n_events, int K, int cap,
                                                           const uint32_t *cand_idx, const int32_t *count,
                                                           double *S64, double *chi2, int32_t *nm)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    load_layers(A.g, s_layer);
    const int64_t wid = ((int64_t)blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int e = (int)(wid / cap), j = (int)(wid % cap);
    if (e >= n_events) return;
    const int n = mode == 0 ? min(count[e], cap) : count[e] * kSubSeeds;
    if (j >= n) return;
    Eval64 ev;
    if (mode == 0) eval_seed64(A, s_layer, e, e, cand_idx[(size_t)e * cap + j], ev, nullptr, nullptr, nullptr, nullptr);
    else eval_seed64(A, s_layer, e * K + j / kSubSeeds, e, (uint32_t)(j % kSubSeeds), ev, nullptr, nullptr, nullptr, nullptr);
    if ((threadIdx.x & 31) == 0) {
        const size_t o = (size_t)e * cap + j;
        S64[o] = (double)ev.n_match - ev.chi2 / A.lambda;      // C10
        chi2[o] = ev.chi2; nm[o] = ev.n_match;
    }
}

struct Cmp {               // selection order: S descending, then rank, then index
    double S; int rank, idx, j;
};
__device__ __forceinline__ bool better(const Cmp &a, const Cmp &b)
{
    if (a.S != b.S) return a.S > b.S;
    if (a.rank != b.rank) return a.rank < b.rank;
    return a.idx < b.idx;
}

// one block per event: the K best distinct lattice points among the entries just evaluated
__global__ void __launch_bounds__(256) select_kernel(int mode, int K, int cap, long long scale /* 2^T or d */,
                                                     const GridDev *grids0, const uint32_t *cand_idx, const int32_t *count,
                                                     const double *S64, const double *chi2, const int32_t *nm,
                                                     const RefineParent *prev, RefineParent *out, int32_t *n_out)
{
    __shared__ Cmp s_best[256];
    __shared__ long long s_q[8][5];
    const int e = blockIdx.x;
    const int n = mode == 0 ? min(count[e], cap) : count[e] * kSubSeeds;
    int taken = 0;
    for (int r = 0; r < K; ++r) {
        Cmp mine; mine.S = -1.0; mine.rank = 0x7fffffff; mine.idx = 0x7fffffff; mine.j = -1;
        for (int j = threadIdx.x; j < n; j += blockDim.x) {
            Cmp c; c.S = S64[(size_t)e * cap + j]; c.j = j;
            long long q[5];
            if (mode == 0) {
                c.rank = 0; c.idx = (int)cand_idx[(size_t)e * cap + j];
                uint32_t t = (uint32_t)c.idx;
                for (int a = 4; a >= 0; --a) { q[a] = (long long)(t % (uint32_t)grids0[e].n[a]) * scale; t /= (uint32_t)grids0[e].n[a]; }
            } else {
                c.rank = j / kSubSeeds; c.idx = j % kSubSeeds;
                int t = c.idx;
                for (int a = 4; a >= 0; --a) { q[a] = prev[e * K + c.rank].q[a] + (long long)(t % kSub - 1) * scale; t /= kSub; }
            }
            bool dup = false;
            for (int k = 0; k < taken; ++k) {
                bool same = true;
                for (int a = 0; a < 5; ++a) same = same && (s_q[k][a] == q[a]);
                dup = dup || same;
            }
            if (!dup && (mine.j < 0 || better(c, mine))) mine = c;
        }
        s_best[threadIdx.x] = mine;
        __syncthreads();
        for (int o = 128; o > 0; o >>= 1) {
            if (threadIdx.x < o) {
                const Cmp b = s_best[threadIdx.x + o];
                if (b.j >= 0 && (s_best[threadIdx.x].j < 0 || better(b, s_best[threadIdx.x]))) s_best[threadIdx.x] = b;
            }
            __syncthreads();
        }
        const Cmp w = s_best[0];
        __syncthreads();
        if (w.j < 0) break;                      // fewer distinct entries than K
        if (threadIdx.x == 0) {
            RefineParent P;
            if (mode == 0) {
                uint32_t t = (uint32_t)w.idx;
                for (int a = 4; a >= 0; --a) { P.q[a] = (long long)(t % (uint32_t)grids0[e].n[a]) * scale; t /= (uint32_t)grids0[e].n[a]; }
            } else {
                int t = w.idx;
                for (int a = 4; a >= 0; --a) { P.q[a] = prev[e * K + w.rank].q[a] + (long long)(t % kSub - 1) * scale; t /= kSub; }
            }
            P.S = w.S; P.chi2 = chi2[(size_t)e * cap + w.j]; P.n_match = nm[(size_t)e * cap + w.j];
            P.rank = w.rank; P.idx = w.idx; P.pad = 0;
            out[e * K + taken] = P;
            for (int a = 0; a < 5; ++a) s_q[taken][a] = P.q[a];
        }
        taken += 1;
        __syncthreads();
    }
    if (threadIdx.x == 0) n_out[e] = taken;
}

// labels of the final best seed: one warp per event re-propagates it with the label tables on
__global__ void __launch_bounds__(128) refine_label_kernel(const BestArgs A, int n_events, int K, int mode,
                                                           const RefineParent *best /* [E][K], entry 0 */,
                                                           int32_t *wire_label, double *wire_best)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    load_layers(A.g, s_layer);
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    if (e >= n_events) return;
    const RefineParent P = best[e * K];
    Eval64 ev;
    eval_seed64(A, s_layer, mode == 0 ? e : e * K + P.rank, e, (uint32_t)P.idx, ev, wire_label + (size_t)e * A.W,
                wire_best + (size_t)e * A.W, nullptr, nullptr);
}

__global__ void fill_i32r(int32_t *p, size_t n, int32_t v)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

__global__ void gather_labels_r(int32_t W, const int32_t *offsets, const int32_t *wire_id, const int32_t *wire_label,
                                int32_t *labels)
{
    const int e = blockIdx.y;
    const int i = offsets[e] + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= offsets[e + 1]) return;
    labels[i] = wire_label[(size_t)e * W + wire_id[i]];
}

BestArgs make_args(const RefineLaunch &L, const GridDev *grids, const double *axes, int stride)
{
    BestArgs A;
    A.g = L.g; A.grids = grids; A.axes = axes; A.axis_stride = stride;
    A.drift_tab = L.d_drift_tab; A.bits = L.d_bits; A.W = L.W; A.n_bit_words = L.n_bit_words;
    A.h = L.h; A.lambda = L.window * L.window; A.eloss_h = L.eloss * L.h; A.kq = CDC_KAPPA * (double)L.charge;
    A.max_steps = L.max_steps; A.lookup_every = L.lookup_every64;
    return A;
}

}  // namespace

cudaError_t refine_kth_pass(const RefineLaunch &L, const unsigned long long *d_prev, unsigned long long *d_cur, cudaStream_t s)
{
    cudaError_t e = cudaMemsetAsync(d_cur, 0, sizeof(unsigned long long) * (size_t)L.n_events, s);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)std::min<int64_t>((L.max_seeds_per_event + 255) / 256, 1024), (unsigned)L.n_events);
    kth_key_kernel<<<grid, 256, 0, s>>>(L.d_grids0, L.d_n_match, L.d_chi2, 1.0f / (float)(L.window * L.window), d_prev, d_cur);
    cdc_count_launch();
    return cudaGetLastError();
}

cudaError_t refine_candidates(const RefineLaunch &L, const unsigned long long *d_kth, cudaStream_t s)
{
    cudaError_t e = cudaMemsetAsync(L.d_count, 0, sizeof(int32_t) * (size_t)L.n_events, s);
    if (e != cudaSuccess) return e;
    dim3 grid((unsigned)std::min<int64_t>((L.max_seeds_per_event + 255) / 256, 1024), (unsigned)L.n_events);
    cand_kernel<<<grid, 256, 0, s>>>(L.d_grids0, L.d_n_match, L.d_chi2, 1.0f / (float)(L.window * L.window), d_kth, L.margin,
                                     L.d_cand_idx, L.d_count, L.cap);
    cdc_count_launch();
    return cudaGetLastError();
}

cudaError_t refine_eval_select(const RefineLaunch &L, int mode, long long scale, const GridDev *d_grids, const double *d_axes,
                               int stride, const RefineParent *d_prev, RefineParent *d_out, int32_t *d_n_out, cudaStream_t s)
{
    const BestArgs A = make_args(L, d_grids, d_axes, stride);
    const int64_t warps = (int64_t)L.n_events * L.cap;
    eval_entries_kernel<<<(unsigned)((warps + 3) / 4), 128, 0, s>>>(A, mode, L.n_events, L.K, L.cap, L.d_cand_idx, L.d_count,
                                                                   L.d_S64, L.d_chi2_64, L.d_nm64);
    select_kernel<<<L.n_events, 256, 0, s>>>(mode, L.K, L.cap, scale, L.d_grids0, L.d_cand_idx, L.d_count, L.d_S64, L.d_chi2_64,
                                             L.d_nm64, d_prev, d_out, d_n_out);
    cdc_count_launch(2);
    return cudaGetLastError();
}

cudaError_t refine_labels(const RefineLaunch &L, int mode, const GridDev *d_grids, const double *d_axes, int stride,
                          const RefineParent *d_best, int32_t *d_labels, cudaStream_t s)
{
    const BestArgs A = make_args(L, d_grids, d_axes, stride);
    const size_t nw = (size_t)L.n_events * L.W;
    fill_i32r<<<(unsigned)((nw + 255) / 256), 256, 0, s>>>(L.d_wire_label, nw, -1);
    refine_label_kernel<<<(L.n_events + 3) / 4, 128, 0, s>>>(A, L.n_events, L.K, mode, d_best, L.d_wire_label, L.d_wire_best);
    cdc_count_launch(2);
    if (L.max_hits_per_event > 0) {
        dim3 grid((unsigned)((L.max_hits_per_event + 127) / 128), (unsigned)L.n_events);
        gather_labels_r<<<grid, 128, 0, s>>>(L.W, L.d_offsets, L.d_wire_id, L.d_wire_label, d_labels);
        cdc_count_launch();
    }
    return cudaGetLastError();
}
