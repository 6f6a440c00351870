// A8-A9: exact re-score of the near-best seeds and hit -> turn labels of the best seed.
//
// THIS FILE IS COMPILED WITH -fmad=false: every fp64 +, -, *, /, sqrt below is a single IEEE-754 operation in
// the order DESIGN.md section 3 (readings C4-C10, C12) writes the formulas, left to right, so the result is a
// function of the inputs only and can be compared bit for bit with any other IEEE evaluation of the same
// formulas (reading C11).  Transcendentals appear only where they cannot change the result: in the choice of
// candidate wires (a superset by construction, reading C8).
//
//   PAPER.md:55      RKN propagation                           -> rkn_step64()
//   PAPER.md:55,:69  DCA, left/right ambiguity                 -> eval_seed64()
//   PAPER.md:65-69   Eq. (1), S = n_match - chi2 / lambda      -> rescore_kernel / pick_kernel
//   PAPER.md:69      "hits with d^2 < lambda are classified"   -> label_kernel
#include <algorithm>

#include "cdc_internal.cuh"

#include "eval64.cuh"

namespace {

__device__ __forceinline__ uint32_t pool_size(const unsigned long long *counters, uint32_t cap)
{
    const unsigned long long c = counters[CNT_POOL];
    return (uint32_t)(c < (unsigned long long)cap ? c : (unsigned long long)cap);
}

__device__ __forceinline__ bool qualifies(const PoolEntry &pe, const uint64_t *best_key, float margin)
{
    const float Smax = __uint_as_float((uint32_t)(best_key[pe.event] >> 32));
    return pe.S32 >= Smax - margin;
}

// one warp per pool entry: fp64 score of the entries within the margin of the final fp32 maximum
__global__ void __launch_bounds__(128) rescore_kernel(const BestArgs A, const PoolEntry *pool, uint32_t pool_cap,
                               const unsigned long long *counters, const uint64_t *best_key, float margin,
                               double *pool_S64, double *pool_chi2, int32_t *pool_nmatch,
                               unsigned long long *ev_maxS, ApproachRec *rec, int32_t *rec_count, int32_t *pool_slot,
                               int32_t *slot_counter)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    load_layers(A.g, s_layer);
    const uint32_t i = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;
    const int lane = threadIdx.x & 31;
    if (i >= pool_size(counters, pool_cap)) return;
    const PoolEntry pe = pool[i];
    if (!qualifies(pe, best_key, margin)) {
        if (lane == 0) { pool_S64[i] = -1.0; pool_slot[i] = -1; }
        return;
    }
    Eval64 ev;
    int slot = 0;
    if (lane == 0) slot = atomicAdd(slot_counter, 1);
    slot = __shfl_sync(0xffffffffu, slot, 0);
    const bool have = slot < kRecSlots;
    eval_seed64(A, s_layer, (int)pe.event, (int)pe.event, pe.index, ev, nullptr, nullptr, have ? rec + (size_t)slot * kRecCap : nullptr,
                have ? rec_count + slot : nullptr);
    if (lane == 0) {
        const double S = (double)ev.n_match - ev.chi2 / A.lambda;       // C10
        pool_slot[i] = have ? slot : -1;
        pool_S64[i] = S; pool_chi2[i] = ev.chi2; pool_nmatch[i] = ev.n_match;
        atomicMax(ev_maxS + pe.event, (unsigned long long)__double_as_longlong(S > 0.0 ? S : 0.0));
    }
}

// ties -> lowest linear index
__global__ void pick_kernel(const PoolEntry *pool, uint32_t pool_cap, const unsigned long long *counters,
                            const double *pool_S64, const unsigned long long *ev_maxS, unsigned long long *ev_best)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= pool_size(counters, pool_cap)) return;
    const double S = pool_S64[i];
    if (S < 0.0) return;
    const PoolEntry pe = pool[i];
    if ((unsigned long long)__double_as_longlong(S) == ev_maxS[pe.event]) atomicMin(ev_best + pe.event, (unsigned long long)pe.index);
}

// the record slot of each event's best seed (several pool entries may carry the same seed: any of them serves)
__global__ void slot_kernel(const PoolEntry *pool, uint32_t pool_cap, const unsigned long long *counters,
                            const double *pool_S64, const unsigned long long *ev_best, const int32_t *pool_slot,
                            const int32_t *rec_count, int32_t *ev_slot)
{
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= pool_size(counters, pool_cap)) return;
    if (pool_S64[i] < 0.0) return;
    const PoolEntry pe = pool[i];
    const int slot = pool_slot[i];
    if ((unsigned long long)pe.index == ev_best[pe.event] && slot >= 0 && rec_count[slot] <= kRecCap)
        atomicMax(ev_slot + pe.event, slot);
}

// one thread per event: re-propagate the best seed, label wires, report (index, n_match, chi2)
__global__ void label_kernel(const BestArgs A, int n_events, const unsigned long long *ev_best, int32_t *wire_label,
                             double *wire_best, int64_t *best_seed, uint32_t *best_n_match, double *best_chi2,
                             const PoolEntry *pool, uint32_t pool_cap, const unsigned long long *counters,
                             const double *pool_chi2, const int32_t *pool_nmatch, const int32_t *pool_slot,
                             const ApproachRec *rec, const int32_t *rec_count, const int32_t *ev_slot)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    load_layers(A.g, s_layer);
    const int e = (blockIdx.x * blockDim.x + threadIdx.x) >> 5;        // one warp per event
    const int lane = threadIdx.x & 31;
    if (e >= n_events) return;
    const unsigned long long b = ev_best[e];
    if (b == ~0ull) {                      // no candidate survived (pool overflow): report "none"
        if (lane == 0) { best_seed[e] = -1; best_n_match[e] = 0; best_chi2[e] = 0.0; }
        return;
    }
    const int slot = ev_slot[e];
    if (slot >= 0) {                       // replay the recorded matched approaches (path order) -- reading C12
        if (lane != 0) return;
        int32_t *lab = wire_label + (size_t)e * A.W;
        double *bst = wire_best + (size_t)e * A.W;
        const ApproachRec *r = rec + (size_t)slot * kRecCap;
        const int n = rec_count[slot];
        double chi2 = 0.0;
        for (int i = 0; i < n; ++i) {
            const int w = r[i].wire;
            if (lab[w] < 0 || r[i].absd < bst[w]) { lab[w] = r[i].turn; bst[w] = r[i].absd; }
        }
        // n_match / chi2 of that pool entry
        const uint32_t np = pool_size(counters, pool_cap);
        for (uint32_t i = 0; i < np; ++i)
            if (pool_slot[i] == slot) { chi2 = pool_chi2[i]; best_n_match[e] = (uint32_t)pool_nmatch[i]; break; }
        best_seed[e] = (int64_t)b; best_chi2[e] = chi2;
        return;
    }
    Eval64 ev;                             // no usable record (slot table full or list overflow): propagate again
    eval_seed64(A, s_layer, e, e, (uint32_t)b, ev, wire_label + (size_t)e * A.W, wire_best + (size_t)e * A.W, nullptr, nullptr);
    if (lane == 0) { best_seed[e] = (int64_t)b; best_n_match[e] = (uint32_t)ev.n_match; best_chi2[e] = ev.chi2; }
}

__global__ void fill_i32(int32_t *p, size_t n, int32_t v)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

__global__ void gather_labels(int32_t W, const int32_t *offsets, const int32_t *wire_id, const int32_t *wire_label,
                              int32_t *labels)
{
    const int e = blockIdx.y;
    const int i = offsets[e] + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= offsets[e + 1]) return;
    labels[i] = wire_label[(size_t)e * W + wire_id[i]];
}

}  // namespace

cudaError_t launch_best_track(const BestLaunch &L, cudaStream_t s)
{
    BestArgs A;
    A.g = L.g; A.grids = L.d_grids; A.axes = L.d_axes; A.axis_stride = L.axis_stride;
    A.drift_tab = L.d_drift_tab; A.bits = L.d_bits; A.W = L.W; A.n_bit_words = L.n_bit_words;
    A.h = L.h; A.lambda = L.window * L.window; A.eloss_h = L.eloss * L.h; A.kq = CDC_KAPPA * (double)L.charge;
    A.max_steps = L.max_steps; A.lookup_every = L.lookup_every64;
    cudaError_t e;
    if ((e = cudaMemsetAsync(L.d_ev_maxS, 0, sizeof(unsigned long long) * (size_t)L.n_events, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(L.d_ev_best, 0xFF, sizeof(unsigned long long) * (size_t)L.n_events, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(L.d_ev_slot, 0xFF, sizeof(int32_t) * (size_t)L.n_events, s)) != cudaSuccess) return e;
    if ((e = cudaMemsetAsync(L.d_slot_counter, 0, sizeof(int32_t), s)) != cudaSuccess) return e;
    // grids sized by the number of entries the pool actually holds (read back by cdc_best_track), not by its capacity
    const unsigned ne = std::max(1u, std::min(L.n_entries, L.pool_cap));
    const unsigned nb = (ne + 63) / 64;
    rescore_kernel<<<(ne + 3) / 4, 128, 0, s>>>(A, L.d_pool, L.pool_cap, L.d_counters, L.d_best_key, L.margin, L.d_pool_S64,
                                     L.d_pool_chi2, L.d_pool_nmatch, L.d_ev_maxS, L.d_rec, L.d_rec_count, L.d_pool_slot,
                                     L.d_slot_counter);
    pick_kernel<<<nb, 64, 0, s>>>(L.d_pool, L.pool_cap, L.d_counters, L.d_pool_S64, L.d_ev_maxS, L.d_ev_best);
    slot_kernel<<<nb, 64, 0, s>>>(L.d_pool, L.pool_cap, L.d_counters, L.d_pool_S64, L.d_ev_best, L.d_pool_slot,
                                  L.d_rec_count, L.d_ev_slot);
    const size_t nw = (size_t)L.n_events * L.W;
    fill_i32<<<(unsigned)((nw + 255) / 256), 256, 0, s>>>(L.d_wire_label, nw, -1);
    label_kernel<<<(L.n_events + 3) / 4, 128, 0, s>>>(A, L.n_events, L.d_ev_best, L.d_wire_label, L.d_wire_best,
                                                         L.d_best_seed, L.d_best_n_match, L.d_best_chi2, L.d_pool,
                                                         L.pool_cap, L.d_counters, L.d_pool_chi2, L.d_pool_nmatch,
                                                         L.d_pool_slot, L.d_rec, L.d_rec_count, L.d_ev_slot);
    cdc_count_launch(5);
    if (L.max_hits_per_event > 0 && L.d_labels) {
        cdc_count_launch();
        dim3 grid((unsigned)((L.max_hits_per_event + 127) / 128), (unsigned)L.n_events);
        gather_labels<<<grid, 128, 0, s>>>(L.W, L.d_offsets, L.d_wire_id, L.d_wire_label, L.d_labels);
    }
    return cudaGetLastError();
}
