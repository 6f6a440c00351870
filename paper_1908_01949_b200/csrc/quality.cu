// Classification efficiency and purity per turn partition (Eq. (2), (3)) and the number of hits two
// scans found in common, N_c.  Integer counting with shared-memory atomics, one block per event; the two
// ratios are the only floating-point operations (fp64, one division each).
#include "cdc_internal.cuh"

namespace {

constexpr int kMaxTurns = 8;

__global__ void __launch_bounds__(256) quality_kernel(int n_turns, const int32_t *offsets, const int32_t *labels,
                                                      const int32_t *truth, int32_t *confusion, int32_t *c_true,
                                                      int32_t *noise_into, double *eff, double *pur)
{
    __shared__ int s_C[kMaxTurns * kMaxTurns], s_true[kMaxTurns], s_noise[kMaxTurns];
    const int e = blockIdx.x;
    for (int i = threadIdx.x; i < kMaxTurns * kMaxTurns; i += blockDim.x) s_C[i] = 0;
    if (threadIdx.x < kMaxTurns) { s_true[threadIdx.x] = 0; s_noise[threadIdx.x] = 0; }
    __syncthreads();
    for (int i = offsets[e] + threadIdx.x; i < offsets[e + 1]; i += blockDim.x) {
        const int lab = labels[i], tr = truth[i];
        if (tr >= 0 && tr < n_turns) {
            atomicAdd(&s_true[tr], 1);
            if (lab >= 0 && lab < n_turns) atomicAdd(&s_C[tr * kMaxTurns + lab], 1);      // C_{tr -> lab}
        } else if (lab >= 0 && lab < n_turns) {
            atomicAdd(&s_noise[lab], 1);
        }
    }
    __syncthreads();
    for (int i = threadIdx.x; i < n_turns * n_turns; i += blockDim.x)
        confusion[(size_t)e * n_turns * n_turns + i] = s_C[(i / n_turns) * kMaxTurns + i % n_turns];
    if (threadIdx.x < n_turns) {
        const int k = threadIdx.x;
        int den = 0;
        for (int i = 0; i < n_turns; ++i) den += s_C[i * kMaxTurns + k];
        c_true[(size_t)e * n_turns + k] = s_true[k];
        noise_into[(size_t)e * n_turns + k] = s_noise[k];
        eff[(size_t)e * n_turns + k] = s_true[k] ? (double)s_C[k * kMaxTurns + k] / (double)s_true[k] : -1.0;   // Eq. (2)
        pur[(size_t)e * n_turns + k] = den ? (double)s_C[k * kMaxTurns + k] / (double)den : -1.0;               // Eq. (3)
    }
}

__global__ void __launch_bounds__(256) common_kernel(const int32_t *offsets, const int32_t *la, const int32_t *lb, int ta, int tb,
                                                     int32_t *n_common)
{
    const int e = blockIdx.x;
    int c = 0;
    for (int i = offsets[e] + threadIdx.x; i < offsets[e + 1]; i += blockDim.x) c += ((ta < 0 ? la[i] >= 0 : la[i] == ta) && (tb < 0 ? lb[i] >= 0 : lb[i] == tb)) ? 1 : 0;
    c = __reduce_add_sync(0xffffffffu, c);
    __shared__ int s[8];
    if ((threadIdx.x & 31) == 0) s[threadIdx.x >> 5] = c;
    __syncthreads();
    if (threadIdx.x == 0) {
        int t = 0;
        for (int w = 0; w < 8; ++w) t += s[w];
        n_common[e] = t;
    }
}

}  // namespace

extern "C" int32_t cdc_classification_quality(const cdc_events *ev, int32_t n_turns, const int32_t *d_labels,
                                              const int32_t *d_truth_turn, int32_t *d_confusion, int32_t *d_c_true,
                                              int32_t *d_noise_into, double *d_efficiency, double *d_purity, void *stream)
{
    return cdc_guard("cdc_classification_quality", [&]() -> int32_t {
    if (!ev || !d_labels || !d_truth_turn || !d_confusion || !d_c_true || !d_noise_into || !d_efficiency || !d_purity)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_classification_quality: null argument");
    if (n_turns < 1 || n_turns > kMaxTurns) CDC_FAIL(CDC_ERR_INVALID, "cdc_classification_quality: n_turns must be in [1, 8]");
    quality_kernel<<<ev->n_events, 256, 0, (cudaStream_t)stream>>>(n_turns, ev->d_offsets, d_labels, d_truth_turn, d_confusion,
                                                                   d_c_true, d_noise_into, d_efficiency, d_purity);
    cdc_count_launch();
    CDC_CUDA(cudaGetLastError());
    return CDC_OK;
    });
}

extern "C" int32_t cdc_common_hits(const cdc_events *ev, const int32_t *d_labels_a, const int32_t *d_labels_b,
                                   int32_t turn_a, int32_t turn_b, int32_t *d_n_common, void *stream)
{
    return cdc_guard("cdc_common_hits", [&]() -> int32_t {
    if (!ev || !d_labels_a || !d_labels_b || !d_n_common) CDC_FAIL(CDC_ERR_INVALID, "cdc_common_hits: null argument");
    common_kernel<<<ev->n_events, 256, 0, (cudaStream_t)stream>>>(ev->d_offsets, d_labels_a, d_labels_b, turn_a, turn_b, d_n_common);
    cdc_count_launch();
    CDC_CUDA(cudaGetLastError());
    return CDC_OK;
    });
}
