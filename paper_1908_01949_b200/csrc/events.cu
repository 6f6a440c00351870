// A1: event binning.  Hits (wire id, drift distance) -> per-event dense drift table indexed by wire
// (sentinel -1 = no hit) + per-wire hit bitmask, so that the scan's per-step lookup is O(1)
// (the hits are uploaded to GPU memory; BJ north_star: "hits binned by (layer, phi-cell)" --
// the global wire id IS (layer, cell): id = offset[layer] + cell).
#include "cdc_internal.cuh"

namespace {

__global__ void fill_f32(float *p, size_t n, float v)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) p[i] = v;
}

__global__ void bin_hits(int32_t W, int32_t n_bit_words, const int32_t *offsets, const int32_t *wire_id,
                         const float *drift, float *drift_tab, uint32_t *bits, int32_t *err)
{
    const int e = blockIdx.y;
    const int i = offsets[e] + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= offsets[e + 1]) return;
    const int w = wire_id[i];
    const float d = drift[i];
    if (w < 0 || w >= W) { atomicOr(err, 1); return; }
    if (!(d >= 0.0f) || !(d <= 8.0f)) { atomicOr(err, 2); return; }     // 0 <= drift <= 8 mm (cell half-width; BJ configs[0])
    const uint32_t bit = 1u << (w & 31);
    const uint32_t old = atomicOr(bits + (size_t)e * n_bit_words + (w >> 5), bit);
    if (old & bit) { atomicOr(err, 4); return; }     // duplicate wire id within the event
    drift_tab[(size_t)e * W + w] = d;
}

}  // namespace

cudaError_t launch_bin_events(int32_t n_events, int32_t W, int32_t n_bit_words, int32_t max_hits_per_event,
                              const int32_t *d_offsets, const int32_t *d_wire_id, const float *d_drift,
                              float *d_drift_tab, uint32_t *d_bits, int32_t *d_err, cudaStream_t s)
{
    const size_t n_tab = (size_t)n_events * W;
    cudaError_t e = cudaMemsetAsync(d_bits, 0, (size_t)n_events * n_bit_words * sizeof(uint32_t), s);
    if (e != cudaSuccess) return e;
    e = cudaMemsetAsync(d_err, 0, sizeof(int32_t), s);
    if (e != cudaSuccess) return e;
    fill_f32<<<(unsigned)((n_tab + 255) / 256), 256, 0, s>>>(d_drift_tab, n_tab, -1.0f);
    cdc_count_launch();
    if (max_hits_per_event > 0) {
        dim3 grid((unsigned)((max_hits_per_event + 127) / 128), (unsigned)n_events);
        bin_hits<<<grid, 128, 0, s>>>(W, n_bit_words, d_offsets, d_wire_id, d_drift, d_drift_tab, d_bits, d_err);
        cdc_count_launch();
    }
    return cudaGetLastError();
}
