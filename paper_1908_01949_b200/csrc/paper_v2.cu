// The paper's SECOND thread mapping ("kernel function separation"), re-created on sm_100a as a
// MEASURED COMPARISON POINT -- not the product path:
//   kernel 1: "each seed was delivered to each thread, and recorded the track parameters of all steps during the RKN
//             extrapolation to the end of the turn partition"  -> paper_v2_record_kernel, O(steps x seeds) memory;
//   kernel 2: "finds DCA to the wires ... same with the description in Section 2.2 [one block per seed, one thread
//             per fired wire], except that the track propagation starts from the recorded track parameter which is
//             closest to the corresponding wire"               -> paper_v2_dca_kernel.
// Here every approach of a wire is scored (reading C9: once per passage, not only the closest one), so kernel 2 walks
// the whole record of its block's seed and, where g changes sign, takes the approach between the two recorded
// vertices -- what is left of "propagating from the closest recorded parameter" when the DCA is taken on the chord of
// one step.  Same arithmetic as paper_v1.cu, so the per-seed (n_match, chi2) are bit-equal to v1's.
#include "paper_common.cuh"

namespace {

// vertex record: {x, xlo, y, ylo}, {z, Tx, Ty, Tz}; layout [vertex][seed][2] so that kernel 1's writes coalesce
template <int FIELD>
__global__ void __launch_bounds__(128) paper_v2_record_kernel(const PaperArgs A)
{
    const int s = blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= A.n_seeds) return;
    PaperState S;
    paper_seed(A, (uint32_t)A.seed_index[s], S);
    float4 *rec = A.rec + 2 * (size_t)s;
    const size_t stride = 2 * (size_t)A.n_seeds;
    rec[0] = make_float4(S.x, S.xlo, S.y, S.ylo); rec[1] = make_float4(S.z, S.Tx, S.Ty, S.Tz);
    int n = 0;
    while (n < A.max_steps) {
        paper_step<FIELD>(A, S);
        n += 1;
        rec += stride;
        rec[0] = make_float4(S.x, S.xlo, S.y, S.ylo); rec[1] = make_float4(S.z, S.Tx, S.Ty, S.Tz);
        const float rho2 = fmaf(S.x, S.x, S.y * S.y);
        if (!(fabsf(S.z) <= A.gd.z_half) || !(rho2 <= A.gd.r_out_sq) || S.low_p) break;
    }
    A.rec_steps[s] = n;
}

__global__ void __launch_bounds__(1024) paper_v2_dca_kernel(const PaperArgs A)
{
    __shared__ unsigned s_nm;
    __shared__ float s_chi2;
    if (threadIdx.x == 0) { s_nm = 0u; s_chi2 = 0.0f; }
    __syncthreads();
    const int s = blockIdx.x;
    const int steps = A.rec_steps[s];
    const size_t stride = 2 * (size_t)A.n_seeds;
    uint32_t nm = 0;
    float chi2 = 0.0f;
    for (int hit = threadIdx.x; hit < A.n_hits; hit += blockDim.x) {
        const int w = A.wire_id[hit];
        const float4 wr = __ldg(A.gd.wire4 + w);
        const float drift = A.drift[hit];
        const float4 *rec = A.rec + 2 * (size_t)s;
        float4 p = rec[0], q = rec[1];
        float ex0, ey0, eu0;
        float g = wire_g(wr, A.uz, A.inv_uz, p.x, p.y, p.z, p.w, q.x, q.y, q.z, q.w, ex0, ey0, eu0);
        bool cn = true;
        for (int n = 0; n < steps; ++n) {
            rec += stride;
            const float4 p1 = rec[0], q1 = rec[1];
            float ex1, ey1, eu1;
            const float gn = wire_g(wr, A.uz, A.inv_uz, p1.x, p1.y, p1.z, p1.w, q1.x, q1.y, q1.z, q1.w, ex1, ey1, eu1);
            if (cn && g <= 0.0f && gn > 0.0f) paper_approach(A, wr, drift, g, gn, p.x, p.y, p.z, p.w, q.x, ex1, ey1, q1.x, nm, chi2);
            g = gn;
            cn = fmaf(p1.x, p1.x, p1.z * p1.z) >= A.gd.R0sq;
            p = p1; q = q1;
        }
    }
    if (nm) { atomicAdd(&s_nm, nm); atomicAdd(&s_chi2, chi2); }
    __syncthreads();
    if (threadIdx.x == 0) { A.n_match[s] = s_nm; A.chi2[s] = s_chi2; }
}

}  // namespace

extern "C" int32_t cdc_seed_scan_paper_mapping_v2(const cdc_geometry *g, cdc_events *ev, int32_t event,
                                                  const cdc_grid_spec *h_grid, const cdc_scan_params *p,
                                                  const int64_t *d_seed_index, int32_t n_seeds, uint32_t *d_n_match,
                                                  float *d_chi2, double *h_ms2_or_null, void *stream)
{
    return cdc_guard("cdc_seed_scan_paper_mapping_v2", [&]() -> int32_t {
    cudaStream_t s = (cudaStream_t)stream;
    PaperArgs A;
    double *d_axes = nullptr;
    int32_t rc = paper_prepare("cdc_seed_scan_paper_mapping_v2", g, ev, event, h_grid, p, d_seed_index, n_seeds, d_n_match,
                               d_chi2, s, A, &d_axes);
    if (rc != CDC_OK) { if (d_axes) cudaFreeAsync(d_axes, s); return rc; }
    const size_t n_rec = 2 * (size_t)n_seeds * ((size_t)p->max_steps + 1);
    if (n_rec * sizeof(float4) > ((size_t)16 << 30)) {
        cudaFreeAsync(d_axes, s);
        CDC_FAIL(CDC_ERR_RANGE, "cdc_seed_scan_paper_mapping_v2: the step record would exceed 16 GiB (32 B x seeds x (max_steps + 1))");
    }
    cudaError_t e = cudaMallocAsync((void **)&A.rec, n_rec * sizeof(float4), s);
    if (e == cudaSuccess) e = cudaMallocAsync((void **)&A.rec_steps, sizeof(int32_t) * (size_t)n_seeds, s);
    cudaEvent_t t0 = nullptr, t1 = nullptr, t2 = nullptr;
    if (e == cudaSuccess && h_ms2_or_null) {
        if ((e = cudaEventCreate(&t0)) == cudaSuccess && (e = cudaEventCreate(&t1)) == cudaSuccess) e = cudaEventCreate(&t2);
    }
    if (e == cudaSuccess) {
        if (t0) cudaEventRecord(t0, s);
        if (g->fd.kind == 0) paper_v2_record_kernel<0><<<(n_seeds + 127) / 128, 128, 0, s>>>(A);
        else paper_v2_record_kernel<1><<<(n_seeds + 127) / 128, 128, 0, s>>>(A);
        if (t1) cudaEventRecord(t1, s);
        const int threads = std::min(1024, std::max(32, (A.n_hits + 31) / 32 * 32));
        paper_v2_dca_kernel<<<n_seeds, threads, 0, s>>>(A);
        if (t2) cudaEventRecord(t2, s);
        cdc_count_launch(2);
        e = cudaGetLastError();
    }
    if (e == cudaSuccess && h_ms2_or_null) {
        float a = 0.f, b = 0.f;
        if ((e = cudaEventSynchronize(t2)) == cudaSuccess && (e = cudaEventElapsedTime(&a, t0, t1)) == cudaSuccess)
            e = cudaEventElapsedTime(&b, t1, t2);
        h_ms2_or_null[0] = a; h_ms2_or_null[1] = b;
    }
    if (t0) cudaEventDestroy(t0);
    if (t1) cudaEventDestroy(t1);
    if (t2) cudaEventDestroy(t2);
    if (A.rec) cudaFreeAsync(A.rec, s);
    if (A.rec_steps) cudaFreeAsync(A.rec_steps, s);
    cudaFreeAsync(d_axes, s);
    CDC_CUDA(e);
    return CDC_OK;
    });
}
