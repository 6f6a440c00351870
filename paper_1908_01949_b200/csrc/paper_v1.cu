// The paper's own thread mapping (v1, Fig. 6), re-created on sm_100a as a MEASURED COMPARISON POINT
// -- not the product path: "each tracking seed is delivered to each block, and each thread in a block
// calculates the DCA for each wire ... the number of blocks to be launched in the GPU is same with the number of
// scanning seeds, and the number of threads in a block is same with the number of the fired wires".
// Every thread therefore repeats the whole RKN propagation of its block's seed and watches ONE fired wire; the block
// sums min(d^2, lambda) terms.  Same arithmetic as the scan kernel (scan_common.cuh), same scoring rule (reading C9),
// so the per-seed (n_match, chi2) must equal the product's; what differs is only who computes what.
#include "paper_common.cuh"

namespace {

template <int FIELD>
__global__ void __launch_bounds__(1024) paper_v1_kernel(const PaperArgs A)
{
    __shared__ unsigned s_nm;
    __shared__ float s_chi2;
    if (threadIdx.x == 0) { s_nm = 0u; s_chi2 = 0.0f; }
    __syncthreads();
    PaperState S0;
    paper_seed(A, (uint32_t)A.seed_index[blockIdx.x], S0);
    uint32_t nm = 0;
    float chi2 = 0.0f;
    // this thread's fired wires: hit threadIdx.x, threadIdx.x + blockDim.x, ... (one each unless > 1024 hits)
    for (int hit = threadIdx.x; hit < A.n_hits; hit += blockDim.x) {
        const int w = A.wire_id[hit];
        const float4 wr = __ldg(A.gd.wire4 + w);
        const float drift = A.drift[hit];
        PaperState S = S0;
        float ex0, ey0, eu0;
        float g = wire_g(wr, A.uz, A.inv_uz, S.x, S.xlo, S.y, S.ylo, S.z, S.Tx, S.Ty, S.Tz, ex0, ey0, eu0);
        bool cn = true;
        for (int n = 0; n < A.max_steps; ++n) {
            const float x0 = S.x, xl0 = S.xlo, y0 = S.y, yl0 = S.ylo, z0 = S.z;
            paper_step<FIELD>(A, S);
            float ex1, ey1, eu1;
            const float gn = wire_g(wr, A.uz, A.inv_uz, S.x, S.xlo, S.y, S.ylo, S.z, S.Tx, S.Ty, S.Tz, ex1, ey1, eu1);
            if (cn && g <= 0.0f && gn > 0.0f) paper_approach(A, wr, drift, g, gn, x0, xl0, y0, yl0, z0, ex1, ey1, S.z, nm, chi2);
            g = gn;
            const float rho2 = fmaf(S.x, S.x, S.y * S.y);
            cn = rho2 >= A.gd.R0sq;
            if (!(fabsf(S.z) <= A.gd.z_half) || !(rho2 <= A.gd.r_out_sq) || S.low_p) break;
        }
    }
    if (nm) { atomicAdd(&s_nm, nm); atomicAdd(&s_chi2, chi2); }
    __syncthreads();
    if (threadIdx.x == 0) { A.n_match[blockIdx.x] = s_nm; A.chi2[blockIdx.x] = s_chi2; }
}

}  // namespace

extern "C" int32_t cdc_seed_scan_paper_mapping(const cdc_geometry *g, cdc_events *ev, int32_t event, const cdc_grid_spec *h_grid,
                                               const cdc_scan_params *p, const int64_t *d_seed_index, int32_t n_seeds,
                                               uint32_t *d_n_match, float *d_chi2, void *stream)
{
    return cdc_guard("cdc_seed_scan_paper_mapping", [&]() -> int32_t {
    cudaStream_t s = (cudaStream_t)stream;
    PaperArgs A;
    double *d_axes = nullptr;
    const int32_t rc = paper_prepare("cdc_seed_scan_paper_mapping", g, ev, event, h_grid, p, d_seed_index, n_seeds, d_n_match,
                                     d_chi2, s, A, &d_axes);
    if (rc != CDC_OK) { if (d_axes) cudaFreeAsync(d_axes, s); return rc; }
    const int threads = std::min(1024, std::max(32, (A.n_hits + 31) / 32 * 32));     // "threads in a block = fired wires"
    if (g->fd.kind == 0) paper_v1_kernel<0><<<n_seeds, threads, 0, s>>>(A);
    else paper_v1_kernel<1><<<n_seeds, threads, 0, s>>>(A);
    cdc_count_launch();
    const cudaError_t e = cudaGetLastError();
    cudaFreeAsync(d_axes, s);
    CDC_CUDA(e);
    return CDC_OK;
    });
}
