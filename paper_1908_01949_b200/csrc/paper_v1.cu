// The paper's own thread mapping (v1, Fig. 6), re-created on sm_100a as a MEASURED COMPARISON POINT
// -- not the product path: "each tracking seed is delivered to each block, and each thread in a block
// calculates the DCA for each wire ... the number of blocks to be launched in the GPU is same with the number of
// scanning seeds, and the number of threads in a block is same with the number of the fired wires".
// Every thread therefore repeats the whole RKN propagation of its block's seed and watches ONE fired wire; the block
// sums min(d^2, lambda) terms.  Same arithmetic as the scan kernel (scan_common.cuh), same scoring rule (reading C9),
// so the per-seed (n_match, chi2) must equal the product's; what differs is only who computes what.
#include "scan_common.cuh"

namespace {

struct V1Args {
    GeomDev gd;
    FieldDev fd;
    GridDev grid;
    const double *axes;              // [6][stride] of the event's grid
    int32_t axis_stride;
    const int32_t *wire_id;          // hits of the event
    const float *drift;
    int32_t n_hits;
    const int64_t *seed_index;       // seeds to evaluate (linear indices), one block each
    float h, h_half, h2_8, h2_2, h_6, h2_6;
    double kq, h6_64;
    float lambda, uz, inv_uz;
    int32_t max_steps;
    uint32_t *n_match;               // [n]
    float *chi2;
};

template <int FIELD>
__global__ void __launch_bounds__(1024) paper_v1_kernel(const V1Args A)
{
    __shared__ unsigned s_nm;
    __shared__ float s_chi2;
    if (threadIdx.x == 0) { s_nm = 0u; s_chi2 = 0.0f; }
    __syncthreads();
    uint32_t q = (uint32_t)A.seed_index[blockIdx.x];
    const GridDev &G = A.grid;
    const int i_pz = q % G.n[4]; q /= G.n[4];
    const int i_py = q % G.n[3]; q /= G.n[3];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_z = q % G.n[1];
    const int i_th = q / G.n[1];
    float xh, xl, yh, yl, zh, zl, Txh, Txl, Tyh, Tyl, Tzh, Tzl, a, epsT;
    bool low_p;
    {
        const int st = A.axis_stride;
        const double x0 = A.axes[i_th], y0 = A.axes[st + i_th], z0 = A.axes[2 * st + i_z];
        const double px = A.axes[3 * st + i_px], py = A.axes[4 * st + i_py], pz = A.axes[5 * st + i_pz];
        const double p0 = sqrt(px * px + py * py + pz * pz);
        const double tx = px / p0, ty = py / p0, tz = pz / p0;
        xh = (float)x0; xl = (float)(x0 - (double)xh); yh = (float)y0; yl = (float)(y0 - (double)yh);
        zh = (float)z0; zl = (float)(z0 - (double)zh);
        Txh = (float)tx; Txl = (float)(tx - (double)Txh); Tyh = (float)ty; Tyl = (float)(ty - (double)Tyh);
        Tzh = (float)tz; Tzl = (float)(tz - (double)Tzh);
        const double a64 = A.kq / p0;
        a = (float)a64;
        epsT = (float)((a64 * A.h6_64) / ((double)a * (double)A.h_6) - 1.0);
        low_p = !((float)p0 > 1.0f);
    }
    uint32_t nm = 0;
    float chi2 = 0.0f;
    const float h = A.h;
    // this thread's fired wires: hit threadIdx.x, threadIdx.x + blockDim.x, ... (one each unless > 1024 hits)
    for (int hit = threadIdx.x; hit < A.n_hits; hit += blockDim.x) {
        const int w = A.wire_id[hit];
        const float4 wr = __ldg(A.gd.wire4 + w);
        const float drift = A.drift[hit];
        float x = xh, xlo = xl, y = yh, ylo = yl, z = zh, zlo = zl, Tx = Txh, Txlo = Txl, Ty = Tyh, Tylo = Tyl, Tz = Tzh, Tzlo = Tzl;
        float ex0, ey0, eu0;
        float g = wire_g(wr, A.uz, A.inv_uz, x, xlo, y, ylo, z, Tx, Ty, Tz, ex0, ey0, eu0);
        bool cn = true;
        for (int n = 0; n < A.max_steps; ++n) {
            const float x0 = x, xl0 = xlo, y0 = y, yl0 = ylo, z0 = z;
            float Bx, By, Bz;
            field_at<FIELD>(A.fd, x, y, z, Bx, By, Bz);
            const float k1x = a * fmaf(Ty, Bz, -Tz * By), k1y = a * fmaf(Tz, Bx, -Tx * Bz), k1z = a * fmaf(Tx, By, -Ty * Bx);
            float Ux = fmaf(A.h_half, k1x, Tx), Uy = fmaf(A.h_half, k1y, Ty), Uz = fmaf(A.h_half, k1z, Tz);
            if (FIELD != 0)
                field_at<FIELD>(A.fd, fmaf(A.h2_8, k1x, fmaf(A.h_half, Tx, x)), fmaf(A.h2_8, k1y, fmaf(A.h_half, Ty, y)),
                                fmaf(A.h2_8, k1z, fmaf(A.h_half, Tz, z)), Bx, By, Bz);
            const float k2x = a * fmaf(Uy, Bz, -Uz * By), k2y = a * fmaf(Uz, Bx, -Ux * Bz), k2z = a * fmaf(Ux, By, -Uy * Bx);
            Ux = fmaf(A.h_half, k2x, Tx); Uy = fmaf(A.h_half, k2y, Ty); Uz = fmaf(A.h_half, k2z, Tz);
            const float k3x = a * fmaf(Uy, Bz, -Uz * By), k3y = a * fmaf(Uz, Bx, -Ux * Bz), k3z = a * fmaf(Ux, By, -Uy * Bx);
            Ux = fmaf(h, k3x, Tx); Uy = fmaf(h, k3y, Ty); Uz = fmaf(h, k3z, Tz);
            if (FIELD != 0)
                field_at<FIELD>(A.fd, fmaf(A.h2_2, k3x, fmaf(h, Tx, x)), fmaf(A.h2_2, k3y, fmaf(h, Ty, y)),
                                fmaf(A.h2_2, k3z, fmaf(h, Tz, z)), Bx, By, Bz);
            const float k4x = a * fmaf(Uy, Bz, -Uz * By), k4y = a * fmaf(Uz, Bx, -Ux * Bz), k4z = a * fmaf(Ux, By, -Uy * Bx);
            const float dx = fmaf(A.h2_6, (k1x + k2x) + k3x, h * Tx), dy = fmaf(A.h2_6, (k1y + k2y) + k3y, h * Ty);
            const float dz = fmaf(A.h2_6, (k1z + k2z) + k3z, h * Tz);
            const float dTx = A.h_6 * fmaf(2.0f, k2x + k3x, k1x + k4x), dTy = A.h_6 * fmaf(2.0f, k2y + k3y, k1y + k4y);
            const float dTz = A.h_6 * fmaf(2.0f, k2z + k3z, k1z + k4z);
            comp_add(x, xlo, fmaf(h, Txlo, dx)); comp_add(y, ylo, fmaf(h, Tylo, dy)); comp_add(z, zlo, fmaf(h, Tzlo, dz));
            comp_add(Tx, Txlo, fmaf(dTx, epsT, dTx)); comp_add(Ty, Tylo, fmaf(dTy, epsT, dTy));
            comp_add(Tz, Tzlo, fmaf(dTz, epsT, dTz));
            float ex1, ey1, eu1;
            const float gn = wire_g(wr, A.uz, A.inv_uz, x, xlo, y, ylo, z, Tx, Ty, Tz, ex1, ey1, eu1);
            if (cn && g <= 0.0f && gn > 0.0f) {
                const float zt0 = __fmul_rn(z0, A.inv_uz);
                const float e0x = __fadd_rn(__fmaf_rn(-zt0, wr.z, __fsub_rn(x0, wr.x)), xl0);
                const float e0y = __fadd_rn(__fmaf_rn(-zt0, wr.w, __fsub_rn(y0, wr.y)), yl0);
                const float tau = __fdividef(g, g - gn);
                const float ex = fmaf(tau, ex1 - e0x, e0x), ey = fmaf(tau, ey1 - e0y, e0y);
                const float eu = fmaf(ex, wr.z, ey * wr.w);
                const float D = sqrtf(fmaxf(fmaf(ex, ex, fmaf(ey, ey, -eu * eu)), 0.0f));
                const float zw = fmaf(eu, A.uz, fmaf(tau, z - z0, z0));
                const float resid = D - drift, r2 = resid * resid;
                if (fabsf(zw) <= A.gd.z_half && r2 < A.lambda) { nm += 1u; chi2 += r2; }
            }
            g = gn;
            const float rho2 = fmaf(x, x, y * y);
            cn = rho2 >= A.gd.R0sq;
            if (!(fabsf(z) <= A.gd.z_half) || !(rho2 <= A.gd.r_out_sq) || low_p) break;
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
    if (!g || !ev || !h_grid || !p || !d_seed_index || !d_n_match || !d_chi2)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_paper_mapping: null argument");
    if (event < 0 || event >= ev->n_events || n_seeds < 1) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_paper_mapping: bad event / n_seeds");
    if (p->eloss_MeV_per_mm != 0.0) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_paper_mapping: energy loss is not part of the comparison kernel");
    cudaStream_t s = (cudaStream_t)stream;
    // axis tables of this one grid, built exactly as cdc_seed_scan builds them (reading C4)
    int stride = 1;
    int64_t prod = 1;
    for (int a = 0; a < 5; ++a) {
        if (h_grid->n[a] < 1 || h_grid->n[a] > CDC_MAX_AXIS) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_paper_mapping: grid n must be in [1, 4096]");
        stride = std::max(stride, h_grid->n[a]); prod *= h_grid->n[a];
    }
    if (prod > 2147483647LL) CDC_FAIL(CDC_ERR_INVALID, "cdc_seed_scan_paper_mapping: more than 2^31 - 1 seeds");
    std::vector<double> tab((size_t)6 * stride, 0.0);
    for (int i = 0; i < h_grid->n[0]; ++i) {
        const double th = h_grid->lo[0] + (double)i * h_grid->step[0];
        tab[i] = g->R0 * cos(th); tab[stride + i] = g->R0 * sin(th);
    }
    for (int a = 1; a < 5; ++a)
        for (int i = 0; i < h_grid->n[a]; ++i) tab[(size_t)(a + 1) * stride + i] = h_grid->lo[a] + (double)i * h_grid->step[a];
    double *d_axes = nullptr;
    CDC_CUDA(cudaMallocAsync((void **)&d_axes, sizeof(double) * tab.size(), s));
    CDC_CUDA(cudaMemcpyAsync(d_axes, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice, s));
    CDC_CUDA(cudaStreamSynchronize(s));          // tab is pageable
    V1Args A;
    A.gd = g->gd; A.fd = g->fd;
    for (int a = 0; a < 5; ++a) A.grid.n[a] = h_grid->n[a];
    A.grid.n_seeds = (int32_t)prod; A.grid.out_offset = 0;
    A.axes = d_axes; A.axis_stride = stride;
    const int h0 = ev->offsets[event];
    A.n_hits = ev->offsets[event + 1] - h0;
    A.wire_id = ev->d_wire_id + h0; A.drift = ev->d_drift + h0;
    A.seed_index = d_seed_index;
    const double h = p->h_mm;
    A.h = (float)h; A.h_half = (float)(h / 2.0); A.h2_8 = (float)(h * h / 8.0); A.h2_2 = (float)(h * h / 2.0);
    A.h_6 = (float)(h / 6.0); A.h2_6 = (float)(h * h / 6.0);
    A.kq = CDC_KAPPA * (double)p->charge; A.h6_64 = h / 6.0;
    A.lambda = (float)(p->window_mm * p->window_mm); A.uz = g->uz; A.inv_uz = (float)(1.0 / (double)g->uz);
    A.max_steps = p->max_steps; A.n_match = d_n_match; A.chi2 = d_chi2;
    const int threads = std::min(1024, std::max(32, (A.n_hits + 31) / 32 * 32));     // "threads in a block = fired wires"
    if (g->fd.kind == 0) paper_v1_kernel<0><<<n_seeds, threads, 0, s>>>(A);
    else paper_v1_kernel<1><<<n_seeds, threads, 0, s>>>(A);
    cdc_count_launch();
    CDC_CUDA(cudaGetLastError());
    CDC_CUDA(cudaFreeAsync(d_axes, s));
    return CDC_OK;
}
