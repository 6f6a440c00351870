// Shared by the two re-creations of the paper's thread mappings (paper_v1.cu: PAPER.md:73; paper_v2.cu: PAPER.md:133-135):
// the seed state, one textbook RKN step in the arithmetic of the scan kernel's stage form, and the approach test of
// one wire over one interval (reading C9).  MEASURED COMPARISON POINTS, not the product path.
#pragma once
#include <algorithm>
#include <vector>

#include "scan_common.cuh"

namespace {

struct PaperArgs {
    GeomDev gd;
    FieldDev fd;
    GridDev grid;
    const double *axes;              // [6][stride] of the event's grid
    int32_t axis_stride;
    const int32_t *wire_id;          // hits of the event
    const float *drift;
    int32_t n_hits;
    const int64_t *seed_index;       // seeds to evaluate (linear indices)
    int32_t n_seeds;
    float h, h_half, h2_8, h2_2, h_6, h2_6;
    double kq, h6_64;
    float lambda, uz, inv_uz;
    int32_t max_steps;
    uint32_t *n_match;               // [n]
    float *chi2;
    float4 *rec;                     // v2 only: [max_steps + 1][n_seeds][2] recorded vertices
    int32_t *rec_steps;              // v2 only: [n_seeds] intervals recorded
};

struct PaperState {                  // hi + lo position and direction, as the scan kernel carries them
    float x, xlo, y, ylo, z, zlo, Tx, Txlo, Ty, Tylo, Tz, Tzlo, a, epsT;
    bool low_p;
};

__device__ __forceinline__ void paper_seed(const PaperArgs &A, uint32_t q, PaperState &S)
{
    const GridDev &G = A.grid;
    const int i_pz = q % G.n[4]; q /= G.n[4];
    const int i_py = q % G.n[3]; q /= G.n[3];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_z = q % G.n[1];
    const int i_th = q / G.n[1];
    const int st = A.axis_stride;
    const double x0 = A.axes[i_th], y0 = A.axes[st + i_th], z0 = A.axes[2 * st + i_z];
    const double px = A.axes[3 * st + i_px], py = A.axes[4 * st + i_py], pz = A.axes[5 * st + i_pz];
    const double p0 = sqrt(px * px + py * py + pz * pz);
    const double tx = px / p0, ty = py / p0, tz = pz / p0;
    S.x = (float)x0; S.xlo = (float)(x0 - (double)S.x); S.y = (float)y0; S.ylo = (float)(y0 - (double)S.y);
    S.z = (float)z0; S.zlo = (float)(z0 - (double)S.z);
    S.Tx = (float)tx; S.Txlo = (float)(tx - (double)S.Tx); S.Ty = (float)ty; S.Tylo = (float)(ty - (double)S.Ty);
    S.Tz = (float)tz; S.Tzlo = (float)(tz - (double)S.Tz);
    const double a64 = A.kq / p0;
    S.a = (float)a64;
    S.epsT = (float)((a64 * A.h6_64) / ((double)S.a * (double)A.h_6) - 1.0);
    S.low_p = !((float)p0 > 1.0f);
}

// one RKN step (reading C5, stage form), compensated updates
template <int FIELD>
__device__ __forceinline__ void paper_step(const PaperArgs &A, PaperState &S)
{
    const float h = A.h, a = S.a, x = S.x, y = S.y, z = S.z, Tx = S.Tx, Ty = S.Ty, Tz = S.Tz;
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
    comp_add(S.x, S.xlo, fmaf(h, S.Txlo, dx)); comp_add(S.y, S.ylo, fmaf(h, S.Tylo, dy)); comp_add(S.z, S.zlo, fmaf(h, S.Tzlo, dz));
    comp_add(S.Tx, S.Txlo, fmaf(dTx, S.epsT, dTx)); comp_add(S.Ty, S.Tylo, fmaf(dTy, S.epsT, dTy));
    comp_add(S.Tz, S.Tzlo, fmaf(dTz, S.epsT, dTz));
}

// the approach of one wire inside the interval from vertex 0 (x0, xl0, y0, yl0, z0; g <= 0) to vertex 1 (gn > 0)
__device__ __forceinline__ void paper_approach(const PaperArgs &A, const float4 wr, float drift, float g, float gn,
                                               float x0, float xl0, float y0, float yl0, float z0, float ex1, float ey1,
                                               float z1, uint32_t &nm, float &chi2)
{
    const float zt0 = __fmul_rn(z0, A.inv_uz);
    const float e0x = __fadd_rn(__fmaf_rn(-zt0, wr.z, __fsub_rn(x0, wr.x)), xl0);
    const float e0y = __fadd_rn(__fmaf_rn(-zt0, wr.w, __fsub_rn(y0, wr.y)), yl0);
    const float tau = __fdividef(g, g - gn);
    const float ex = fmaf(tau, ex1 - e0x, e0x), ey = fmaf(tau, ey1 - e0y, e0y);
    const float eu = fmaf(ex, wr.z, ey * wr.w);
    const float D = sqrtf(fmaxf(fmaf(ex, ex, fmaf(ey, ey, -eu * eu)), 0.0f));
    const float zw = fmaf(eu, A.uz, fmaf(tau, z1 - z0, z0));
    const float resid = D - drift, r2 = resid * resid;
    if (fabsf(zw) <= A.gd.z_half && r2 < A.lambda) { nm += 1u; chi2 += r2; }
}

// host side shared by both entry points: argument checks, axis tables of the one grid, constants
inline int32_t paper_prepare(const char *who, const cdc_geometry *g, cdc_events *ev, int32_t event, const cdc_grid_spec *h_grid,
                             const cdc_scan_params *p, const int64_t *d_seed_index, int32_t n_seeds, uint32_t *d_n_match,
                             float *d_chi2, cudaStream_t s, PaperArgs &A, double **d_axes_out)
{
    const std::string w(who);
    if (!g || !ev || !h_grid || !p || !d_seed_index || !d_n_match || !d_chi2) CDC_FAIL(CDC_ERR_INVALID, w + ": null argument");
    if (event < 0 || event >= ev->n_events || n_seeds < 1) CDC_FAIL(CDC_ERR_INVALID, w + ": bad event / n_seeds");
    if (p->eloss_MeV_per_mm != 0.0) CDC_FAIL(CDC_ERR_INVALID, w + ": energy loss is not part of the comparison kernel");
    if (!(p->h_mm > 0.0) || p->max_steps < 1 || !(p->window_mm > 0.0) || (p->charge != 1 && p->charge != -1))
        CDC_FAIL(CDC_ERR_INVALID, w + ": bad scan parameters");
    // axis tables of this one grid, built exactly as cdc_seed_scan builds them (reading C4)
    int stride = 1;
    int64_t prod = 1;
    for (int a = 0; a < 5; ++a) {
        if (h_grid->n[a] < 1 || h_grid->n[a] > CDC_MAX_AXIS) CDC_FAIL(CDC_ERR_INVALID, w + ": grid n must be in [1, 4096]");
        stride = std::max(stride, h_grid->n[a]); prod *= h_grid->n[a];
    }
    if (prod > 2147483647LL) CDC_FAIL(CDC_ERR_INVALID, w + ": more than 2^31 - 1 seeds");
    std::vector<double> tab((size_t)6 * stride, 0.0);
    for (int i = 0; i < h_grid->n[0]; ++i) {
        const double th = h_grid->lo[0] + (double)i * h_grid->step[0];
        tab[i] = g->R0 * cos(th); tab[stride + i] = g->R0 * sin(th);
    }
    for (int a = 1; a < 5; ++a)
        for (int i = 0; i < h_grid->n[a]; ++i) tab[(size_t)(a + 1) * stride + i] = h_grid->lo[a] + (double)i * h_grid->step[a];
    double *d_axes = nullptr;
    CDC_CUDA(cudaMallocAsync((void **)&d_axes, sizeof(double) * tab.size(), s));
    *d_axes_out = d_axes;
    CDC_CUDA(cudaMemcpyAsync(d_axes, tab.data(), sizeof(double) * tab.size(), cudaMemcpyHostToDevice, s));
    CDC_CUDA(cudaStreamSynchronize(s));          // tab is pageable
    A.gd = g->gd; A.fd = g->fd;
    for (int a = 0; a < 5; ++a) A.grid.n[a] = h_grid->n[a];
    A.grid.n_seeds = (int32_t)prod; A.grid.out_offset = 0;
    A.axes = d_axes; A.axis_stride = stride;
    const int h0 = ev->offsets[event];
    A.n_hits = ev->offsets[event + 1] - h0;
    A.wire_id = ev->d_wire_id + h0; A.drift = ev->d_drift + h0;
    A.seed_index = d_seed_index; A.n_seeds = n_seeds;
    const double h = p->h_mm;
    A.h = (float)h; A.h_half = (float)(h / 2.0); A.h2_8 = (float)(h * h / 8.0); A.h2_2 = (float)(h * h / 2.0);
    A.h_6 = (float)(h / 6.0); A.h2_6 = (float)(h * h / 6.0);
    A.kq = CDC_KAPPA * (double)p->charge; A.h6_64 = h / 6.0;
    A.lambda = (float)(p->window_mm * p->window_mm); A.uz = g->uz; A.inv_uz = (float)(1.0 / (double)g->uz);
    A.max_steps = p->max_steps; A.n_match = d_n_match; A.chi2 = d_chi2;
    A.rec = nullptr; A.rec_steps = nullptr;
    return CDC_OK;
}

}  // namespace
