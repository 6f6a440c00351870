// Host side of the C ABI (include/cdc_seedscan.h): handles, validation, table building (A0, A3 axis tables)
// and kernel launches.  No arithmetic of the method runs here except the one-off fp64 table construction.
#include <math.h>
#include <string.h>

#include <algorithm>
#include <atomic>
#include <new>

#include "cdc_internal.cuh"

static thread_local std::string g_last_error;
void cdc_set_error(const std::string &msg) { g_last_error = msg; }

extern "C" const char *cdc_last_error(void) { return g_last_error.c_str(); }

static std::atomic<uint64_t> g_launches{0};
void cdc_count_launch(int n) { g_launches.fetch_add((uint64_t)n, std::memory_order_relaxed); }
extern "C" uint64_t cdc_kernel_launch_count(void) { return g_launches.load(std::memory_order_relaxed); }

namespace {

constexpr double kLookupReach = 9.5;     // mm: wires farther than this from a step vertex cannot own a match (C8)
constexpr double kFieldMargin = 8.0;     // mm: stage points reach at most 2 h_max beyond the exit surfaces

template <typename T>
cudaError_t dev_alloc(T **p, size_t n)
{
    *p = nullptr;
    return cudaMalloc((void **)p, std::max<size_t>(n, 1) * sizeof(T));
}

void free_geometry(cdc_geometry *g)
{
    if (!g) return;
    cudaFree(g->d_wire4); cudaFree(g->d_wire5); cudaFree(g->d_field); cudaFree(g->d_cells); cudaFree(g->d_layers);
    delete g;
}

}  // namespace

// ------------------------------------------------------------------------------------------------ A0
extern "C" int32_t cdc_geometry_create(const cdc_geometry_desc *gd, const cdc_field_desc *fd, cdc_geometry **out)
{
    return cdc_guard("cdc_geometry_create", [&]() -> int32_t {
    if (!gd || !fd || !out) CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: null argument");
    *out = nullptr;
    const int L = gd->n_layers;
    if (L < 1 || L > CDC_MAX_LAYERS) CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: n_layers must be in [1, 32]");
    if (!gd->r_mm || !gd->n_wires || !gd->phi0_rad || !gd->stereo_rad)
        CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: null layer array");
    if (!(gd->z_half_mm > 0) || !(gd->R0_mm > 0) || !(gd->r_out_mm > gd->R0_mm))
        CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: need z_half > 0, 0 < R0 < r_out");
    cdc_geometry *g = new (std::nothrow) cdc_geometry;
    if (!g) CDC_FAIL(CDC_ERR_NOMEM, "cdc_geometry_create: host allocation failed");
    g->n_layers = L;
    g->r.assign(gd->r_mm, gd->r_mm + L);
    g->phi0.assign(gd->phi0_rad, gd->phi0_rad + L);
    g->stereo.assign(gd->stereo_rad, gd->stereo_rad + L);
    g->n_wires.assign(gd->n_wires, gd->n_wires + L);
    g->offset.assign(L + 1, 0);
    for (int j = 0; j < L; ++j) {
        if (g->n_wires[j] < 3) { delete g; CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: a layer needs >= 3 wires"); }
        g->offset[j + 1] = g->offset[j] + g->n_wires[j];
    }
    g->W = g->offset[L];
    if (g->W > 8192) { delete g; CDC_FAIL(CDC_ERR_RANGE, "cdc_geometry_create: more than 8192 wires"); }
    g->z_half = gd->z_half_mm; g->R0 = gd->R0_mm; g->r_out = gd->r_out_mm;
    // the O(1) layer lookup needs equally spaced layers and one |tan(stereo)|
    const double pitch = L > 1 ? (g->r[L - 1] - g->r[0]) / (L - 1) : 16.5;
    const double tan_abs = fabs(tan(g->stereo[0]));
    for (int j = 0; j < L; ++j) {
        if (fabs(g->r[j] - (g->r[0] + pitch * j)) > 1e-6 * pitch || !(pitch > 0) ||
            fabs(fabs(tan(g->stereo[j])) - tan_abs) > 1e-9) {
            delete g;
            CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: layers must be equally spaced with equal |stereo|");
        }
    }
    if (L > 1 && pitch < 2.0 * kLookupReach - 3.0) {
        delete g;
        CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: layer pitch too small for the two-layer lookup");
    }
    // per-wire table: canonical fp32 [W][5], given or built in fp64 and rounded once (reading C2)
    g->wire5.resize((size_t)g->W * 5);
    if (gd->h_wire) {
        memcpy(g->wire5.data(), gd->h_wire, sizeof(float) * 5 * (size_t)g->W);
    } else {
        for (int j = 0; j < L; ++j) {
            const double se = sin(g->stereo[j]), ce = cos(g->stereo[j]);
            for (int k = 0; k < g->n_wires[j]; ++k) {
                const double phi = g->phi0[j] + 2.0 * M_PI * (double)k / (double)g->n_wires[j];
                float *w = g->wire5.data() + 5 * (size_t)(g->offset[j] + k);
                w[0] = (float)(g->r[j] * cos(phi)); w[1] = (float)(g->r[j] * sin(phi));
                w[2] = (float)(-se * sin(phi));     w[3] = (float)(se * cos(phi));
                w[4] = (float)ce;
            }
        }
    }
    // one cos(eps) for every wire (equal |stereo|); the scan kernel folds it into constants
    g->uz = g->wire5[4];
    for (int w = 0; w < g->W; ++w)
        if (g->wire5[5 * (size_t)w + 4] != g->uz) {
            delete g;
            CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: wire table must carry one u_z (equal |stereo|)");
        }
    // a wire outside the 2 x 2 candidate set of a vertex is at least `excl` away from it (reading C8): one layer
    // pitch radially, or one cell along the arc at the smallest radius a candidate can be looked up from
    g->pitch = pitch;
    g->excl = pitch;
    for (int j = 0; j < L; ++j)
        g->excl = std::min(g->excl, 2.0 * M_PI * (g->r[j] - pitch) / (double)g->n_wires[j]);
    g->excl = 0.9975 * g->excl - 0.2;
    {
        const double ze = g->z_half * tan_abs;
        g->cell_max = 0.0;
        for (int j = 0; j < L; ++j)
            g->cell_max = std::max(g->cell_max, 2.0 * M_PI * (sqrt(g->r[j] * g->r[j] + ze * ze) + pitch) / (double)g->n_wires[j]);
    }
    // field
    g->field = *fd;
    if (fd->kind == 1) {
        if (!fd->h_br_bz || fd->nr < 2 || fd->nz < 2 || !(fd->dr_mm > 0) || !(fd->dz_mm > 0)) {
            delete g;
            CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: bad field table description");
        }
        const double r_hi = fd->r0_mm + fd->dr_mm * (fd->nr - 1), z_hi = fd->z0_mm + fd->dz_mm * (fd->nz - 1);
        if (fd->r0_mm > 0.0 || r_hi < g->r_out + kFieldMargin || fd->z0_mm > -(g->z_half + kFieldMargin) ||
            z_hi < g->z_half + kFieldMargin) {
            delete g;
            CDC_FAIL(CDC_ERR_RANGE, "cdc_geometry_create: field table does not cover rho <= r_out + 8, |z| <= z_half + 8");
        }
        g->field_tab.assign(fd->h_br_bz, fd->h_br_bz + (size_t)fd->nr * fd->nz * 2);
        for (size_t i = 0; i < (size_t)fd->nr * fd->nz; ++i)
            g->b_max = std::max(g->b_max, hypot((double)fd->h_br_bz[2 * i], (double)fd->h_br_bz[2 * i + 1]));
        g->field.h_br_bz = g->field_tab.data();
    } else if (fd->kind == 0) {
        g->b_max = fabs(fd->bz_T);
    } else {
        delete g;
        CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_create: field kind must be 0 or 1");
    }

    // ---- device tables
    std::vector<float4> w4(g->W);
    for (int w = 0; w < g->W; ++w)
        w4[w] = make_float4(g->wire5[5 * w], g->wire5[5 * w + 1], g->wire5[5 * w + 2], g->wire5[5 * w + 3]);
    std::vector<LayerDev> lay(L);
    for (int j = 0; j < L; ++j) {
        LayerDev &d = lay[j];
        const double sgn = g->stereo[j] >= 0 ? 1.0 : -1.0;
        d.r = (float)g->r[j];
        d.shift_k = (float)(sgn * tan_abs / g->r[j]);
        double p0 = fmod(g->phi0[j], 2.0 * M_PI);
        if (p0 > M_PI) p0 -= 2.0 * M_PI;
        if (p0 <= -M_PI) p0 += 2.0 * M_PI;
        d.phi0 = (float)p0;
        d.kscale = (float)((double)g->n_wires[j] / (2.0 * M_PI));
        d.uz = g->wire5[5 * (size_t)g->offset[j] + 4];
        d.inv_uz = (float)(1.0 / (double)d.uz);
        d.n = g->n_wires[j];
        d.offset = g->offset[j];
    }
#define G_CUDA(expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { free_geometry(g); \
    cdc_set_error(std::string(#expr) + ": " + cudaGetErrorString(e_)); \
    return e_ == cudaErrorMemoryAllocation ? CDC_ERR_NOMEM : CDC_ERR_CUDA; } } while (0)
    G_CUDA(dev_alloc(&g->d_wire4, (size_t)g->W));
    G_CUDA(dev_alloc(&g->d_wire5, (size_t)g->W * 5));
    G_CUDA(dev_alloc(&g->d_layers, (size_t)L));
    G_CUDA(cudaMemcpy(g->d_wire4, w4.data(), sizeof(float4) * g->W, cudaMemcpyHostToDevice));
    G_CUDA(cudaMemcpy(g->d_wire5, g->wire5.data(), sizeof(float) * 5 * g->W, cudaMemcpyHostToDevice));
    G_CUDA(cudaMemcpy(g->d_layers, lay.data(), sizeof(LayerDev) * L, cudaMemcpyHostToDevice));
    if (fd->kind == 1) {
        G_CUDA(dev_alloc(&g->d_field, (size_t)fd->nr * fd->nz));
        G_CUDA(cudaMemcpy(g->d_field, g->field_tab.data(), sizeof(float2) * (size_t)fd->nr * fd->nz, cudaMemcpyHostToDevice));
        // per-cell bilinear coefficients for the fp32 scan, taken about the CELL CENTRE:
        //   B(wr, wz) = c0 + c_r wr + c_z wz + c_rz wr wz,  wr, wz in [-1/2, 1/2] = offset from the centre in cell units
        // (combinations of the fp32 node values formed in fp64, rounded once), stored as (c0, c_z, c_r, c_rz): the two
        // register pairs of one 128-bit load are then the operands of ONE packed FMA, (c0, c_z) + wr (c_r, c_rz).
        // Cell (ir, iz) is record ir (nz - 1) + iz: z runs fastest, because the 32 tracks of a warp differ in z0 first
        // (same rho, a spread of z): their cells are then neighbours in memory and one gather touches 2-3 lines
        // instead of one line per track (the L1 data pipe was 70 % busy with [iz][ir], ncu r2)
        const int ncr = fd->nr - 1, ncz = fd->nz - 1;
        std::vector<float4> cells((size_t)ncr * ncz * 2);
        for (int iz = 0; iz < ncz; ++iz)
            for (int ir = 0; ir < ncr; ++ir)
                for (int c = 0; c < 2; ++c) {
                    const double n00 = g->field_tab[((size_t)iz * fd->nr + ir) * 2 + c];
                    const double n01 = g->field_tab[((size_t)iz * fd->nr + ir + 1) * 2 + c];
                    const double n10 = g->field_tab[((size_t)(iz + 1) * fd->nr + ir) * 2 + c];
                    const double n11 = g->field_tab[((size_t)(iz + 1) * fd->nr + ir + 1) * 2 + c];
                    const double crz = n11 - n10 - n01 + n00;
                    cells[((size_t)ir * ncz + iz) * 2 + c] =
                        make_float4((float)(0.25 * (n00 + n01 + n10 + n11)), (float)((n10 - n00) + 0.5 * crz),
                                    (float)((n01 - n00) + 0.5 * crz), (float)crz);
                }
        // bound of the Cartesian gradient of B = (B_r x / rho, B_r y / rho, B_z) over the table: within a bilinear cell a
        // partial derivative lies between its values on the two opposite edges; the azimuthal term is B_r / rho
        double gz[2] = {0, 0}, gr[2] = {0, 0}, gphi = 0;
        for (int iz = 0; iz < fd->nz; ++iz)
            for (int ir = 0; ir < fd->nr; ++ir)
                for (int c = 0; c < 2; ++c) {
                    const double v = g->field_tab[((size_t)iz * fd->nr + ir) * 2 + c];
                    if (iz + 1 < fd->nz) gz[c] = std::max(gz[c], fabs(g->field_tab[((size_t)(iz + 1) * fd->nr + ir) * 2 + c] - v) / fd->dz_mm);
                    if (ir + 1 < fd->nr) gr[c] = std::max(gr[c], fabs(g->field_tab[((size_t)iz * fd->nr + ir + 1) * 2 + c] - v) / fd->dr_mm);
                    if (c == 0) {
                        const double rho = fd->r0_mm + ir * fd->dr_mm;
                        // |B_r| / rho on the cell [rho_i, rho_i+1]: node value over the inner radius; on the axis B_r
                        // must vanish (then B_r / rho <= the radial slope, already in gr[0])
                        if (rho > 0) gphi = std::max(gphi, fabs(v) / rho);
                        else if (v != 0.0) gphi = INFINITY;
                        if (ir > 0 && fd->r0_mm + (ir - 1) * fd->dr_mm > 0) gphi = std::max(gphi, fabs(v) / (fd->r0_mm + (ir - 1) * fd->dr_mm));
                    }
                }
        g->grad_max = gz[0] + gz[1] + gr[0] + gr[1] + gphi;
        G_CUDA(dev_alloc(&g->d_cells, cells.size()));
        G_CUDA(cudaMemcpy(g->d_cells, cells.data(), sizeof(float4) * cells.size(), cudaMemcpyHostToDevice));
    }
#undef G_CUDA
    GeomDev &d = g->gd;
    d.n_layers = L; d.n_wires_total = g->W; d.n_bit_words = (g->W + 31) / 32;
    d.r_first = (float)g->r[0]; d.inv_pitch = (float)(1.0 / pitch); d.tan_abs = (float)tan_abs;
    const double ulo = std::max(g->r[0] - kLookupReach, 0.0), uhi = g->r[L - 1] + kLookupReach;
    d.u2_lo = (float)(ulo * ulo); d.u2_hi = (float)(uhi * uhi);
    d.R0sq = (float)(g->R0 * g->R0); d.z_half = (float)g->z_half; d.r_out_sq = (float)(g->r_out * g->r_out);
    d.wire4 = g->d_wire4; d.layers = g->d_layers;
    FieldDev &f = g->fd;
    f.kind = fd->kind; f.bz = (float)fd->bz_T; f.nr = fd->nr; f.nz = fd->nz;
    f.r0 = (float)fd->r0_mm; f.z0 = (float)fd->z0_mm;
    f.inv_dr = fd->kind == 1 ? (float)(1.0 / fd->dr_mm) : 0.f; f.inv_dz = fd->kind == 1 ? (float)(1.0 / fd->dz_mm) : 0.f;
    f.grad_max = (float)g->grad_max;
    f.tab = g->d_field; f.cells = g->d_cells; f.n_cells = fd->kind == 1 ? (fd->nr - 1) * (fd->nz - 1) : 0;
    f.cr = fd->kind == 1 ? (float)(-fd->r0_mm / fd->dr_mm - 0.5) : 0.f; f.cz = fd->kind == 1 ? (float)(-fd->z0_mm / fd->dz_mm - 0.5) : 0.f;
    Geom64 &q = g->g64;
    q.n_layers = L; q.n_wires_total = g->W; q.R0 = g->R0; q.z_half = g->z_half; q.r_out = g->r_out;
    q.wire5 = g->d_wire5; q.layers = g->d_layers; q.r_first = d.r_first; q.inv_pitch = d.inv_pitch; q.tan_abs = d.tan_abs;
    q.field_kind = fd->kind; q.bz = fd->bz_T; q.nr = fd->nr; q.nz = fd->nz; q.r0 = fd->r0_mm; q.z0 = fd->z0_mm;
    q.dr = fd->dr_mm; q.dz = fd->dz_mm; q.tab = (const float *)g->d_field;
    *out = g;
    return CDC_OK;
    });
}

extern "C" int32_t cdc_geometry_destroy(cdc_geometry *g)
{
    return cdc_guard("cdc_geometry_destroy", [&]() -> int32_t {
    free_geometry(g);
    return CDC_OK;
    });
}

extern "C" int32_t cdc_geometry_wire_table(const cdc_geometry *g, float *h_wire, int32_t *n_wires_total)
{
    return cdc_guard("cdc_geometry_wire_table", [&]() -> int32_t {
    if (!g) CDC_FAIL(CDC_ERR_INVALID, "cdc_geometry_wire_table: null geometry");
    if (n_wires_total) *n_wires_total = g->W;
    if (h_wire) memcpy(h_wire, g->wire5.data(), sizeof(float) * 5 * (size_t)g->W);
    return CDC_OK;
    });
}
