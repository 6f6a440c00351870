// fp32 device helpers shared by the scan kernel (scan.cu) and the re-creation of the paper's thread mapping
// (paper_v1.cu): field evaluation, compensated accumulation, the wire function g, warp max.
#pragma once
#include "cdc_internal.cuh"

namespace {

// MUFU.RSQ / MUFU.RCP without the denormal-input scaling that rsqrtf() / __fdividef() wrap around them: only for
// arguments known to be normal numbers (same result there)
__device__ __forceinline__ float rsqrt_normal(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float rcp_normal(float x)
{
    float r;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// atan2 good to ~2e-5 rad: it only selects candidate cells (a superset with ~7 mm of slack, reading C8).
__device__ __forceinline__ float coarse_atan2(float y, float x)
{
    float ax = fabsf(x), ay = fabsf(y);
    float mx = fmaxf(ax, ay), mn = fminf(ax, ay);
    float t = mn * rcp_normal(fmaxf(mx, 1e-30f));
    float t2 = t * t;
    float p = fmaf(t2, -0.0117212f, 0.05265332f);
    p = fmaf(p, t2, -0.11643287f);
    p = fmaf(p, t2, 0.19354346f);
    p = fmaf(p, t2, -0.33262347f);
    p = fmaf(p, t2, 0.99997726f);
    p = p * t;
    if (ay > ax) p = 1.57079637f - p;
    if (x < 0.0f) p = 3.14159274f - p;
    return copysignf(p, y);
}

constexpr float kMagicRound = 12582912.0f;          // 1.5 * 2^23
constexpr int kMagicRoundBits = 0x4B400000;

template <int FIELD>
__device__ __forceinline__ void field_at(const FieldDev &F, float x, float y, float z, float &Bx, float &By,
                                         float &Bz)
{
    if (FIELD == 0) {
        Bx = 0.0f; By = 0.0f; Bz = F.bz;
    } else {
        // validated at create time: the table covers every point a live track or its stages can reach; the unsigned
        // min on the cell number only keeps a non-finite state inside the allocation.
        // Nearest cell centre by the magic-number rounding (adding 1.5 * 2^23 leaves the rounded integer in the low
        // mantissa bits): no F2I / I2F, and in the two-seed kernel one packed add serves both seeds.  The per-cell
        // coefficients are taken about the cell centre, so the offsets wr, wz lie in [-1/2, 1/2].
        const float rho2 = fmaf(x, x, y * y);
        const float inv_rho = rsqrt_normal(fmaxf(rho2, 1e-30f));
        const float rho = rho2 * inv_rho;
        const float fr = fmaf(rho, F.inv_dr, F.cr), fz = fmaf(z, F.inv_dz, F.cz);     // cell coordinate - 1/2
        const float tr = fr + kMagicRound, tz = fz + kMagicRound;
        const float wr = fr - (tr - kMagicRound), wz = fz - (tz - kMagicRound);
        const int ir = __float_as_int(tr) - kMagicRoundBits, iz = __float_as_int(tz) - kMagicRoundBits;
        const unsigned cell = min((unsigned)(ir * (F.nz - 1) + iz), (unsigned)(F.n_cells - 1));
        const float4 *c = F.cells + 2u * cell;
        const float4 cr = __ldg(c), cz = __ldg(c + 1);                   // (c0, c_z, c_r, c_rz) of B_r, of B_z
        const float Br = fmaf(wz, fmaf(wr, cr.w, cr.y), fmaf(wr, cr.z, cr.x));
        Bz = fmaf(wz, fmaf(wr, cz.w, cz.y), fmaf(wr, cz.z, cz.x));
        const float s = Br * inv_rho;
        Bx = s * x; By = s * y;
    }
}

// Kahan-compensated accumulation: (hi, lo) += d, lo holds what the last rounding lost.
__device__ __forceinline__ void comp_add(float &hi, float &lo, float d)
{
    float y = d + lo;
    float t = hi + y;
    lo = y - (t - hi);
    hi = t;
}

// g = delta . T for wire wr = (w0x, w0y, ux, uy) at a vertex; also returns e (offset of the vertex from the wire
// point at the vertex' own height: a horizontal vector of at most ~17 mm) and e.u.  Written with explicit
// round-to-nearest intrinsics only: the value of g at a vertex must not depend on the call site (it is evaluated
// once as the far end of interval n - 1 or at a lookup, and reused as the near end of interval n).
__device__ __forceinline__ float wire_g(const float4 wr, float uz, float inv_uz, float x, float xl, float y, float yl,
                                        float z, float Tx, float Ty, float Tz, float &ex, float &ey, float &eu)
{
    const float zt = __fmul_rn(z, inv_uz);
    ex = __fadd_rn(__fmaf_rn(-zt, wr.z, __fsub_rn(x, wr.x)), xl);
    ey = __fadd_rn(__fmaf_rn(-zt, wr.w, __fsub_rn(y, wr.y)), yl);
    const float uT = __fmaf_rn(wr.z, Tx, __fmaf_rn(wr.w, Ty, __fmul_rn(uz, Tz)));
    eu = __fmaf_rn(ex, wr.z, __fmul_rn(ey, wr.w));
    return __fmaf_rn(ex, Tx, __fmaf_rn(ey, Ty, -__fmul_rn(eu, uT)));
}

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, v, o);
        v = other > v ? other : v;
    }
    return v;
}

}  // namespace
