// Per-step building blocks of the one-seed-per-thread scan kernels (scan.cu, scan_refill.cu): live-wire slots, the
// layer / cell lookup (A5), g and the approach code of a live wire (A6), the packed tabulated-field evaluation.
#pragma once
#include "cdc_internal.cuh"
#include "scan_common.cuh"
#include "scan_args.cuh"
#include "pair_math.cuh"

namespace {

struct Slots {             // live candidate wires of this thread (those that carry a hit), and g at the current vertex
    int w0, w1, w2, w3;
    float g0, g1, g2, g3;
    int n;
};

__device__ __forceinline__ void slot_push(Slots &S, int w, float g)
{
    if (S.n == 0) { S.w0 = w; S.g0 = g; } else if (S.n == 1) { S.w1 = w; S.g1 = g; }
    else if (S.n == 2) { S.w2 = w; S.g2 = g; } else { S.w3 = w; S.g3 = g; }
    S.n += 1;
}

struct LookupCtx {         // the vertex a lookup is made from
    float x, xl, y, yl, z, Tx, Ty, Tz;     // the vertex itself: g of a new slot is evaluated here
    float cz, phi, g_dead, g_far;          // height and azimuth of the lookup centre
    float curv, ptol, hold;                // |a| B_max (0: no pruning by distance, tight curls); window + deviation
                                           // bound; path to the next lookup
};

// a candidate with a hit becomes a live slot unless the track has already passed it for good: once g exceeds
// g_dead it cannot return to <= 0 while the wire is in reach (g' >= |T_perp|^2 - |delta| |T'| >= -(|delta| |a| B)^2 / 4)
__device__ __forceinline__ void consider(const ScanArgs &A, const uint32_t *s_bits, const float *drift_e, int w,
                                         const LookupCtx &V, Slots &S, uint32_t &cnt)
{
    if (!((s_bits[w >> 5] >> (w & 31)) & 1u)) return;
    float ex, ey, eu;
    cnt += 1u;
    const float4 wr = __ldg(A.gd.wire4 + w);
    const float g = wire_g(wr, A.uz, A.inv_uz, V.x, V.xl, V.y, V.yl, V.z, V.Tx, V.Ty, V.Tz, ex, ey, eu);
    if (!(g <= V.g_dead && g > V.g_far)) return;
    // A wire still ahead (g <= 0) comes no closer to the TANGENT than D0 = sqrt(|delta|^2 - g^2 / |T_w|^2), at the path
    // s = -g / |T_w|^2 (T_w: T without its component along the wire).  After a path t the track is within
    // |a| B t^2 / 2 of its tangent and the distance to a line is 1-Lipschitz.  An approach owned before the next lookup
    // (path t* <= hold = K h) is the one minimum of the true distance over the hold, so
    //   D >= D0 - dev,  dev = |a| B hold^2 / 2            (the tangent is nowhere closer than D0), and
    //   D <= D0 + dev  provided s <= hold                 (the true distance at s is a value the minimum cannot exceed).
    // If the drift circle cannot be met within the window even so, the wire is not made a live slot.
    if (g <= 0.0f && V.curv > 0.0f) {
        const float uT = fmaf(wr.z, V.Tx, fmaf(wr.w, V.Ty, A.uz * V.Tz));
        const float tw2 = fmaf(-uT, uT, 1.0f);
        if (tw2 > 0.25f) {
            const float D2 = fmaxf(fmaf(-g, g * rcp_normal(tw2), fmaf(ex, ex, fmaf(ey, ey, -eu * eu))), 0.0f);
            const float d = __ldg(drift_e + w);
            const float hi = d + V.ptol, lo = d - V.ptol;
            if (D2 > hi * hi) return;
            if (lo > 0.0f && D2 < lo * lo && -g <= V.hold * tw2) return;
        }
    }
    slot_push(S, w, g);
}

// cells kc and its nearer neighbour of layer j around azimuth phi at height z -> push those with a hit
__device__ __forceinline__ void lookup_layer(const ScanArgs &A, const LayerDev *s_layer, const uint32_t *s_bits,
                                             const float *drift_e, int j, const LookupCtx &V, Slots &S, uint32_t &cnt)
{
    if ((unsigned)j >= (unsigned)A.gd.n_layers) return;
    const LayerDev L = s_layer[j];
    const float phi = V.phi, z = V.cz;
    const float tau = z * L.shift_k;
    const float sh = fmaf(-0.333333343f * tau * tau, tau, tau);      // atan(tau), |tau| < 0.1
    const float kf = (phi - L.phi0 - sh) * L.kscale;
    const float kn = rintf(kf);
    int k1 = (int)kn;
    int k2 = k1 + ((kf - kn) >= 0.0f ? 1 : -1);
    k1 += (k1 < 0) ? L.n : 0; k1 += (k1 < 0) ? L.n : 0; k1 -= (k1 >= L.n) ? L.n : 0;
    k2 += (k2 < 0) ? L.n : 0; k2 += (k2 < 0) ? L.n : 0; k2 -= (k2 >= L.n) ? L.n : 0;
    consider(A, s_bits, drift_e, L.offset + k1, V, S, cnt);
    consider(A, s_bits, drift_e, L.offset + k2, V, S, cnt);
}

struct Vtx {               // position part of a step vertex: (x, y) and the lo parts the wire offset uses, as pairs
    f2 xy, xyl;
    float z;
};

// g = delta . T for wire wr = (w0x, w0y, ux, uy) at a vertex: wire_g() of scan_common.cuh with the two horizontal
// components of e carried as ONE packed pair (the register pairs of the 128-bit wire load are its operands).  Every
// half rounds like the scalar operation and the order is the same, so the value is bit-identical to wire_g().
__device__ __forceinline__ float wire_gp(const float4 wr, float uz, float inv_uz, f2 xy, f2 xyl, float z, f2 Txy, float Tz,
                                         f2 &exy, float &eu)
{
    const float zt = __fmul_rn(z, inv_uz);
    exy = add2(fma2(bc(-zt), pk(wr.z, wr.w), sub2(xy, pk(wr.x, wr.y))), xyl);
    const float Tx = lo(Txy), Ty = hi(Txy), ex = lo(exy), ey = hi(exy);
    const float uT = __fmaf_rn(wr.z, Tx, __fmaf_rn(wr.w, Ty, __fmul_rn(uz, Tz)));
    eu = __fmaf_rn(ex, wr.z, __fmul_rn(ey, wr.w));
    return __fmaf_rn(ex, Tx, __fmaf_rn(ey, Ty, -__fmul_rn(eu, uT)));
}

// One live wire over interval n: g at the far vertex; on g_n <= 0 < g_{n+1} the interval owns an approach (C9).
__device__ __forceinline__ void slot_step(const ScanArgs &A, const float *drift_e, int w, float &g, bool score,
                                          f2 sdxy, float sdz, const Vtx &v1, f2 Txy1, float Tz1,
                                          uint32_t &nm, float &chi2, uint32_t &cnt)
{
    const float4 wr = __ldg(A.gd.wire4 + w);
    f2 exy1;
    float eu1;
    const float gn = wire_gp(wr, A.uz, A.inv_uz, v1.xy, v1.xyl, v1.z, Txy1, Tz1, exy1, eu1);
    if (score && g <= 0.0f && gn > 0.0f) {
        cnt += 1u << 16;
        // chord point P = r_{n+1} - (1 - tau)(r_{n+1} - r_n): e is linear in the position, and r_{n+1} - r_n is the
        // increment (sdx, sdy, sdz) this step has just added, so e(P) follows from e_{n+1} without the old vertex
        const float zd = sdz * A.inv_uz;
        const f2 dexy = fma2(bc(-zd), pk(wr.z, wr.w), sdxy);
        const float sm = __fdividef(g, g - gn) - 1.0f;         // tau - 1, in [-1, 0)
        const f2 exy = fma2(bc(sm), dexy, exy1);
        const float ex = lo(exy), ey = hi(exy);
        const float eu = fmaf(ex, wr.z, ey * wr.w);
        const float D2 = fmaf(ex, ex, fmaf(ey, ey, -eu * eu));
        const float D = sqrtf(fmaxf(D2, 0.0f));
        const float zP = fmaf(sm, sdz, v1.z);
        const float zw = fmaf(eu, A.uz, zP);
        const float resid = D - __ldg(drift_e + w);
        const float r2 = resid * resid;
        if (fabsf(zw) <= A.gd.z_half && r2 < A.lambda) { nm += 1u; chi2 += r2; }
    }
    g = gn;
}

// a B at (x, y, z), a = kappa q / p: the tabulated field of field_at<1>() (scan_common.cuh) with (B_x, B_y), the two cell
// coordinates and the two halves of each bilinear form carried as packed pairs, and the seed's a folded in here (two
// multiplies per evaluation) instead of into each component of each stage derivative (three per stage: k = U x (a B))
__device__ __forceinline__ void field_at_p(const FieldDev &F, float a, f2 xy, float z, f2 &Bxy, float &Bz)
{
    const float x = lo(xy), y = hi(xy);
    const float rho2 = fmaf(x, x, y * y);
    const float inv_rho = rsqrt_normal(fmaxf(rho2, 1e-30f));
    const float rho = rho2 * inv_rho;
    const f2 f = pk(fmaf(rho, F.inv_dr, F.cr), fmaf(z, F.inv_dz, F.cz));          // (r, z) cell coordinates - 1/2
    const f2 t = add2(f, kMagicRound);
    const f2 w = sub2(f, sub2(t, kMagicRound));                                     // offsets from the cell centre
    const int ir = __float_as_int(lo(t)) - kMagicRoundBits, iz = __float_as_int(hi(t)) - kMagicRoundBits;
    const unsigned cell = min((unsigned)(ir * (F.nz - 1) + iz), (unsigned)(F.n_cells - 1));
    // (keeping the cell's coefficients in registers and loading only on a cell change was measured: no gain, r2)
    const float4 *c = F.cells + 2u * cell;
    const float4 cr = __ldg(c), cz = __ldg(c + 1);                                  // (c0, c_z, c_r, c_rz) of B_r, of B_z
    const f2 tr = fma2(bc(lo(w)), pk(cr.z, cr.w), pk(cr.x, cr.y)), tz = fma2(bc(lo(w)), pk(cz.z, cz.w), pk(cz.x, cz.y));
    const float Br = fmaf(hi(w), hi(tr), lo(tr));
    Bz = a * fmaf(hi(w), hi(tz), lo(tz));
    Bxy = mul2(bc((a * Br) * inv_rho), xy);
}

}  // namespace
