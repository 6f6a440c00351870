// A3-A7, the COMPARISON variant (params.kernel_variant = 1): TWO seeds per thread, arithmetic in packed fp32 pairs
// (pair_math.cuh).  Measured slower than the one-seed kernel of scan.cu on B200 (profiles/r2_pair_kernel.md: fewer
// instructions per seed, but 128 / 94 registers, 16 / 20 warps per SM, and the FP32 pipe time is unchanged by packing);
// kept, tested (tests/test_gpu_pair.py), as the measured answer to "carry pairs in f32x2".
//
// The two seeds of a thread are neighbours on the z0 axis of the grid: same theta, px, py, pz, hence the same start
// point in (x, y), the same momentum p (one curvature constant a = kappa q / p for both) and the same start direction.
//   * FIELD == 0 (uniform Bz): the (x, y, Tx, Ty) motion does not depend on z at all, so ONE scalar copy of it serves both
//     seeds exactly (bit for bit what each would compute alone); z, the wire offsets and g are packed pairs.
//   * FIELD == 1 (tabulated field): the two tracks differ through B(r, z): all twelve compensated state components, the
//     three field evaluations, the stage derivatives and the updates are packed pairs -- every FFMA2 / FADD2 / FMUL2 is one
//     issue slot for both seeds.
// Every half of a packed instruction rounds like the scalar instruction, and the operation order is that of the
// one-seed kernel (scan.cu), so per-seed match counts, step counts, the exact best seed and the labels are identical to
// its results (tests/test_gpu_pair.py).
//
//   PAPER.md:51      seed (theta0, z0, px0, py0, pz0) at R0                     -> prologue
//   PAPER.md:55      RKN propagation (textbook Nystroem scheme, reading C5)     -> step body
//   PAPER.md:55,:69  DCA to fired wires, sign-change ownership (reading C9)     -> wire_g2(), score_changes()
//   PAPER.md:65-69   Eq. (1): S = sum (1 - d^2/lambda) over matched terms       -> epilogue
//   PAPER.md:69      lowest E (= highest S) wins                                -> packed-key atomicMax
//
// ONE wire lookup serves both seeds.  It is made around the midpoint of the two seeds' lookup centres, and the number of
// steps K it is good for is chosen per lookup from their measured separation: a wire that can own a match for seed X
// within K steps lies within reach + K h / 2 + sag of X's centre, hence within that + sep of the midpoint, where
// sep = (|d_xy| + sin(eps) |d_z|) / 2 is how far half the centre-to-centre vector can move a point relative to a wire
// (distance to a line is 1-Lipschitz and ignores the component along the wire, which is nearly along z); every wire
// outside the 2 x 2 set is at least `excl` from the midpoint, so K = floor(2 (excl - reach - sag - sep) / h) keeps the
// set a superset for BOTH seeds (reading C8).  In the uniform field d_xy = 0 and d_z is the grid's z0 pitch: K is a
// constant of the thread.  A pair that has drifted too far apart for K >= 1 (never seen; needs > 13 mm) falls back to
// two lookups whose union goes into the slot list (four register slots + four spill slots in shared memory).
// A live wire is evaluated for both seeds (packed g); any sign change of g on a fired wire is a genuine owned approach
// (reading C9), and a wire is in the list once, so no (wire, interval) is scored twice.
//
// Shape of a step: straight-line packed arithmetic (propagation, g of the live wires at the new vertex); on a sign
// change the approach is computed for both seeds at once (packed) and credited to the seed(s) whose g changed sign.
#include <type_traits>

#include "cdc_internal.cuh"
#include "scan_common.cuh"
#include "scan_args.cuh"
#include "pair_math.cuh"

namespace {

constexpr int kSpill = 4;                          // spill slots per thread (shared memory)
#ifndef PAIR_MB0
#define PAIR_MB0 5                                 // resident blocks per SM the register budget is set for: uniform field
#endif
#ifndef PAIR_MB1
#define PAIR_MB1 4                                 // ... tabulated field
#endif

template <typename V> struct is_scalar : std::is_same<V, float> {};

__device__ __forceinline__ f2 P(float v) { return bc(v); }
__device__ __forceinline__ f2 P(f2 v) { return v; }
__device__ __forceinline__ float half_of(float v, int) { return v; }
__device__ __forceinline__ float half_of(f2 v, int which) { return which ? hi(v) : lo(v); }

// g = delta . T of both seeds for wire wr = (w0x, w0y, ux, uy): the packed form of wire_g() in scan_common.cuh, same
// operations in the same order (explicit round-to-nearest: g at a vertex must not depend on the call site).
// V = float: x, y, T shared by the two seeds (uniform field); V = f2: per seed.
template <typename V>
__device__ __forceinline__ f2 wire_g2(const float4 wr, float uz, float inv_uz, V x, V xl, V y, V yl, f2 z, V Tx, V Ty, V Tz,
                                      f2 &ex, f2 &ey, f2 &eu, V &uT)
{
    const f2 zt = mul2(z, inv_uz);
    if constexpr (is_scalar<V>::value) {
        ex = add2(fma2(zt, bc(-wr.z), bc(__fsub_rn(x, wr.x))), bc(xl));
        ey = add2(fma2(zt, bc(-wr.w), bc(__fsub_rn(y, wr.y))), bc(yl));
        uT = __fmaf_rn(wr.z, Tx, __fmaf_rn(wr.w, Ty, __fmul_rn(uz, Tz)));
        eu = fma2(ex, bc(wr.z), mul2(ey, wr.w));
        return fma2(ex, bc(Tx), fma2(ey, bc(Ty), mul2(eu, -uT)));
    } else {
        ex = add2(fma2(zt, bc(-wr.z), sub2(x, wr.x)), xl);
        ey = add2(fma2(zt, bc(-wr.w), sub2(y, wr.y)), yl);
        uT = fma2(bc(wr.z), Tx, fma2(bc(wr.w), Ty, mul2(uz, Tz)));
        eu = fma2(ex, bc(wr.z), mul2(ey, wr.w));
        return fma2(ex, Tx, fma2(ey, Ty, neg2(mul2(eu, uT))));
    }
}

struct LookupBounds {       // shared by the two seeds (same |a|): see consider() in scan.cu for the derivations
    float g_dead, g_far, curv, ptol, hold;
};

// May a candidate wire that carries a hit own a MATCHING approach of seed A or of seed B before the next lookup?
// The per-seed test is keep_wire() of scan.cu (bounds, not approximations), evaluated for both seeds at once.
template <typename V>
__device__ __forceinline__ bool keep_wire2(const LookupBounds &B, float drift, f2 g, f2 ex, f2 ey, f2 eu, V uT)
{
    bool okA = lo(g) <= B.g_dead && lo(g) > B.g_far, okB = hi(g) <= B.g_dead && hi(g) > B.g_far;
    if (!(okA || okB)) return false;
    if (B.curv > 0.0f) {
        f2 tw2;
        if constexpr (is_scalar<V>::value) tw2 = bc(fmaf(-uT, uT, 1.0f));
        else tw2 = fma2(neg2(uT), uT, bc(1.0f));
        const f2 rc = pk(rcp_normal(lo(tw2)), rcp_normal(hi(tw2)));
        const f2 e2 = fma2(ex, ex, fma2(ey, ey, neg2(mul2(eu, eu))));
        const f2 D2 = fma2(neg2(g), mul2(g, rc), e2);
        const float D2A = fmaxf(lo(D2), 0.0f), D2B = fmaxf(hi(D2), 0.0f);
        const float hi_ = drift + B.ptol, lo_ = drift - B.ptol;
        const float hi2 = hi_ * hi_, lo2 = lo_ * lo_;
        const bool near_ok = lo_ > 0.0f;
        const bool prA = lo(g) <= 0.0f && lo(tw2) > 0.25f && (D2A > hi2 || (near_ok && D2A < lo2 && -lo(g) <= B.hold * lo(tw2)));
        const bool prB = hi(g) <= 0.0f && hi(tw2) > 0.25f && (D2B > hi2 || (near_ok && D2B < lo2 && -hi(g) <= B.hold * hi(tw2)));
        okA = okA && !prA; okB = okB && !prB;
    }
    return okA || okB;
}

// cells kc and its nearer neighbour of layer j around azimuth phi at height z (the arithmetic of lookup_layer in scan.cu)
__device__ __forceinline__ void layer_cells(const ScanArgs &A, const LayerDev *s_layer, int j, float phi, float z, int &ca,
                                            int &cb)
{
    ca = -1; cb = -1;
    if ((unsigned)j >= (unsigned)A.gd.n_layers) return;
    const LayerDev L = s_layer[j];
    const float tau = z * L.shift_k;
    const float sh = fmaf(-0.333333343f * tau * tau, tau, tau);      // atan(tau), |tau| < 0.1
    const float kf = (phi - L.phi0 - sh) * L.kscale;
    const float kn = rintf(kf);
    int k1 = (int)kn;
    int k2 = k1 + ((kf - kn) >= 0.0f ? 1 : -1);
    k1 += (k1 < 0) ? L.n : 0; k1 += (k1 < 0) ? L.n : 0; k1 -= (k1 >= L.n) ? L.n : 0;
    k2 += (k2 < 0) ? L.n : 0; k2 += (k2 < 0) ? L.n : 0; k2 -= (k2 >= L.n) ? L.n : 0;
    ca = L.offset + k1; cb = L.offset + k2;
}

__device__ __forceinline__ bool wire_hit(const uint32_t *s_bits, int w)
{
    return w >= 0 && ((s_bits[w >> 5] >> (w & 31)) & 1u);
}

// The owned approach of interval n to one wire, computed for both seeds at once (the operations of approach() in
// scan.cu, packed) and credited to the seed(s) whose g changed sign: g_n <= 0 < g_{n+1} (reading C9).  For a seed
// whose g did not change sign the packed halves hold don't-care values.
template <typename V>
__device__ __forceinline__ void approach2(const ScanArgs &A, const float4 wr, float drift, f2 g, f2 gn, f2 ex1, f2 ey1, V sdx,
                                          V sdy, V sdz, f2 z1, bool doA, bool doB, uint32_t &nmA, uint32_t &nmB, float &chi2A,
                                          float &chi2B)
{
    // chord point P = r_{n+1} - (1 - tau)(r_{n+1} - r_n): e is linear in the position, and r_{n+1} - r_n is the increment
    // (sdx, sdy, sdz) this step has just added, so e(P) follows from e_{n+1} without the old vertex
    f2 dex, dey;
    if constexpr (is_scalar<V>::value) {
        const float zd = sdz * A.inv_uz;
        dex = bc(fmaf(-zd, wr.z, sdx)); dey = bc(fmaf(-zd, wr.w, sdy));
    } else {
        const f2 zd = mul2(sdz, A.inv_uz);
        dex = fma2(zd, bc(-wr.z), sdx); dey = fma2(zd, bc(-wr.w), sdy);
    }
    const f2 den = sub2(g, gn);
    const f2 sm = sub2(pk(__fdividef(lo(g), lo(den)), __fdividef(hi(g), hi(den))), 1.0f);     // tau - 1, in [-1, 0)
    const f2 ex = fma2(sm, dex, ex1), ey = fma2(sm, dey, ey1);
    const f2 eu = fma2(ex, bc(wr.z), mul2(ey, wr.w));
    const f2 D2 = fma2(ex, ex, fma2(ey, ey, neg2(mul2(eu, eu))));
    const f2 D = pk(sqrtf(fmaxf(lo(D2), 0.0f)), sqrtf(fmaxf(hi(D2), 0.0f)));
    const f2 zw = fma2(eu, bc(A.uz), fma2(sm, P(sdz), z1));
    const f2 resid = sub2(D, drift);
    const f2 r2 = mul2(resid, resid);
    // chi2 += resid^2 as ONE fused operation, as the compiler contracts it in the one-seed kernel
    if (doA && fabsf(lo(zw)) <= A.gd.z_half && lo(r2) < A.lambda) { nmA += 1u; chi2A = __fmaf_rn(lo(resid), lo(resid), chi2A); }
    if (doB && fabsf(hi(zw)) <= A.gd.z_half && hi(r2) < A.lambda) { nmB += 1u; chi2B = __fmaf_rn(hi(resid), hi(resid), chi2B); }
}

// bilinear field of both seeds (FIELD == 1): field_at<1>() of scan_common.cuh for two seeds.  Cell search and the cell
// offsets are packed (one magic-number add rounds both seeds' coordinates); each seed then loads its own cell and
// forms (c0, c_z) + wr (c_r, c_rz) with ONE packed FMA on the two register pairs of the 128-bit load; the last FMA of
// each component is scalar and its two results land side by side as the pair the packed stage arithmetic consumes.
__device__ __forceinline__ void field_at2(const FieldDev &F, f2 x, f2 y, f2 z, f2 &Bx, f2 &By, f2 &Bz)
{
    const f2 rho2 = fma2(x, x, mul2(y, y));
    const f2 inv_rho = pk(rsqrt_normal(fmaxf(lo(rho2), 1e-30f)), rsqrt_normal(fmaxf(hi(rho2), 1e-30f)));
    const f2 rho = mul2(rho2, inv_rho);
    const f2 fr = fma2(rho, bc(F.inv_dr), bc(F.cr)), fz = fma2(z, bc(F.inv_dz), bc(F.cz));      // cell coordinate - 1/2
    const f2 tr = add2(fr, kMagicRound), tz = add2(fz, kMagicRound);
    const f2 wr = sub2(fr, sub2(tr, kMagicRound)), wz = sub2(fz, sub2(tz, kMagicRound));
    const int nzc = F.nz - 1;
    const unsigned cellA = min((unsigned)((__float_as_int(lo(tr)) - kMagicRoundBits) * nzc + (__float_as_int(lo(tz)) - kMagicRoundBits)),
                               (unsigned)(F.n_cells - 1));
    const unsigned cellB = min((unsigned)((__float_as_int(hi(tr)) - kMagicRoundBits) * nzc + (__float_as_int(hi(tz)) - kMagicRoundBits)),
                               (unsigned)(F.n_cells - 1));
    const float4 *cA = F.cells + 2u * cellA, *cB = F.cells + 2u * cellB;
    const float4 rA = __ldg(cA), zA = __ldg(cA + 1), rB = __ldg(cB), zB = __ldg(cB + 1);
    // per seed: (t0, t1) = (c0, c_z) + wr (c_r, c_rz); B = t0 + wz t1 -- the operations of the scalar form
    const f2 trA = fma2(bc(lo(wr)), pk(rA.z, rA.w), pk(rA.x, rA.y)), tzA = fma2(bc(lo(wr)), pk(zA.z, zA.w), pk(zA.x, zA.y));
    const f2 trB = fma2(bc(hi(wr)), pk(rB.z, rB.w), pk(rB.x, rB.y)), tzB = fma2(bc(hi(wr)), pk(zB.z, zB.w), pk(zB.x, zB.y));
    const f2 Br = pk(fmaf(lo(wz), hi(trA), lo(trA)), fmaf(hi(wz), hi(trB), lo(trB)));
    Bz = pk(fmaf(lo(wz), hi(tzA), lo(tzA)), fmaf(hi(wz), hi(tzB), lo(tzB)));
    const f2 s = mul2(Br, inv_rho);
    Bx = mul2(s, x); By = mul2(s, y);
}

// a (T x B) of both seeds
__device__ __forceinline__ void lorentz2(float a, f2 Ux, f2 Uy, f2 Uz, f2 Bx, f2 By, f2 Bz, f2 &kx, f2 &ky, f2 &kz)
{
    kx = mul2(a, fma2(Uy, Bz, neg2(mul2(Uz, By))));
    ky = mul2(a, fma2(Uz, Bx, neg2(mul2(Ux, Bz))));
    kz = mul2(a, fma2(Ux, By, neg2(mul2(Uy, Bx))));
}

// TRACK: keep the in-gas flag, the in-gas step count and the turn counter (needed with energy loss, for the debug record,
// and when a held wire could be scored from a vertex inside R0; see launch_seed_scan).
// FIELD == 0 with ELOSS: the momentum p_n = p0 - eps h m_n follows the (x, y) path, which the two seeds share: one a.
template <int FIELD, bool ELOSS, bool TRACK>
__global__ void __launch_bounds__(kBlock, FIELD == 0 ? PAIR_MB0 : PAIR_MB1) seed_scan_pair_kernel(const ScanArgs A)
{
    using V = typename std::conditional<FIELD == 0, float, f2>::type;
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    __shared__ uint32_t s_bits[kMaxBitWords];
    __shared__ int s_spw[kSpill * kBlock];
    __shared__ unsigned long long s_spg[kSpill * kBlock];

    const int e = blockIdx.y;
    const GridDev G = A.grids[e];
    const int nzp = (G.n[1] + 1) >> 1;                       // z0 nodes are taken two at a time
    const int n_pairs = (int)(((int64_t)G.n_seeds / G.n[1]) * nzp);
    if ((int64_t)blockIdx.x * kBlock >= (int64_t)n_pairs) return;
    for (int i = threadIdx.x; i < A.gd.n_layers; i += kBlock) s_layer[i] = A.gd.layers[i];
    for (int i = threadIdx.x; i < A.gd.n_bit_words; i += kBlock)
        s_bits[i] = A.bits[(size_t)e * A.gd.n_bit_words + i];
    __syncthreads();
    const float *drift_e = A.drift_tab + (size_t)e * A.gd.n_wires_total;
    int *sp_w = s_spw + threadIdx.x;
    unsigned long long *sp_g = s_spg + threadIdx.x;

    // ---- A3: thread -> two seeds.  The z0 pair index is the lane-fastest axis, then theta, px, py, pz: the 64 tracks of a
    // warp pass the same wires within a step or two of one another.
    const int t = blockIdx.x * kBlock + threadIdx.x;
    const bool valid = t < n_pairs;
    int q = valid ? t : 0;
    const int i_zp = q % nzp; q /= nzp;
    const int i_th = q % G.n[0]; q /= G.n[0];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_py = q % G.n[3];
    const int i_pz = q / G.n[3];
    const int i_zA = 2 * i_zp, i_zB = min(i_zA + 1, G.n[1] - 1);
    const bool validB = valid && (i_zA + 1 < G.n[1]);
    const uint32_t indexA = (uint32_t)((((i_th * G.n[1] + i_zA) * G.n[2] + i_px) * G.n[3] + i_py) * G.n[4] + i_pz);
    const uint32_t indexB = (uint32_t)((((i_th * G.n[1] + i_zB) * G.n[2] + i_px) * G.n[3] + i_py) * G.n[4] + i_pz);

    V xh, xl, yh, yl, Txh, Txl, Tyh, Tyl, Tzh, Tzl;
    f2 zh, zl;
    float a, epsT, p0h, p0l;
    float ub_h = 0.f, ub_l = 0.f, ue1 = 0.f, up1 = 0.f, up2_h = 0.f, up2_l = 0.f;   // uniform-field step map (FIELD == 0)
    {
        const double *ax = A.axes + (size_t)e * 6 * A.axis_stride;
        const double x0 = ax[i_th], y0 = ax[A.axis_stride + i_th];
        const double zA0 = ax[2 * A.axis_stride + i_zA], zB0 = ax[2 * A.axis_stride + i_zB];
        const double px = ax[3 * A.axis_stride + i_px], py = ax[4 * A.axis_stride + i_py], pz = ax[5 * A.axis_stride + i_pz];
        const double p0 = sqrt(px * px + py * py + pz * pz);
        const double tx = px / p0, ty = py / p0, tz = pz / p0;
        const float fxh = (float)x0, fxl = (float)(x0 - (double)fxh), fyh = (float)y0, fyl = (float)(y0 - (double)fyh);
        const float ftxh = (float)tx, ftxl = (float)(tx - (double)ftxh), ftyh = (float)ty, ftyl = (float)(ty - (double)ftyh);
        const float ftzh = (float)tz, ftzl = (float)(tz - (double)ftzh);
        const float zAh = (float)zA0, zAl = (float)(zA0 - (double)zAh), zBh = (float)zB0, zBl = (float)(zB0 - (double)zBh);
        zh = pk(zAh, zBh); zl = pk(zAl, zBl);
        if constexpr (FIELD == 0) {
            xh = fxh; xl = fxl; yh = fyh; yl = fyl; Txh = ftxh; Txl = ftxl; Tyh = ftyh; Tyl = ftyl; Tzh = ftzh; Tzl = ftzl;
        } else {
            xh = bc(fxh); xl = bc(fxl); yh = bc(fyh); yl = bc(fyl); Txh = bc(ftxh); Txl = bc(ftxl);
            Tyh = bc(ftyh); Tyl = bc(ftyl); Tzh = bc(ftzh); Tzl = bc(ftzl);
        }
        const double a64 = A.kq / p0;
        a = (float)a64;
        // the fp32 roundings of a and h/6 are the same every step; fold their ratio into the T update
        epsT = (float)((a64 * A.h6_64) / ((double)a * (double)A.h_6) - 1.0);
        if (ELOSS) epsT = (float)((A.kq * A.h6_64) / ((double)(float)A.kq * (double)A.h_6) - 1.0);
        p0h = (float)p0; p0l = (float)(p0 - (double)p0h);
        if (FIELD == 0) {                              // step-map constants in fp64, the two O(theta) ones as hi + lo
            const double h64 = 6.0 * A.h6_64, th = a64 * (double)A.fd.bz * h64, th2 = th * th;
            const double b = th - th * th2 / 6.0, p2 = h64 * (th / 2.0 - th * th2 / 24.0);
            ub_h = (float)b; ub_l = (float)(b - (double)ub_h);
            up2_h = (float)p2; up2_l = (float)(p2 - (double)up2_h);
            ue1 = (float)(-th2 / 2.0 + th2 * th2 / 24.0);
            up1 = (float)(-h64 * th2 / 6.0);
        }
    }
    // p <= 1 MeV/c ends a track after its first step (C7); a thread beyond the grid takes no step
    const int max_steps = !valid ? 0 : ((p0h > 1.0f) ? A.max_steps : min(A.max_steps, 1));

    uint32_t nmA = 0, nmB = 0, cnt = 0, tests = 0, lookups = 0;
    float chi2A = 0.0f, chi2B = 0.0f;
    int n = 0, kcount = 0;
    int nA = 0, nB = 0;                               // steps taken by each seed
    bool aliveA = valid && max_steps > 0, aliveB = validB && max_steps > 0;
    // in-gas flag, in-gas step count, turn counter: one set in the uniform field (shared path), one per seed otherwise
    bool cn = true, cnB = true;                       // c_0 := true (reading C7)
    int m = 0, mB = 0, turn = 0, turnB = 0;
    const float h = A.h;
    int w0 = 0, w1 = 0, w2 = 0, w3 = 0, ns = 0;       // live wires: ids, count
    f2 g0 = bc(0.0f), g1 = bc(0.0f), g2 = bc(0.0f), g3 = bc(0.0f);   // ... and g of both seeds at the current vertex
    // final state of a seed that ended before its partner (debug record only)
    double fxA = 0, fyA = 0, fzA = 0, fxB = 0, fyB = 0, fzB = 0;
    int fmA = 0, fmB = 0, ftA = 0, ftB = 0;
    // uniform field: the two seeds differ by the constant z0 pitch only -> the separation term of K is a constant
    const float sep_z = 0.5f * A.sin_eps * fabsf(hi(zh) - lo(zh)) + 0.02f;

#pragma unroll 1
    while (n < max_steps) {
        // ---- A5: every K steps, the wires near the two tracks that carry a hit -> slots, with g at this vertex
        if (kcount == 0) {
            ns = 0;
            // half the separation of the two seeds as a wire sees it (see the header): with one seed left, none
            float sep;
            if constexpr (FIELD == 0) sep = sep_z;
            else {
                const f2 ddx = sub2(xh, pk(hi(xh), lo(xh))), ddy = sub2(yh, pk(hi(yh), lo(yh)));
                const float dxy2 = fmaf(lo(ddx), lo(ddx), lo(ddy) * lo(ddy));
                sep = fmaf(0.5f, dxy2 * rsqrt_normal(fmaxf(dxy2, 1e-30f)), 0.5f * A.sin_eps * fabsf(hi(zh) - lo(zh)) + 0.03f);
            }
            if (!(aliveA && aliveB)) sep = 0.0f;
            const bool tight = !(fabsf(a) * A.b_max < A.tight_curv);
            int K = tight ? 0 : min(A.lookup_every, (int)((A.k_margin - sep) * A.two_inv_h));           // floor: the operand is > 0 or K <= 0
            float ahead = 0.5f * h * (float)K;
            if (K < 1) { K = min(A.lookup_every_tight, 1 + (int)((A.k_margin0 - sep) * A.inv_h)); ahead = 0.0f; }
            const bool split = K < 1 || !(sep <= A.sep_cap);             // too far apart: one lookup per seed, union of the sets
            if (split) K = A.lookup_every_tight;
            kcount = K;
            LookupBounds Bd;
            {
                const float cbend = (ELOSS ? 1.05f : 1.0f) * A.delta_max * fabsf(a) * A.b_max;
                Bd.g_dead = fmaf(A.hold_path * 0.25f, cbend * cbend, 0.02f);
                Bd.g_far = -fmaf((float)K * h, 1.0f + cbend, 0.25f);
                Bd.curv = (tight || ahead == 0.0f) ? 0.0f : (ELOSS ? 1.05f : 1.0f) * fabsf(a) * A.b_max;
                const float hold = (float)K * h + 0.5f;                // path to the next lookup (+ margin)
                Bd.ptol = fmaf(0.6f * Bd.curv, hold * hold, A.window + 0.05f);
                Bd.hold = hold;
            }
            const int n_pass = split ? 2 : 1;
#pragma unroll 1
            for (int pass = 0; pass < n_pass; ++pass) {
                // lookup centre: the midpoint of the two seeds' centres r + ahead T, or (split) one seed's own position
                float cx, cy, cz;
                {
                    const f2 czz = fma2(bc(ahead), P(Tzh), zh);
                    float cxA, cxB, cyA, cyB;
                    if constexpr (FIELD == 0) { cxA = cxB = fmaf(ahead, Txh, xh); cyA = cyB = fmaf(ahead, Tyh, yh); }
                    else {
                        const f2 cxx = fma2(bc(ahead), Txh, xh), cyy = fma2(bc(ahead), Tyh, yh);
                        cxA = lo(cxx); cxB = hi(cxx); cyA = lo(cyy); cyB = hi(cyy);
                    }
                    const bool useA = split ? pass == 0 : aliveA, useB = split ? pass == 1 : aliveB;
                    if (useA && useB) { cx = 0.5f * (cxA + cxB); cy = 0.5f * (cyA + cyB); cz = 0.5f * (lo(czz) + hi(czz)); }
                    else if (useA) { cx = cxA; cy = cyA; cz = lo(czz); }
                    else { cx = cxB; cy = cyB; cz = hi(czz); }
                    if (split && !(pass == 0 ? aliveA : aliveB)) continue;
                }
                const float zeta = cz * A.gd.tan_abs;
                const float u2 = fmaf(cx, cx, fmaf(cy, cy, -zeta * zeta));
                if (!(u2 > A.u2_lo && u2 < A.u2_hi)) continue;
                lookups += 1u;
                const float u = u2 * rsqrt_normal(u2);                  // u2 > u2_lo > 0
                const float fj = (u - A.gd.r_first) * A.gd.inv_pitch;
                const float jn = rintf(fj);
                const int jc = (int)jn;
                const int j2 = jc + ((fj - jn) >= 0.0f ? 1 : -1);
                const float phi = coarse_atan2(cy, cx);
                int c0, c1, c2, c3;
                layer_cells(A, s_layer, jc, phi, cz, c0, c1);
                layer_cells(A, s_layer, j2, phi, cz, c2, c3);
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int w = i == 0 ? c0 : i == 1 ? c1 : i == 2 ? c2 : c3;
                    if (!wire_hit(s_bits, w)) continue;
                    if (pass == 1) {                                    // split: the other seed's pass may have it already
                        bool dup = (ns > 0 && w == w0) || (ns > 1 && w == w1) || (ns > 2 && w == w2) || (ns > 3 && w == w3);
                        for (int k = 4; k < ns; ++k) dup = dup || w == sp_w[(k - 4) * kBlock];
                        if (dup) continue;
                    }
                    const float4 wr = __ldg(A.gd.wire4 + w);
                    const float drift = __ldg(drift_e + w);
                    f2 ex, ey, eu;
                    V uT;
                    const f2 g = wire_g2<V>(wr, A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex, ey, eu, uT);
                    cnt += (aliveA ? 1u : 0u) + (aliveB ? 1u : 0u);
                    if (!keep_wire2<V>(Bd, drift, g, ex, ey, eu, uT)) continue;
                    if (ns == 0) { w0 = w; g0 = g; } else if (ns == 1) { w1 = w; g1 = g; }
                    else if (ns == 2) { w2 = w; g2 = g; } else if (ns == 3) { w3 = w; g3 = g; }
                    else { sp_w[(ns - 4) * kBlock] = w; sp_g[(ns - 4) * kBlock] = g.v; }
                    ns += 1;
                }
            }
        }
        kcount -= 1;
        V sdx, sdy, sdz;                               // the increment this step adds to the position

        // ---- A4: one Nystroem-RK4 step of r'' = a (r' x B(r))
        if constexpr (FIELD == 0) {
            // uniform field: the closed-form step map of scan.cu, one scalar copy for both seeds; z packed
            if (ELOSS) {
                const float th = a * A.fd.bz * h, th2 = th * th;
                ub_h = fmaf(-th * th2, 0.166666672f, th); ub_l = ub_h * A.kq_rel;
                ue1 = th2 * fmaf(th2, 0.0416666679f, -0.5f);
                up1 = -h * th2 * 0.166666672f;
                up2_h = h * th * fmaf(th2, -0.0416666679f, 0.5f); up2_l = up2_h * A.kq_rel;
            }
            const float dTx = fmaf(ue1, Txh, fmaf(ub_h, Tyh, ub_l * Tyh));
            const float dTy = fmaf(ue1, Tyh, -fmaf(ub_h, Txh, ub_l * Txh));
            const float dx = fmaf(up1, Txh, fmaf(up2_h, Tyh, fmaf(up2_l, Tyh, h * Txh)));
            const float dy = fmaf(up1, Tyh, -fmaf(up2_h, Txh, fmaf(up2_l, Txh, -h * Tyh)));
            sdx = fmaf(h, Txl, dx); sdy = fmaf(h, Tyl, dy); sdz = fmaf(h, Tzl, h * Tzh);
            comp_add(xh, xl, sdx);
            comp_add(yh, yl, sdy);
            comp_add2(zh, zl, bc(sdz));
            comp_add(Txh, Txl, dTx);
            comp_add(Tyh, Tyl, dTy);
        } else {
            f2 Bx, By, Bz, k1x, k1y, k1z, k2x, k2y, k2z, k3x, k3y, k3z, k4x, k4y, k4z;
            field_at2(A.fd, xh, yh, zh, Bx, By, Bz);
            lorentz2(a, Txh, Tyh, Tzh, Bx, By, Bz, k1x, k1y, k1z);
            f2 Ux = fma2(A.h_half, k1x, Txh), Uy = fma2(A.h_half, k1y, Tyh), Uz = fma2(A.h_half, k1z, Tzh);
            {
                const f2 mx = fma2(A.h2_8, k1x, fma2(A.h_half, Txh, xh));
                const f2 my = fma2(A.h2_8, k1y, fma2(A.h_half, Tyh, yh));
                const f2 mz = fma2(A.h2_8, k1z, fma2(A.h_half, Tzh, zh));
                field_at2(A.fd, mx, my, mz, Bx, By, Bz);
            }
            lorentz2(a, Ux, Uy, Uz, Bx, By, Bz, k2x, k2y, k2z);
            Ux = fma2(A.h_half, k2x, Txh); Uy = fma2(A.h_half, k2y, Tyh); Uz = fma2(A.h_half, k2z, Tzh);
            lorentz2(a, Ux, Uy, Uz, Bx, By, Bz, k3x, k3y, k3z);
            Ux = fma2(h, k3x, Txh); Uy = fma2(h, k3y, Tyh); Uz = fma2(h, k3z, Tzh);
            {
                const f2 qx = fma2(A.h2_2, k3x, fma2(h, Txh, xh));
                const f2 qy = fma2(A.h2_2, k3y, fma2(h, Tyh, yh));
                const f2 qz = fma2(A.h2_2, k3z, fma2(h, Tzh, zh));
                field_at2(A.fd, qx, qy, qz, Bx, By, Bz);
            }
            lorentz2(a, Ux, Uy, Uz, Bx, By, Bz, k4x, k4y, k4z);
            const f2 dx = fma2(A.h2_6, add2(add2(k1x, k2x), k3x), mul2(h, Txh));
            const f2 dy = fma2(A.h2_6, add2(add2(k1y, k2y), k3y), mul2(h, Tyh));
            const f2 dz = fma2(A.h2_6, add2(add2(k1z, k2z), k3z), mul2(h, Tzh));
            const f2 dTx = mul2(A.h_6, fma2(bc(2.0f), add2(k2x, k3x), add2(k1x, k4x)));
            const f2 dTy = mul2(A.h_6, fma2(bc(2.0f), add2(k2y, k3y), add2(k1y, k4y)));
            const f2 dTz = mul2(A.h_6, fma2(bc(2.0f), add2(k2z, k3z), add2(k1z, k4z)));
            sdx = fma2(h, Txl, dx); sdy = fma2(h, Tyl, dy); sdz = fma2(h, Tzl, dz);
            comp_add2(xh, xl, sdx);
            comp_add2(yh, yl, sdy);
            comp_add2(zh, zl, sdz);
            comp_add2(Txh, Txl, fma2(dTx, bc(epsT), dTx));
            comp_add2(Tyh, Tyl, fma2(dTy, bc(epsT), dTy));
            comp_add2(Tzh, Tzl, fma2(dTz, bc(epsT), dTz));
        }

        // ---- A6: live wires over interval n: g of both seeds at the new vertex; on a sign change g_n <= 0 < g_{n+1}
        // (reading C9) of a seed that is alive and whose interval starts in the gas, the approach is scored
        if (ns > 0) {
            tests += (uint32_t)ns * ((aliveA ? 1u : 0u) + (aliveB ? 1u : 0u));
            const bool scA = aliveA && cn, scB = aliveB && (FIELD == 0 ? cn : cnB);
            auto slot = [&](int w, f2 &g) {
                const float4 wr = __ldg(A.gd.wire4 + w);
                f2 ex1, ey1, eu1;
                V uT;
                const f2 gn = wire_g2<V>(wr, A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex1, ey1, eu1, uT);
                const bool chA = scA && lo(g) <= 0.0f && lo(gn) > 0.0f, chB = scB && hi(g) <= 0.0f && hi(gn) > 0.0f;
                if (chA || chB) {
                    cnt += (chA ? 1u << 16 : 0u) + (chB ? 1u << 16 : 0u);
                    approach2<V>(A, wr, __ldg(drift_e + w), g, gn, ex1, ey1, sdx, sdy, sdz, zh, chA, chB, nmA, nmB, chi2A, chi2B);
                }
                g = gn;
            };
            slot(w0, g0);
            if (ns > 1) slot(w1, g1);
            if (ns > 2) slot(w2, g2);
            if (ns > 3) {
                slot(w3, g3);
#pragma unroll 1
                for (int i = 4; i < ns; ++i) {             // spilled slots (split lookups with more than four fired wires in reach)
                    f2 g; g.v = sp_g[(i - 4) * kBlock];
                    slot(sp_w[(i - 4) * kBlock], g);
                    sp_g[(i - 4) * kBlock] = g.v;
                }
            }
        }
        if (TRACK) {
            if (FIELD == 0) { if (cn) m += 1; }
            else { if (cn && aliveA) m += 1; if (cnB && aliveB) mB += 1; }
        }

        // ---- advance, energy loss (reading C6), turn counter and termination (reading C7)
        n += 1;
        bool outA, outB;                               // beyond r_out
        if constexpr (FIELD == 0) {
            const float rho2 = fmaf(xh, xh, yh * yh);
            if (TRACK) {
                const bool cnext = rho2 >= A.gd.R0sq;
                if (!cn && cnext) turn += 1;
                cn = cnext;
            }
            outA = outB = !(rho2 <= A.gd.r_out_sq);
            if (ELOSS) {
                const float p = fmaf(-A.eloss_h, (float)m, p0h) + p0l;
                a = (float)A.kq / p;      // IEEE division
                if (!(p > 1.0f)) outA = outB = true;
            }
        } else {
            const f2 rho2 = fma2(xh, xh, mul2(yh, yh));
            if (TRACK) {
                const bool cnextA = lo(rho2) >= A.gd.R0sq, cnextB = hi(rho2) >= A.gd.R0sq;
                if (aliveA) { if (!cn && cnextA) turn += 1; cn = cnextA; }
                if (aliveB) { if (!cnB && cnextB) turnB += 1; cnB = cnextB; }
            }
            outA = !(lo(rho2) <= A.gd.r_out_sq); outB = !(hi(rho2) <= A.gd.r_out_sq);
        }
        const bool endA = aliveA && (outA || !(fabsf(lo(zh)) <= A.gd.z_half));
        const bool endB = aliveB && (outB || !(fabsf(hi(zh)) <= A.gd.z_half));
        if (endA || endB) {
            if (endA) {
                aliveA = false; nA = n;
                if (TRACK) {
                    fxA = (double)half_of(xh, 0) + (double)half_of(xl, 0); fyA = (double)half_of(yh, 0) + (double)half_of(yl, 0);
                    fzA = (double)lo(zh) + (double)lo(zl); fmA = m; ftA = turn;
                }
            }
            if (endB) {
                aliveB = false; nB = n;
                if (TRACK) {
                    fxB = (double)half_of(xh, 1) + (double)half_of(xl, 1); fyB = (double)half_of(yh, 1) + (double)half_of(yl, 1);
                    fzB = (double)hi(zh) + (double)hi(zl); fmB = FIELD == 0 ? m : mB; ftB = FIELD == 0 ? turn : turnB;
                }
            }
            if (!(aliveA || aliveB)) break;
        }
    }
    if (aliveA) {                                      // ended on the step cap
        nA = n;
        if (TRACK) {
            fxA = (double)half_of(xh, 0) + (double)half_of(xl, 0); fyA = (double)half_of(yh, 0) + (double)half_of(yl, 0);
            fzA = (double)lo(zh) + (double)lo(zl); fmA = m; ftA = turn;
        }
    }
    if (aliveB) {
        nB = n;
        if (TRACK) {
            fxB = (double)half_of(xh, 1) + (double)half_of(xl, 1); fyB = (double)half_of(yh, 1) + (double)half_of(yl, 1);
            fzB = (double)hi(zh) + (double)hi(zl); fmB = FIELD == 0 ? m : mB; ftB = FIELD == 0 ? turn : turnB;
        }
    }

    // ---- A7: per-seed output, per-event argmax, candidate pool
    const float ScA = valid ? fmaxf(fmaf(-chi2A, A.inv_lambda, (float)nmA), 0.0f) : 0.0f;   // S >= 0 by construction
    const float ScB = validB ? fmaxf(fmaf(-chi2B, A.inv_lambda, (float)nmB), 0.0f) : 0.0f;
    if (valid) {
        const int64_t o = G.out_offset + (int64_t)indexA;
        if (A.n_match) A.n_match[o] = nmA;
        if (A.chi2) A.chi2[o] = chi2A;
        if (TRACK && A.debug) {
            cdc_seed_debug d;
            d.n_steps = nA; d.turns = ftA; d.m_gas = fmA; d.pad = 0; d.x = fxA; d.y = fyA; d.z = fzA;
            A.debug[o] = d;
        }
    }
    if (validB) {
        const int64_t o = G.out_offset + (int64_t)indexB;
        if (A.n_match) A.n_match[o] = nmB;
        if (A.chi2) A.chi2[o] = chi2B;
        if (TRACK && A.debug) {
            cdc_seed_debug d;
            d.n_steps = nB; d.turns = ftB; d.m_gas = fmB; d.pad = 0; d.x = fxB; d.y = fyB; d.z = fzB;
            A.debug[o] = d;
        }
    }
    const unsigned long long keyA = valid ? (((unsigned long long)__float_as_uint(ScA) << 32) | (0xFFFFFFFFu - indexA)) : 0ull;
    const unsigned long long keyB = validB ? (((unsigned long long)__float_as_uint(ScB) << 32) | (0xFFFFFFFFu - indexB)) : 0ull;
    const unsigned long long wkey = warp_max_u64(keyA > keyB ? keyA : keyB);
    const int lane = threadIdx.x & 31;
    unsigned long long run = 0ull;
    if (lane == 0) {
        const unsigned long long old = atomicMax(A.best_key + e, wkey);
        run = old > wkey ? old : wkey;
    }
    run = __shfl_sync(0xffffffffu, run, 0);
    const float S_run = __uint_as_float((uint32_t)(run >> 32));
    // a seed without any match (S = 0 exactly) cannot beat index 0, which ties with it and wins on the index: only
    // index 0 stands in for all of them, so an event (or a neighbourhood) without hits cannot flood the pool
    const bool candA = valid && (ScA >= S_run - A.margin) && (ScA > 0.0f || indexA == 0u);
    const bool candB = validB && (ScB >= S_run - A.margin) && (ScB > 0.0f || indexB == 0u);
    const unsigned balA = __ballot_sync(0xffffffffu, candA), balB = __ballot_sync(0xffffffffu, candB);
    if (balA | balB) {
        unsigned base = 0;
        if (lane == 0) base = (unsigned)atomicAdd(A.counters + CNT_POOL, (unsigned long long)(__popc(balA) + __popc(balB)));
        base = __shfl_sync(0xffffffffu, base, 0);
        const unsigned below = (1u << lane) - 1u;
        if (candA) {
            const unsigned pos = base + __popc(balA & below);
            if (pos < A.pool_cap) { PoolEntry pe; pe.event = (uint32_t)e; pe.index = indexA; pe.S32 = ScA; pe.pad = 0; A.pool[pos] = pe; }
        }
        if (candB) {
            const unsigned pos = base + __popc(balA) + __popc(balB & below);
            if (pos < A.pool_cap) { PoolEntry pe; pe.event = (uint32_t)e; pe.index = indexB; pe.S32 = ScB; pe.pad = 0; A.pool[pos] = pe; }
        }
    }
    const unsigned sn = __reduce_add_sync(0xffffffffu, (valid ? (unsigned)nA : 0u) + (validB ? (unsigned)nB : 0u));
    const unsigned sm = __reduce_add_sync(0xffffffffu, (valid ? (unsigned)fmA : 0u) + (validB ? (unsigned)fmB : 0u));
    const unsigned st = __reduce_add_sync(0xffffffffu, tests);
    const unsigned sl = __reduce_add_sync(0xffffffffu, lookups);
    const unsigned sg = __reduce_add_sync(0xffffffffu, cnt & 0xFFFFu);
    const unsigned sa = __reduce_add_sync(0xffffffffu, cnt >> 16);
    if (lane == 0) {
        atomicAdd(A.counters + CNT_STEPS, (unsigned long long)sn);
        atomicAdd(A.counters + CNT_GAS, (unsigned long long)sm);
        atomicAdd(A.counters + CNT_TESTS, (unsigned long long)st);
        atomicAdd(A.counters + CNT_LOOKUP, (unsigned long long)sl);
        atomicAdd(A.counters + CNT_G1, (unsigned long long)sg);
        atomicAdd(A.counters + CNT_APPROACH, (unsigned long long)sa);
    }
}

}  // namespace

cudaError_t launch_seed_scan_pair(const ScanArgs &A, const ScanLaunch &L, bool eloss, bool track, cudaStream_t s)
{
    dim3 grid((unsigned)((L.max_pairs_per_event + kBlock - 1) / kBlock), (unsigned)L.n_events);
    if (L.fd.kind == 0) {
        if (eloss) seed_scan_pair_kernel<0, true, true><<<grid, kBlock, 0, s>>>(A);
        else if (track) seed_scan_pair_kernel<0, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_pair_kernel<0, false, false><<<grid, kBlock, 0, s>>>(A);
    } else {
        if (eloss) return cudaErrorInvalidValue;                 // routed to the one-seed kernel by the caller
        if (track) seed_scan_pair_kernel<1, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_pair_kernel<1, false, false><<<grid, kBlock, 0, s>>>(A);
    }
    return cudaGetLastError();
}
