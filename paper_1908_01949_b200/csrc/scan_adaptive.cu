// the seed scan with the ADAPTIVE step of the propagator the paper cites ("the RKN method
// was used for the track parameter propagation [5]"; [5] = Lund et al.), reading C19 applied to the scan.
//
// Step lengths h 2^j, j = 0 .. J (h 2^J <= h_max).  A trial of length H = h 2^j has the error estimate of ref. [5],
// err = H^2 max_i |k1 - k2 - k3 + k4|_i; err > tol and j > 0 -> the trial is repeated one level down; after an accepted
// step with err <= tol / 32 the next trial starts one level up.  Path, the step cap and the in-gas count are in units
// of h; p = p0 - eps h m.  Scoring (ownership by the sign change of g over the interval, chord interpolation, window,
// turn counter, termination) is readings C7-C10 unchanged.  One thread per seed, fp32 with compensated state like the
// fixed-step kernel (scan.cu); all step constants of level j are those of level 0 times 2^j or 4^j (exact).
//
// What differs from the fixed-step kernel by construction: the step-size DECISIONS are taken in fp32 here and in fp64
// by the oracle, and a different decision changes every later vertex.  The estimate is a small difference of the four
// stage derivatives (relative size ~ (|a| B H)^2), good to ~1 % in fp32, so a seed whose oracle-side estimate comes
// within 2 % of tol or of tol / 32 at a decision may legitimately take another sequence: such seeds are an explicit
// exception class of the parity protocol (tests/test_gpu_adaptive.py lists and counts them); all other seeds must
// take the identical level sequence (compared through a hash), and then positions and match counts obey the usual bars.
//
// Wire lookup: every step, around the step's start vertex (a step may be as long as h_max, so the fixed-step kernel's
// K-step cadence does not apply); the 2 x 2 candidate set covers every wire within reach(h_max) of the vertex (host
// check).  g is evaluated at both ends of the interval for the candidates that carry a hit.
#include <math.h>

#include <algorithm>

#include "cdc_internal.cuh"
#include "scan_common.cuh"
#include "scan_args.cuh"

namespace {

struct AdaptiveArgs {
    ScanArgs S;
    float tol, tol_up;          // tol, tol / 32
    int32_t J;                  // highest level
    int32_t *levels;            // optional [seeds][8]: accepted steps per level (0..6) and, in [7], the sequence hash
};

__device__ __forceinline__ void cells_of_layer(const ScanArgs &A, const LayerDev *s_layer, int j, float phi, float z, int &ca, int &cb)
{
    ca = -1; cb = -1;
    if ((unsigned)j >= (unsigned)A.gd.n_layers) return;
    const LayerDev L = s_layer[j];
    const float tau = z * L.shift_k;
    const float sh = fmaf(-0.333333343f * tau * tau, tau, tau);
    const float kf = (phi - L.phi0 - sh) * L.kscale;
    const float kn = rintf(kf);
    int k1 = (int)kn;
    int k2 = k1 + ((kf - kn) >= 0.0f ? 1 : -1);
    k1 += (k1 < 0) ? L.n : 0; k1 += (k1 < 0) ? L.n : 0; k1 -= (k1 >= L.n) ? L.n : 0;
    k2 += (k2 < 0) ? L.n : 0; k2 += (k2 < 0) ? L.n : 0; k2 -= (k2 >= L.n) ? L.n : 0;
    ca = L.offset + k1; cb = L.offset + k2;
}

template <int FIELD>
__global__ void __launch_bounds__(kBlock) seed_scan_adaptive_kernel(const AdaptiveArgs P)
{
    const ScanArgs &A = P.S;
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    __shared__ uint32_t s_bits[kMaxBitWords];
    const int e = blockIdx.y;
    const GridDev G = A.grids[e];
    if ((int64_t)blockIdx.x * kBlock >= (int64_t)G.n_seeds) return;
    for (int i = threadIdx.x; i < A.gd.n_layers; i += kBlock) s_layer[i] = A.gd.layers[i];
    for (int i = threadIdx.x; i < A.gd.n_bit_words; i += kBlock) s_bits[i] = A.bits[(size_t)e * A.gd.n_bit_words + i];
    __syncthreads();
    const float *drift_e = A.drift_tab + (size_t)e * A.gd.n_wires_total;

    // thread -> seed: z0 lane-fastest, as in the fixed-step kernel
    const int t = blockIdx.x * kBlock + threadIdx.x;
    const bool valid = t < G.n_seeds;
    int q = valid ? t : 0;
    const int i_z = q % G.n[1]; q /= G.n[1];
    const int i_th = q % G.n[0]; q /= G.n[0];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_py = q % G.n[3];
    const int i_pz = q / G.n[3];
    const uint32_t index = (uint32_t)((((i_th * G.n[1] + i_z) * G.n[2] + i_px) * G.n[3] + i_py) * G.n[4] + i_pz);

    float xh, xl, yh, yl, zh, zl, Txh, Txl, Tyh, Tyl, Tzh, Tzl, a, epsT, p0h, p0l;
    const bool eloss = A.eloss_h != 0.0f;
    {
        const double *ax = A.axes + (size_t)e * 6 * A.axis_stride;
        const double x0 = ax[i_th], y0 = ax[A.axis_stride + i_th], z0 = ax[2 * A.axis_stride + i_z];
        const double px = ax[3 * A.axis_stride + i_px], py = ax[4 * A.axis_stride + i_py], pz = ax[5 * A.axis_stride + i_pz];
        const double p0 = sqrt(px * px + py * py + pz * pz);
        const double tx = px / p0, ty = py / p0, tz = pz / p0;
        xh = (float)x0; xl = (float)(x0 - (double)xh);
        yh = (float)y0; yl = (float)(y0 - (double)yh);
        zh = (float)z0; zl = (float)(z0 - (double)zh);
        Txh = (float)tx; Txl = (float)(tx - (double)Txh);
        Tyh = (float)ty; Tyl = (float)(ty - (double)Tyh);
        Tzh = (float)tz; Tzl = (float)(tz - (double)Tzh);
        const double a64 = A.kq / p0;
        a = (float)a64;
        epsT = (float)((a64 * A.h6_64) / ((double)a * (double)A.h_6) - 1.0);
        if (eloss) epsT = (float)((A.kq * A.h6_64) / ((double)(float)A.kq * (double)A.h_6) - 1.0);
        p0h = (float)p0; p0l = (float)(p0 - (double)p0h);
    }
    const int cap = !valid ? 0 : ((p0h > 1.0f) ? A.max_steps : min(A.max_steps, 1));     // path cap in units of h

    uint32_t nm = 0, hash = 0;
    float chi2 = 0.0f;
    int n = 0, units = 0, m = 0, turn = 0, j = 0;
    int lev[7] = {0, 0, 0, 0, 0, 0, 0};
    bool cn = true;                                   // c_0 := true (reading C7)

#pragma unroll 1
    while (units < cap) {
        while (j > 0 && units + (1 << j) > cap) --j;                  // the path cap: the last steps drop levels until they fit
        // ---- candidate wires of this interval: the 2 x 2 set around the start vertex, those that carry a hit
        int c0 = -1, c1 = -1, c2 = -1, c3 = -1;
        float g00 = 0.f, g01 = 0.f, g02 = 0.f, g03 = 0.f;
        if (cn) {
            const float zeta = zh * A.gd.tan_abs;
            const float u2 = fmaf(xh, xh, fmaf(yh, yh, -zeta * zeta));
            if (u2 > A.u2_lo && u2 < A.u2_hi) {
                const float u = u2 * rsqrt_normal(u2);
                const float fj = (u - A.gd.r_first) * A.gd.inv_pitch;
                const float jn = rintf(fj);
                const int jc = (int)jn;
                const int j2 = jc + ((fj - jn) >= 0.0f ? 1 : -1);
                const float phi = coarse_atan2(yh, xh);
                cells_of_layer(A, s_layer, jc, phi, zh, c0, c1);
                cells_of_layer(A, s_layer, j2, phi, zh, c2, c3);
                float ex, ey, eu;
                if (c0 >= 0 && ((s_bits[c0 >> 5] >> (c0 & 31)) & 1u)) g00 = wire_g(__ldg(A.gd.wire4 + c0), A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex, ey, eu); else c0 = -1;
                if (c1 >= 0 && ((s_bits[c1 >> 5] >> (c1 & 31)) & 1u)) g01 = wire_g(__ldg(A.gd.wire4 + c1), A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex, ey, eu); else c1 = -1;
                if (c2 >= 0 && ((s_bits[c2 >> 5] >> (c2 & 31)) & 1u)) g02 = wire_g(__ldg(A.gd.wire4 + c2), A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex, ey, eu); else c2 = -1;
                if (c3 >= 0 && ((s_bits[c3 >> 5] >> (c3 & 31)) & 1u)) g03 = wire_g(__ldg(A.gd.wire4 + c3), A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex, ey, eu); else c3 = -1;
            }
        }

        // ---- A4: trial steps of length H = h 2^j until the estimate passes (or j = 0)
        float Bx, By, Bz, k1x, k1y, k1z;
        field_at<FIELD>(A.fd, xh, yh, zh, Bx, By, Bz);                 // the first stage does not depend on H
        k1x = a * fmaf(Tyh, Bz, -Tzh * By); k1y = a * fmaf(Tzh, Bx, -Txh * Bz); k1z = a * fmaf(Txh, By, -Tyh * Bx);
        float sdx, sdy, sdz, dTx, dTy, dTz, err, H;
#pragma unroll 1
        for (;;) {
            const float s1 = (float)(1 << j), s2 = s1 * s1;            // exact scalings of the level-0 constants
            H = A.h * s1;
            const float h_half = A.h_half * s1, h2_8 = A.h2_8 * s2, h2_2 = A.h2_2 * s2, h_6 = A.h_6 * s1, h2_6 = A.h2_6 * s2;
            float Ux = fmaf(h_half, k1x, Txh), Uy = fmaf(h_half, k1y, Tyh), Uz = fmaf(h_half, k1z, Tzh);
            field_at<FIELD>(A.fd, fmaf(h2_8, k1x, fmaf(h_half, Txh, xh)), fmaf(h2_8, k1y, fmaf(h_half, Tyh, yh)),
                            fmaf(h2_8, k1z, fmaf(h_half, Tzh, zh)), Bx, By, Bz);
            const float k2x = a * fmaf(Uy, Bz, -Uz * By), k2y = a * fmaf(Uz, Bx, -Ux * Bz), k2z = a * fmaf(Ux, By, -Uy * Bx);
            Ux = fmaf(h_half, k2x, Txh); Uy = fmaf(h_half, k2y, Tyh); Uz = fmaf(h_half, k2z, Tzh);
            const float k3x = a * fmaf(Uy, Bz, -Uz * By), k3y = a * fmaf(Uz, Bx, -Ux * Bz), k3z = a * fmaf(Ux, By, -Uy * Bx);
            Ux = fmaf(H, k3x, Txh); Uy = fmaf(H, k3y, Tyh); Uz = fmaf(H, k3z, Tzh);
            field_at<FIELD>(A.fd, fmaf(h2_2, k3x, fmaf(H, Txh, xh)), fmaf(h2_2, k3y, fmaf(H, Tyh, yh)),
                            fmaf(h2_2, k3z, fmaf(H, Tzh, zh)), Bx, By, Bz);
            const float k4x = a * fmaf(Uy, Bz, -Uz * By), k4y = a * fmaf(Uz, Bx, -Ux * Bz), k4z = a * fmaf(Ux, By, -Uy * Bx);
            // error estimate of ref. [5], each component left to right
            const float ex_ = fabsf(((k1x - k2x) - k3x) + k4x), ey_ = fabsf(((k1y - k2y) - k3y) + k4y), ez_ = fabsf(((k1z - k2z) - k3z) + k4z);
            err = (H * H) * fmaxf(ex_, fmaxf(ey_, ez_));
            if (err > P.tol && j > 0) { --j; continue; }
            const float dx = fmaf(h2_6, (k1x + k2x) + k3x, H * Txh), dy = fmaf(h2_6, (k1y + k2y) + k3y, H * Tyh),
                        dz = fmaf(h2_6, (k1z + k2z) + k3z, H * Tzh);
            dTx = h_6 * fmaf(2.0f, k2x + k3x, k1x + k4x); dTy = h_6 * fmaf(2.0f, k2y + k3y, k1y + k4y);
            dTz = h_6 * fmaf(2.0f, k2z + k3z, k1z + k4z);
            sdx = fmaf(H, Txl, dx); sdy = fmaf(H, Tyl, dy); sdz = fmaf(H, Tzl, dz);
            break;
        }
        comp_add(xh, xl, sdx);
        comp_add(yh, yl, sdy);
        comp_add(zh, zl, sdz);
        comp_add(Txh, Txl, fmaf(dTx, epsT, dTx));
        comp_add(Tyh, Tyl, fmaf(dTy, epsT, dTy));
        comp_add(Tzh, Tzl, fmaf(dTz, epsT, dTz));

        // ---- A6: the interval's approaches (reading C9): g at the far vertex for the candidates that carry a hit
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const int w = i == 0 ? c0 : i == 1 ? c1 : i == 2 ? c2 : c3;
            const float g = i == 0 ? g00 : i == 1 ? g01 : i == 2 ? g02 : g03;
            if (w < 0 || !(g <= 0.0f)) continue;
            const float4 wr = __ldg(A.gd.wire4 + w);
            float ex1, ey1, eu1;
            const float gn = wire_g(wr, A.uz, A.inv_uz, xh, xl, yh, yl, zh, Txh, Tyh, Tzh, ex1, ey1, eu1);
            if (!(gn > 0.0f)) continue;
            const float zd = sdz * A.inv_uz;
            const float dex = fmaf(-zd, wr.z, sdx), dey = fmaf(-zd, wr.w, sdy);
            const float sm = __fdividef(g, g - gn) - 1.0f;
            const float ex = fmaf(sm, dex, ex1), ey = fmaf(sm, dey, ey1);
            const float eu = fmaf(ex, wr.z, ey * wr.w);
            const float D = sqrtf(fmaxf(fmaf(ex, ex, fmaf(ey, ey, -eu * eu)), 0.0f));
            const float zw = fmaf(eu, A.uz, fmaf(sm, sdz, zh));
            const float resid = D - __ldg(drift_e + w);
            const float r2 = resid * resid;
            if (fabsf(zw) <= A.gd.z_half && r2 < A.lambda) { nm += 1u; chi2 += r2; }
        }
        if (cn) m += 1 << j;

        // ---- advance: path, level statistics, energy loss, turn counter, termination (readings C6, C7)
        n += 1; units += 1 << j;
        lev[j < 7 ? j : 6] += 1;
        hash = hash * 31u + (uint32_t)(j + 1);
        const float rho2 = fmaf(xh, xh, yh * yh);
        const bool cnext = rho2 >= A.gd.R0sq;
        if (!cn && cnext) turn += 1;
        cn = cnext;
        if (eloss) {
            const float p = fmaf(-A.eloss_h, (float)m, p0h) + p0l;
            a = (float)A.kq / p;
            if (!(p > 1.0f)) break;
        }
        if (!(fabsf(zh) <= A.gd.z_half)) break;
        if (!(rho2 <= A.gd.r_out_sq)) break;
        if (j < P.J && err <= P.tol_up) ++j;
    }

    // ---- per-seed output and the fused fp32 arg max (no candidate pool: the exact re-score of this variant is not built)
    const float Sc = valid ? fmaxf(fmaf(-chi2, A.inv_lambda, (float)nm), 0.0f) : 0.0f;
    if (valid) {
        const int64_t o = G.out_offset + (int64_t)index;
        if (A.n_match) A.n_match[o] = nm;
        if (A.chi2) A.chi2[o] = chi2;
        if (A.debug) {
            cdc_seed_debug d;
            d.n_steps = n; d.turns = turn; d.m_gas = m; d.pad = units;
            d.x = (double)xh + (double)xl; d.y = (double)yh + (double)yl; d.z = (double)zh + (double)zl;
            A.debug[o] = d;
        }
        if (P.levels) {
            for (int i = 0; i < 7; ++i) P.levels[8 * o + i] = lev[i];
            P.levels[8 * o + 7] = (int32_t)hash;
        }
    }
    const unsigned long long key = valid ? (((unsigned long long)__float_as_uint(Sc) << 32) | (0xFFFFFFFFu - index)) : 0ull;
    const unsigned long long wkey = warp_max_u64(key);
    if ((threadIdx.x & 31) == 0) atomicMax(A.best_key + e, wkey);
    const unsigned sn = __reduce_add_sync(0xffffffffu, valid ? (unsigned)n : 0u);
    const unsigned su = __reduce_add_sync(0xffffffffu, valid ? (unsigned)units : 0u);
    if ((threadIdx.x & 31) == 0) {
        atomicAdd(A.counters + CNT_STEPS, (unsigned long long)sn);
        atomicAdd(A.counters + CNT_GAS, (unsigned long long)su);          // path units (this variant's second counter)
    }
}

}  // namespace

cudaError_t launch_seed_scan_adaptive(const ScanLaunch &L, double tol, int J, int32_t *d_levels, cudaStream_t s, cudaEvent_t k0,
                                      cudaEvent_t k1)
{
    AdaptiveArgs P;
    ScanArgs &A = P.S;
    A.gd = L.gd; A.fd = L.fd; A.grids = L.d_grids; A.axes = L.d_axes; A.axis_stride = L.axis_stride;
    A.drift_tab = L.d_drift_tab; A.bits = L.d_bits;
    const double h = L.h64;
    A.h = (float)h; A.h_half = (float)(h / 2.0); A.h2_8 = (float)(h * h / 8.0); A.h2_2 = (float)(h * h / 2.0);
    A.h_6 = (float)(h / 6.0); A.h2_6 = (float)(h * h / 6.0);
    A.kq = CDC_KAPPA * (double)L.charge; A.h6_64 = h / 6.0;
    A.kq_rel = (float)(A.kq / (double)(float)A.kq - 1.0);
    A.lambda = L.lambda; A.inv_lambda = 1.0f / L.lambda; A.eloss_h = L.eloss_h; A.window = sqrtf(L.lambda) * 1.0001f;
    A.u2_lo = L.u2_lo; A.u2_hi = L.u2_hi; A.uz = L.uz; A.inv_uz = L.inv_uz;
    A.max_steps = L.max_steps; A.margin = L.margin;
    A.n_match = L.d_n_match; A.chi2 = L.d_chi2; A.debug = L.d_debug;
    A.best_key = (unsigned long long *)L.d_best_key; A.pool = nullptr; A.pool_cap = 0; A.counters = L.d_counters;
    A.lookup_every = 1; A.lookup_every_tight = 1; A.lookahead = 0.f; A.tight_curv = 0.f;
    A.delta_max = L.delta_max; A.b_max = L.b_max; A.hold_path = L.hold_path;
    A.k_margin = A.k_margin0 = A.sin_eps = A.sep_cap = 0.f; A.two_inv_h = A.inv_h = 0.f;
    P.tol = (float)tol; P.tol_up = (float)(tol / 32.0); P.J = J; P.levels = d_levels;
    if (L.gd.n_bit_words > kMaxBitWords || L.gd.n_layers > CDC_MAX_LAYERS) return cudaErrorInvalidValue;
    dim3 grid((unsigned)((L.max_seeds_per_event + kBlock - 1) / kBlock), (unsigned)L.n_events);
    if (k0) cudaEventRecord(k0, s);
    if (L.fd.kind == 0) seed_scan_adaptive_kernel<0><<<grid, kBlock, 0, s>>>(P);
    else seed_scan_adaptive_kernel<1><<<grid, kBlock, 0, s>>>(P);
    if (k1) cudaEventRecord(k1, s);
    cdc_count_launch();
    return cudaGetLastError();
}
