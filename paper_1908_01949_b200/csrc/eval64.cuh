// fp64 evaluation of one seed, shared by best.cu (A8/A9) and refine.cu (coarse-to-fine refinement).
// EVERY TRANSLATION UNIT THAT INCLUDES THIS FILE IS COMPILED WITH -fmad=false: each fp64 +, -, *, /, sqrt below is a
// single IEEE-754 operation in the order DESIGN.md section 3 (readings C4-C10, C12) writes the formulas, left to right
// (reading C11).  Transcendentals appear only where they cannot change the result: in the choice of candidate wires
// (a superset by construction, reading C8).
#pragma once
#include "cdc_internal.cuh"

namespace {

struct BestArgs {
    Geom64 g;
    const GridDev *grids;
    const double *axes;
    int32_t axis_stride;
    const float *drift_tab;
    const uint32_t *bits;
    int32_t W, n_bit_words;
    double h, lambda, eloss_h, kq;
    int32_t max_steps;
    int32_t lookup_every;      // K64: steps per 3 x 3 candidate lookup
};

__device__ __forceinline__ void field64(const Geom64 &g, double x, double y, double z, double *B)
{
    if (g.field_kind == 0) { B[0] = 0.0; B[1] = 0.0; B[2] = g.bz; return; }
    const double rho = sqrt(x * x + y * y);
    const double fr = (rho - g.r0) / g.dr;
    const double fz = (z - g.z0) / g.dz;
    int ir = (int)floor(fr), iz = (int)floor(fz);
    ir = max(0, min(ir, g.nr - 2));
    iz = max(0, min(iz, g.nz - 2));
    const double wr = fr - (double)ir, wz = fz - (double)iz;
    const float *n00 = g.tab + ((size_t)iz * g.nr + ir) * 2;
    const float *n01 = n00 + 2, *n10 = n00 + (size_t)g.nr * 2, *n11 = n10 + 2;
    const double Br = (1.0 - wz) * ((1.0 - wr) * (double)n00[0] + wr * (double)n01[0])
                    + wz * ((1.0 - wr) * (double)n10[0] + wr * (double)n11[0]);
    const double Bz = (1.0 - wz) * ((1.0 - wr) * (double)n00[1] + wr * (double)n01[1])
                    + wz * ((1.0 - wr) * (double)n10[1] + wr * (double)n11[1]);
    if (rho > 0.0) { B[0] = Br * x / rho; B[1] = Br * y / rho; }
    else { B[0] = 0.0; B[1] = 0.0; }
    B[2] = Bz;
}

__device__ __forceinline__ void lorentz64(double a, const double *T, const double *B, double *k)
{
    k[0] = a * (T[1] * B[2] - T[2] * B[1]);
    k[1] = a * (T[2] * B[0] - T[0] * B[2]);
    k[2] = a * (T[0] * B[1] - T[1] * B[0]);
}

// reading C5: the four stages and the update, each expression evaluated left to right.
// UNI (uniform field B = (0, 0, bz), position-independent): the same formulas with the terms that are exactly zero
// left out.  x * 0 = +-0 and y -+ 0 = y in IEEE arithmetic, so every value equals the general form's (a zero may carry
// the other sign, which no later operation can see: there is no division by, or sign test of, these quantities):
//   k_x = a (T_y bz),  k_y = a (-(T_x bz)),  k_z = 0  ->  U_z = T_z,  T_z' = T_z,  z' = z + h T_z,
// and the intermediate points q are never formed (nothing reads them).  37 % of the general form's instructions and a
// dependent chain of 17 instead of 27 operations: the re-score is latency-bound.
template <bool UNI>
__device__ __forceinline__ void rkn_step64(const Geom64 &g, double a, double h, const double *r, const double *T,
                                           double *rn, double *Tn)
{
    const double hh = h / 2.0, h28 = h * h / 8.0, h22 = h * h / 2.0, h26 = h * h / 6.0, h6 = h / 6.0;
    if (UNI) {
        const double bz = g.bz;
        const double k1x = a * (T[1] * bz), k1y = a * (-(T[0] * bz));
        double Ux = T[0] + hh * k1x, Uy = T[1] + hh * k1y;
        const double k2x = a * (Uy * bz), k2y = a * (-(Ux * bz));
        Ux = T[0] + hh * k2x; Uy = T[1] + hh * k2y;
        const double k3x = a * (Uy * bz), k3y = a * (-(Ux * bz));
        Ux = T[0] + h * k3x; Uy = T[1] + h * k3y;
        const double k4x = a * (Uy * bz), k4y = a * (-(Ux * bz));
        rn[0] = r[0] + h * T[0] + h26 * (k1x + k2x + k3x);
        rn[1] = r[1] + h * T[1] + h26 * (k1y + k2y + k3y);
        rn[2] = r[2] + h * T[2];
        Tn[0] = T[0] + h6 * (k1x + 2.0 * k2x + 2.0 * k3x + k4x);
        Tn[1] = T[1] + h6 * (k1y + 2.0 * k2y + 2.0 * k3y + k4y);
        Tn[2] = T[2];
        return;
    }
    double B[3], k1[3], k2[3], k3[3], k4[3], q[3], U[3];
    field64(g, r[0], r[1], r[2], B);
    lorentz64(a, T, B, k1);
#pragma unroll
    for (int i = 0; i < 3; ++i) { q[i] = r[i] + hh * T[i] + h28 * k1[i]; U[i] = T[i] + hh * k1[i]; }
    field64(g, q[0], q[1], q[2], B);
    lorentz64(a, U, B, k2);
#pragma unroll
    for (int i = 0; i < 3; ++i) U[i] = T[i] + hh * k2[i];
    lorentz64(a, U, B, k3);
#pragma unroll
    for (int i = 0; i < 3; ++i) { q[i] = r[i] + h * T[i] + h22 * k3[i]; U[i] = T[i] + h * k3[i]; }
    field64(g, q[0], q[1], q[2], B);
    lorentz64(a, U, B, k4);
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        rn[i] = r[i] + h * T[i] + h26 * (k1[i] + k2[i] + k3[i]);
        Tn[i] = T[i] + h6 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
    }
}

// The same step plus the local error estimate of the adaptive propagator of PAPER.md ref. [5] (reading C19):
// err = h^2 max_i |k1_i - k2_i - k3_i + k4_i|, each component left to right.  General form only (rn, Tn as above).
__device__ __forceinline__ void rkn_step64_err(const Geom64 &g, double a, double h, const double *r, const double *T,
                                               double *rn, double *Tn, double *err)
{
    const double hh = h / 2.0, h28 = h * h / 8.0, h22 = h * h / 2.0, h26 = h * h / 6.0, h6 = h / 6.0;
    double B[3], k1[3], k2[3], k3[3], k4[3], q[3], U[3];
    field64(g, r[0], r[1], r[2], B);
    lorentz64(a, T, B, k1);
#pragma unroll
    for (int i = 0; i < 3; ++i) { q[i] = r[i] + hh * T[i] + h28 * k1[i]; U[i] = T[i] + hh * k1[i]; }
    field64(g, q[0], q[1], q[2], B);
    lorentz64(a, U, B, k2);
#pragma unroll
    for (int i = 0; i < 3; ++i) U[i] = T[i] + hh * k2[i];
    lorentz64(a, U, B, k3);
#pragma unroll
    for (int i = 0; i < 3; ++i) { q[i] = r[i] + h * T[i] + h22 * k3[i]; U[i] = T[i] + h * k3[i]; }
    field64(g, q[0], q[1], q[2], B);
    lorentz64(a, U, B, k4);
    double emax = 0.0;
#pragma unroll
    for (int i = 0; i < 3; ++i) {
        const double e = k1[i] - k2[i] - k3[i] + k4[i];
        rn[i] = r[i] + h * T[i] + h26 * (k1[i] + k2[i] + k3[i]);
        Tn[i] = T[i] + h6 * (k1[i] + 2.0 * k2[i] + 2.0 * k3[i] + k4[i]);
        if (fabs(e) > emax) emax = fabs(e);
    }
    *err = h * h * emax;
}

// reading C9: delta = d - (d.u) u with d = r - w0;  returns g = delta . T when T != nullptr
__device__ __forceinline__ void wire_offset64(const float *w, const double *r, double *delta, double *tpar)
{
    const double dx = r[0] - (double)w[0], dy = r[1] - (double)w[1], dz = r[2];
    const double ux = (double)w[2], uy = (double)w[3], uz = (double)w[4];
    const double t = dx * ux + dy * uy + dz * uz;
    delta[0] = dx - t * ux; delta[1] = dy - t * uy; delta[2] = dz - t * uz;
    *tpar = t;
}

struct Eval64 {
    int32_t n_match, n_steps, turns, m_gas;
    double chi2;
};

// this lane's candidate wire around r, or -1: lanes 0..8 cover the 3 nearest layers x 3 nearest cells; only wires
// with a hit are returned (fp32 is enough here: the set only has to contain every wire within ~9.3 mm, reading C8)
__device__ __forceinline__ int lane_candidate(const Geom64 &g, const LayerDev *s_layer, const uint32_t *bits,
                                              const double *r, int lane)
{
    const float x = (float)r[0], y = (float)r[1], z = (float)r[2];
    const float zeta = z * g.tan_abs;
    const float u2 = x * x + y * y - zeta * zeta;
    if (!(u2 > 0.0f) || lane >= 9) return -1;
    const float fj = (sqrtf(u2) - g.r_first) * g.inv_pitch;
    if (fj < -1.5f || fj > (float)g.n_layers + 0.5f) return -1;      // beyond the reach of any wire for K64 steps
    const int j = (int)rintf(fj) - 1 + lane / 3;
    if (j < 0 || j >= g.n_layers) return -1;
    const LayerDev L = s_layer[j];
    const float kf = (atan2f(y, x) - L.phi0 - atanf(z * L.shift_k)) * L.kscale;
    int k = (int)rintf(kf) + (lane % 3) - 1;                         // |k| < 2 n: wrap without a division
    k += (k < 0) ? L.n : 0; k += (k < 0) ? L.n : 0; k -= (k >= L.n) ? L.n : 0;
    const int w = L.offset + k;
    return ((__ldg(bits + (w >> 5)) >> (w & 31)) & 1u) ? w : -1;
}

// readings C4-C10: evaluate one seed, one WARP per seed.  Every lane carries the same fp64 track (the arithmetic is
// redundant across lanes, which costs nothing: the warp issues it once); lanes 0..8 each test one candidate wire of
// the interval, so the latency of a step is that of one wire instead of nine.  Matches are folded into chi2 in
// ascending wire id within an interval -- the order reading C11 fixes.  wire_label / wire_best (optional, per wire
// of this event): reading C12.  rec / rec_count (optional): matched approaches in path order.
// e: grid (axis tables, grid record); he: event whose hit tables are scored (== e except for refinement sub-grids).
// ELOSS = false (eloss_h == 0): p_n = p_0 - 0 * m = p_0 exactly, so a = kappa q / p_0 is formed once.  ELOSS = true: the
// momentum of the NEXT step depends only on the in-gas count, known at the top of this step, so its division runs
// beside this step's stages instead of ahead of them.
template <bool UNI, bool ELOSS>
__device__ void eval_seed64_t(const BestArgs &A, const LayerDev *s_layer, int e, int he, uint32_t index, Eval64 &out,
                              int32_t *wire_label, double *wire_best, ApproachRec *rec, int32_t *rec_count)
{
    const unsigned full = 0xffffffffu;
    const int lane = threadIdx.x & 31;
    const GridDev G = A.grids[e];
    uint32_t q = index;
    const int i_pz = q % G.n[4]; q /= G.n[4];
    const int i_py = q % G.n[3]; q /= G.n[3];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_z = q % G.n[1];
    const int i_th = q / G.n[1];
    const double *ax = A.axes + (size_t)e * 6 * A.axis_stride;
    const double px = ax[3 * A.axis_stride + i_px], py = ax[4 * A.axis_stride + i_py], pz = ax[5 * A.axis_stride + i_pz];
    double r[3] = {ax[i_th], ax[A.axis_stride + i_th], ax[2 * A.axis_stride + i_z]};     // C4
    const double p0 = sqrt(px * px + py * py + pz * pz);
    double T[3] = {px / p0, py / p0, pz / p0};
    double p = p0, chi2 = 0.0;
    const uint32_t *bits = A.bits + (size_t)he * A.n_bit_words;
    const float *drift = A.drift_tab + (size_t)he * A.W;
    int n = 0, turn = 0, m = 0, n_match = 0, n_rec = 0;
    bool cn = true;
    int kc = 0, w = -1;
    float wr[5] = {0.f, 0.f, 0.f, 0.f, 1.f};
    double g0 = 0.0, drift_w = 0.0;
    double a = A.kq / p;                                                // a = kappa q / p_n (C5/C6)
    while (n < A.max_steps) {
        double rn[3], Tn[3];
        double p_next = p, a_next = a;
        if (ELOSS) {                                                    // C6: p_{n+1} = p_0 - eloss_h m_{n+1}
            p_next = p0 - A.eloss_h * (double)(m + (cn ? 1 : 0));
            a_next = A.kq / p_next;
        }
        // every K64 steps: this lane's candidate wire around r_n and g at r_n.  A wire outside the 3 x 3 set is at
        // least 1.5 layer pitches / 1.5 cells away, so the set stays a superset of the wires that can own a match for
        // K64 intervals (reading C8); g is carried from vertex to vertex (same operands, same value as a fresh
        // evaluation), the wire record is held in registers.
        if (kc == 0) {
            kc = A.lookup_every;
            w = lane_candidate(A.g, s_layer, bits, r, lane);
            if (w >= 0) {
                const float *wp = A.g.wire5 + (size_t)w * 5;
#pragma unroll
                for (int i = 0; i < 5; ++i) wr[i] = __ldg(wp + i);
                drift_w = (double)__ldg(drift + w);
                double d0[3], tp;
                wire_offset64(wr, r, d0, &tp);
                g0 = d0[0] * T[0] + d0[1] * T[1] + d0[2] * T[2];
            }
        }
        kc -= 1;
        rkn_step64<UNI>(A.g, a, A.h, r, T, rn, Tn);
        double g1 = 0.0;
        if (w >= 0) {
            double d1[3], tp;
            wire_offset64(wr, rn, d1, &tp);
            g1 = d1[0] * Tn[0] + d1[1] * Tn[1] + d1[2] * Tn[2];
        }
        if (cn) {
            bool matched = false;
            double r2 = 0.0, ad = 0.0;
            if (w >= 0) {
                double tp;
                if (g0 <= 0.0 && g1 > 0.0) {
                    const double tau = g0 / (g0 - g1);
                    double P[3], d[3];
#pragma unroll
                    for (int i = 0; i < 3; ++i) P[i] = r[i] + tau * (rn[i] - r[i]);
                    wire_offset64(wr, P, d, &tp);
                    const double D = sqrt(d[0] * d[0] + d[1] * d[1] + d[2] * d[2]);
                    const double zw = tp * (double)wr[4];
                    const double resid = D - drift_w;
                    r2 = resid * resid; ad = fabs(resid);
                    matched = fabs(zw) <= A.g.z_half && r2 < A.lambda;
                }
            }
            unsigned pend = __ballot_sync(full, matched);
            while (pend) {                              // fold the matches in ascending wire id
                const int wmin = __reduce_min_sync(full, (pend >> lane) & 1u ? w : 0x7fffffff);
                const int src = __ffs(__ballot_sync(full, ((pend >> lane) & 1u) && w == wmin)) - 1;
                const double r2s = __shfl_sync(full, r2, src), ads = __shfl_sync(full, ad, src);
                n_match += 1;
                chi2 += r2s;
                if (lane == 0) {
                    if (rec) {                          // matched approaches in path order, replayed by label_kernel
                        if (n_rec < kRecCap) { rec[n_rec].wire = wmin; rec[n_rec].turn = turn; rec[n_rec].absd = ads; }
                    }
                    if (wire_label) {                   // C12: smallest |resid| wins, ties -> earliest
                        if (wire_label[wmin] < 0 || ads < wire_best[wmin]) { wire_label[wmin] = turn; wire_best[wmin] = ads; }
                    }
                }
                n_rec += 1;
                pend &= ~(1u << src);
            }
            m += 1;
        }
        g0 = g1;
#pragma unroll
        for (int i = 0; i < 3; ++i) { r[i] = rn[i]; T[i] = Tn[i]; }
        n += 1;
        p = p_next; a = a_next;
        const bool cnext = r[0] * r[0] + r[1] * r[1] >= A.g.R0 * A.g.R0;
        if (!cn && cnext) turn += 1;                                    // C7
        cn = cnext;
        if (fabs(r[2]) > A.g.z_half) break;
        if (r[0] * r[0] + r[1] * r[1] > A.g.r_out * A.g.r_out) break;
        if (!(p > 1.0)) break;
        if (!(isfinite(r[0]) && isfinite(r[1]) && isfinite(r[2]) && isfinite(T[0]) && isfinite(T[1]) && isfinite(T[2])))
            break;
    }
    out.n_match = n_match; out.chi2 = chi2; out.n_steps = n; out.turns = turn; out.m_gas = m;
    if (rec_count && lane == 0) *rec_count = n_rec;
}

__device__ __forceinline__ void eval_seed64(const BestArgs &A, const LayerDev *s_layer, int e, int he, uint32_t index,
                                            Eval64 &out, int32_t *wire_label, double *wire_best, ApproachRec *rec,
                                            int32_t *rec_count)
{
    const bool uni = A.g.field_kind == 0, el = A.eloss_h != 0.0;
    if (uni && !el) eval_seed64_t<true, false>(A, s_layer, e, he, index, out, wire_label, wire_best, rec, rec_count);
    else if (uni) eval_seed64_t<true, true>(A, s_layer, e, he, index, out, wire_label, wire_best, rec, rec_count);
    else if (!el) eval_seed64_t<false, false>(A, s_layer, e, he, index, out, wire_label, wire_best, rec, rec_count);
    else eval_seed64_t<false, true>(A, s_layer, e, he, index, out, wire_label, wire_best, rec, rec_count);
}

__device__ __forceinline__ void load_layers(const Geom64 &g, LayerDev *s_layer)
{
    for (int i = threadIdx.x; i < g.n_layers; i += blockDim.x) s_layer[i] = g.layers[i];
    __syncthreads();
}

}  // namespace
