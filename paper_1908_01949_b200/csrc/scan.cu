// A3-A7: the RKN propagate-and-score kernel with fused per-event argmax and candidate pool.
//
// One thread per seed (BJ north_star); the Nystroem-RK4 state lives in registers.  Arithmetic is fp32
// FMA chains; the six state components are carried as (hi, lo) pairs with a Kahan-compensated update so
// that the position after thousands of steps stays within the 1e-3 mm parity bound.
//
//   PAPER.md:51      seed (theta0, z0, px0, py0, pz0) at R0                     -> kernel prologue
//   PAPER.md:55      RKN propagation (textbook Nystroem scheme, reading C5)     -> step body
//   PAPER.md:55,:69  DCA to fired wires, sign-change ownership (reading C9)     -> wire_g(), slot_step()
//   PAPER.md:65-69   Eq. (1): S = sum (1 - d^2/lambda) over matched terms       -> kernel epilogue
//   PAPER.md:69      lowest E (= highest S) wins                                -> packed-key atomicMax
//
// Scoring structure: the layer/cell lookup runs once every K steps around the middle of the next K steps (K from
// the step size: the 2 x 2 candidate set of that point stays a superset of the wires that can own an approach for
// K intervals, reading C8); the candidates that carry a hit are compacted into up to four per-thread slots (wire
// id + g at the current vertex), so each step evaluates g once per live wire and runs the approach code only on a
// sign change.  Lanes of a warp are seeds that differ in z0 first: they cross the same wires together.
#include "cdc_internal.cuh"
#include "scan_common.cuh"
#include "scan_args.cuh"
#include "pair_math.cuh"
#include "scan_one.cuh"

namespace {

// TRACK: keep the in-gas flag, the in-gas step count and the turn counter.  They are needed with energy loss (p_n is
// defined through m_n), for the debug record, and when a held wire could be scored from a vertex inside R0; otherwise
// every vertex a wire can be scored from lies in the gas (host check in launch_seed_scan) and they are dead weight.
#ifndef SCAN_UNROLL
#define SCAN_UNROLL 2
#endif
constexpr int kScanUnroll = SCAN_UNROLL;     // main loop unroll factor
#ifndef SCAN_MB0
#define SCAN_MB0 8           // resident blocks per SM the uniform-field variants are held to (64 registers)
#endif
#ifndef SCAN_MB1
#define SCAN_MB1 0
#endif
template <int FIELD, bool ELOSS, bool TRACK>
__global__ void __launch_bounds__(kBlock, FIELD == 0 ? SCAN_MB0 : SCAN_MB1) seed_scan_kernel(const ScanArgs A)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    __shared__ uint32_t s_bits[kMaxBitWords];

    const int e = blockIdx.y;
    const GridDev G = A.grids[e];
    if ((int64_t)blockIdx.x * kBlock >= (int64_t)G.n_seeds) return;
    for (int i = threadIdx.x; i < A.gd.n_layers; i += kBlock) s_layer[i] = A.gd.layers[i];
    for (int i = threadIdx.x; i < A.gd.n_bit_words; i += kBlock)
        s_bits[i] = A.bits[(size_t)e * A.gd.n_bit_words + i];
    __syncthreads();
    const float *drift_e = A.drift_tab + (size_t)e * A.gd.n_wires_total;

    // ---- A3: thread -> seed.  z0 is the lane-fastest axis, then theta, px, py, pz.  Seeds that differ only in z0 have
    // the same (x, y) path up to the field's z dependence, so the 32 tracks of a warp pass the same wires within a
    // step or two of one another: lookups, live-wire slots and approach code run with most lanes active.  They leave
    // the chamber a few tens of steps apart (the z0 pitch over T_z h), a ~4 % tail.
    const int t = blockIdx.x * kBlock + threadIdx.x;
    const bool valid = t < G.n_seeds;
    int q = valid ? t : 0;
    const int i_z = q % G.n[1]; q /= G.n[1];
    const int i_th = q % G.n[0]; q /= G.n[0];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_py = q % G.n[3];
    const int i_pz = q / G.n[3];
    const uint32_t index = (uint32_t)((((i_th * G.n[1] + i_z) * G.n[2] + i_px) * G.n[3] + i_py) * G.n[4] + i_pz);

    // state: (x, y) and (Tx, Ty) as packed pairs (one FFMA2 / FADD2 serves both components), z and Tz scalar; every
    // component hi + lo (compensated)
    f2 xyh, xyl, Txyh, Txyl;
    float zh, zl, Tzh, Tzl, a, epsT, p0h, p0l;
    float ub_h = 0.f, ub_l = 0.f, ue1 = 0.f, up1 = 0.f, up2_h = 0.f, up2_l = 0.f;   // uniform-field step map (FIELD == 0)
    {
        float xh, xl, yh, yl, Txh, Txl, Tyh, Tyl;
        const double *ax = A.axes + (size_t)e * 6 * A.axis_stride;
        double x0 = ax[i_th], y0 = ax[A.axis_stride + i_th], z0 = ax[2 * A.axis_stride + i_z];
        double px = ax[3 * A.axis_stride + i_px], py = ax[4 * A.axis_stride + i_py], pz = ax[5 * A.axis_stride + i_pz];
        double p0 = sqrt(px * px + py * py + pz * pz);
        double tx = px / p0, ty = py / p0, tz = pz / p0;
        xh = (float)x0; xl = (float)(x0 - (double)xh);
        yh = (float)y0; yl = (float)(y0 - (double)yh);
        zh = (float)z0; zl = (float)(z0 - (double)zh);
        Txh = (float)tx; Txl = (float)(tx - (double)Txh);
        Tyh = (float)ty; Tyl = (float)(ty - (double)Tyh);
        Tzh = (float)tz; Tzl = (float)(tz - (double)Tzh);
        double a64 = A.kq / p0;
        a = (float)a64;
        // the fp32 roundings of a and h/6 are the same every step; fold their ratio into the T update
        epsT = (float)((a64 * A.h6_64) / ((double)a * (double)A.h_6) - 1.0);
        // with energy loss a is recomputed every step as fl32(kq) / p: the systematic roundings are those of kq and h/6
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
        xyh = pk(xh, yh); xyl = pk(xl, yl); Txyh = pk(Txh, Tyh); Txyl = pk(Txl, Tyl);
    }
    // p <= 1 MeV/c ends a track after its first step (C7)
    // (a thread beyond the grid takes no step: its `valid` folded into the step cap keeps the loop test to one compare)
    const int max_steps = !valid ? 0 : ((p0h > 1.0f) ? A.max_steps : min(A.max_steps, 1));

    uint32_t nm = 0, tests = 0, cnt = 0, lookups = 0;
    float chi2 = 0.0f;
    int n = 0, m = 0, turn = 0, kcount = 0;
    bool cn = true;                                   // c_0 := true (reading C7)
    const float h = A.h;
    Slots S;
    S.n = 0; S.w0 = S.w1 = S.w2 = S.w3 = 0; S.g0 = S.g1 = S.g2 = S.g3 = 0.0f;

    // Field reuse (tabulated field, no energy loss).  The 4th stage of step n evaluates B at r_n + h T + h^2/2 k3; the
    // start vertex of step n + 1 is r_n + h T + h^2/6 (k1 + k2 + k3), a distance delta = h^2/6 |k1 + k2 - 2 k3| away.
    // With |k| <= |a| B and G a bound of the field's gradient, |k1 - k3| and |k2 - k3| give
    //     delta <= h^3/6 |a| (|a| B^2 + G)      (~1e-5 mm at 105 MeV/c, 1 T, h = 2 mm)
    // so B moves by at most G delta between the two points.  Where that is below HALF AN ULP of B_max in fp32 -- below
    // what the fp32 field value resolves -- the seed takes the carried value instead of a third table look-up per
    // step (decided once per seed from its |a|; soft seeds and steep fields evaluate all three).  Measured: the
    // position error against the oracle is unchanged to three digits.
    const bool reuse = FIELD == 1 && !ELOSS && A.reuse_c * fabsf(a) * fmaf(fabsf(a), A.reuse_b2, A.fd.grad_max) <= A.reuse_eps;
    const int n_fresh = reuse ? 0 : 0x7fffffff;       // steps n <= n_fresh evaluate B at their start vertex
    f2 Bxy_c = pk(0.f, 0.f);
    float Bz_c = 0.f;
#pragma unroll kScanUnroll
    while (n < max_steps) {
        // ---- A5: every K steps, the wires near r_n that carry a hit -> slots, with g at this vertex
        if (kcount == 0) {
            // centre of the next K steps (straight-line prediction; the arc's sagitta is in the host's margin); a seed
            // curling tighter than that margin allows looks up around its own position instead, at the shorter cadence
            const bool tight = !(fabsf(a) * A.b_max < A.tight_curv);
            kcount = tight ? A.lookup_every_tight : A.lookup_every;
            const float ahead = tight ? 0.0f : A.lookahead;
            S.n = 0;
            const float xh = lo(xyh), yh = hi(xyh), xl = lo(xyl), yl = hi(xyl), Txh = lo(Txyh), Tyh = hi(Txyh);
            const float cx = fmaf(ahead, Txh, xh), cy = fmaf(ahead, Tyh, yh), cz = fmaf(ahead, Tzh, zh);
            const float zeta = cz * A.gd.tan_abs;
            const float u2 = fmaf(cx, cx, fmaf(cy, cy, -zeta * zeta));
            if (u2 > A.u2_lo && u2 < A.u2_hi) {
                lookups += 1u;
                const float u = u2 * rsqrt_normal(u2);                  // u2 > u2_lo > 0
                const float fj = (u - A.gd.r_first) * A.gd.inv_pitch;
                const float jn = rintf(fj);
                const int jc = (int)jn;
                const int j2 = jc + ((fj - jn) >= 0.0f ? 1 : -1);
                LookupCtx V;
                V.x = xh; V.xl = xl; V.y = yh; V.yl = yl; V.z = zh; V.Tx = Txh; V.Ty = Tyh; V.Tz = Tzh;
                V.cz = cz;
                V.phi = coarse_atan2(cy, cx);
                {
                    const float cbend = (ELOSS ? 1.05f : 1.0f) * A.delta_max * fabsf(a) * A.b_max;
                    V.g_dead = fmaf(A.hold_path * 0.25f, cbend * cbend, 0.02f);
                    // nor can a wire own an approach before the next lookup if g is still far below zero: g grows by at
                    // most h (1 + |delta| |a| B) per step (g' = 1 - (T.u)^2 + delta . T')
                    V.g_far = -fmaf((float)kcount * h, 1.0f + cbend, 0.25f);
                    V.curv = tight ? 0.0f : (ELOSS ? 1.05f : 1.0f) * fabsf(a) * A.b_max;
                    const float hold = (float)kcount * h + 0.5f;           // path to the next lookup (+ margin)
                    V.ptol = fmaf(0.6f * V.curv, hold * hold, A.window + 0.05f);
                    V.hold = hold;
                }
                lookup_layer(A, s_layer, s_bits, drift_e, jc, V, S, cnt);
                lookup_layer(A, s_layer, s_bits, drift_e, j2, V, S, cnt);
            }
        }
        kcount -= 1;
        f2 sdxy;                                       // the increment this step adds to the position
        float sdz;

        // ---- A4: one Nystroem-RK4 step of r'' = a (r' x B(r))
        if (FIELD == 0) {
            // uniform field B = (0, 0, Bz): the four stages are linear in T, k = c J U with J (Tx, Ty) = (Ty, -Tx), so
            // the Nystroem step collapses (exactly, theta = a Bz h) to
            //   dT = [ (theta - theta^3/6) J + (-theta^2/2 + theta^4/24) I ] T
            //   dr = h T + h [ (theta/2 - theta^3/24) J - (theta^2/6) I ] T          (k_z == 0, T_z constant)
            // -- the same map as k1..k4 and the weighted sums, with the stage arithmetic done once per seed.
            // Packed: J T = (Ty, -Tx) is the pair with its halves swapped and one negated -- operand modifiers, no instruction.
            if (ELOSS) {                                  // theta follows p_n; constants in fp32 like a itself
                const float th = a * A.fd.bz * h, th2 = th * th;
                ub_h = fmaf(-th * th2, 0.166666672f, th); ub_l = ub_h * A.kq_rel;      // fl(kappa q) is off by the same
                ue1 = th2 * fmaf(th2, 0.0416666679f, -0.5f);                           // relative amount every step
                up1 = -h * th2 * 0.166666672f;
                up2_h = h * th * fmaf(th2, -0.0416666679f, 0.5f); up2_l = up2_h * A.kq_rel;
            }
            const f2 JT = pk(hi(Txyh), -lo(Txyh));     // J T: swap + negate one half, both operand modifiers (LO_HI.NP)
            // dTx = fmaf(ue1, Tx, fmaf(ub_h, Ty, ub_l * Ty)),  dTy = fmaf(ue1, Ty, fmaf(ub_h, -Tx, ub_l * -Tx))
            const f2 dTxy = fma2(bc(ue1), Txyh, fma2(bc(ub_h), JT, mul2(bc(ub_l), JT)));
            // dx = fmaf(up1, Tx, fmaf(up2_h, Ty, fmaf(up2_l, Ty, h * Tx))),  dy likewise with -Tx for Ty and Ty for Tx
            const f2 dxy = fma2(bc(up1), Txyh, fma2(bc(up2_h), JT, fma2(bc(up2_l), JT, mul2(h, Txyh))));
            sdxy = fma2(bc(h), Txyl, dxy); sdz = fmaf(h, Tzl, h * Tzh);      // h * T_lo: the part of T the fp32 products
            comp_add2(xyh, xyl, sdxy);                                       // never saw
            comp_add(zh, zl, sdz);
            comp_add2(Txyh, Txyl, dTxy);
        } else {
            // stage derivatives k = U x (a B) (field_at_p returns a B): the cross products mix components and stay scalar; their x and y results
            // land side by side and everything linear in them (stage directions and positions, increments, compensated
            // updates) is packed
            f2 Bxy;
            float Bz;
            if (n <= n_fresh) field_at_p(A.fd, a, xyh, zh, Bxy_c, Bz_c);         // else: carried from the last 4th stage
            Bxy = Bxy_c; Bz = Bz_c;
            float Ux = lo(Txyh), Uy = hi(Txyh), Uz = Tzh;
            const f2 k1xy = pk(fmaf(Uy, Bz, -Uz * hi(Bxy)), fmaf(Uz, lo(Bxy), -Ux * Bz));
            const float k1z = fmaf(Ux, hi(Bxy), -Uy * lo(Bxy));
            f2 Uxy = fma2(bc(A.h_half), k1xy, Txyh);
            Uz = fmaf(A.h_half, k1z, Tzh);
            field_at_p(A.fd, a, fma2(bc(A.h2_8), k1xy, fma2(bc(A.h_half), Txyh, xyh)), fmaf(A.h2_8, k1z, fmaf(A.h_half, Tzh, zh)), Bxy, Bz);
            Ux = lo(Uxy); Uy = hi(Uxy);
            const f2 k2xy = pk(fmaf(Uy, Bz, -Uz * hi(Bxy)), fmaf(Uz, lo(Bxy), -Ux * Bz));
            const float k2z = fmaf(Ux, hi(Bxy), -Uy * lo(Bxy));
            Uxy = fma2(bc(A.h_half), k2xy, Txyh); Uz = fmaf(A.h_half, k2z, Tzh);
            Ux = lo(Uxy); Uy = hi(Uxy);
            const f2 k3xy = pk(fmaf(Uy, Bz, -Uz * hi(Bxy)), fmaf(Uz, lo(Bxy), -Ux * Bz));
            const float k3z = fmaf(Ux, hi(Bxy), -Uy * lo(Bxy));
            Uxy = fma2(bc(h), k3xy, Txyh); Uz = fmaf(h, k3z, Tzh);
            field_at_p(A.fd, a, fma2(bc(A.h2_2), k3xy, fma2(bc(h), Txyh, xyh)), fmaf(A.h2_2, k3z, fmaf(h, Tzh, zh)), Bxy, Bz);
            Bxy_c = Bxy; Bz_c = Bz;
            Ux = lo(Uxy); Uy = hi(Uxy);
            const f2 k4xy = pk(fmaf(Uy, Bz, -Uz * hi(Bxy)), fmaf(Uz, lo(Bxy), -Ux * Bz));
            const float k4z = fmaf(Ux, hi(Bxy), -Uy * lo(Bxy));
            const f2 dxy = fma2(bc(A.h2_6), add2(add2(k1xy, k2xy), k3xy), mul2(h, Txyh));
            const float dz = fmaf(A.h2_6, (k1z + k2z) + k3z, h * Tzh);
            const f2 dTxy = mul2(A.h_6, fma2(bc(2.0f), add2(k2xy, k3xy), add2(k1xy, k4xy)));
            const float dTz = A.h_6 * fmaf(2.0f, k2z + k3z, k1z + k4z);
            sdxy = fma2(bc(h), Txyl, dxy); sdz = fmaf(h, Tzl, dz);
            comp_add2(xyh, xyl, sdxy);
            comp_add2(Txyh, Txyl, fma2(dTxy, bc(epsT), dTxy));
            {   // z and T_z take the same compensated update: one packed pair for the two (same operations, same rounding)
                f2 zT_h = pk(zh, Tzh), zT_l = pk(zl, Tzl);
                comp_add2(zT_h, zT_l, pk(sdz, fmaf(dTz, epsT, dTz)));
                zh = lo(zT_h); Tzh = hi(zT_h); zl = lo(zT_l); Tzl = hi(zT_l);
            }
        }

        // ---- A6: live wires over interval n (scored only if the interval starts in the gas)
        if (S.n > 0) {
            Vtx v1;
            v1.xy = xyh; v1.xyl = xyl; v1.z = zh;
            tests += (uint32_t)S.n;
            slot_step(A, drift_e, S.w0, S.g0, cn, sdxy, sdz, v1, Txyh, Tzh, nm, chi2, cnt);
            if (S.n > 1) slot_step(A, drift_e, S.w1, S.g1, cn, sdxy, sdz, v1, Txyh, Tzh, nm, chi2, cnt);
            if (S.n > 2) slot_step(A, drift_e, S.w2, S.g2, cn, sdxy, sdz, v1, Txyh, Tzh, nm, chi2, cnt);
            if (S.n > 3) slot_step(A, drift_e, S.w3, S.g3, cn, sdxy, sdz, v1, Txyh, Tzh, nm, chi2, cnt);
        }
        if (TRACK && cn) m += 1;

        // ---- advance, energy loss (reading C6), turn counter and termination (reading C7)
        n += 1;
        float rho2 = fmaf(lo(xyh), lo(xyh), hi(xyh) * hi(xyh));
        if (TRACK) {
            bool cnext = rho2 >= A.gd.R0sq;
            if (!cn && cnext) turn += 1;
            cn = cnext;
        }
        if (ELOSS) {
            float p = fmaf(-A.eloss_h, (float)m, p0h) + p0l;
            a = (float)A.kq / p;      // IEEE division
            if (!(p > 1.0f)) break;
        }
        if (!(fabsf(zh) <= A.gd.z_half)) break;
        if (!(rho2 <= A.gd.r_out_sq)) break;
    }

    // ---- A7: per-seed output, per-event argmax, candidate pool
    const float S32 = valid ? fmaf(-chi2, A.inv_lambda, (float)nm) : -1.0f;
    if (valid) {
        const int64_t o = G.out_offset + (int64_t)index;
        if (A.n_match) A.n_match[o] = nm;
        if (A.chi2) A.chi2[o] = chi2;
        if (A.debug) {
            cdc_seed_debug d;
            d.n_steps = n; d.turns = turn; d.m_gas = m; d.pad = 0;
            d.x = (double)lo(xyh) + (double)lo(xyl); d.y = (double)hi(xyh) + (double)hi(xyl); d.z = (double)zh + (double)zl;
            A.debug[o] = d;
        }
    }
    const float Sc = fmaxf(S32, 0.0f);                // S >= 0 by construction; clamp rounding residue
    unsigned long long key = valid ? (((unsigned long long)__float_as_uint(Sc) << 32) | (0xFFFFFFFFu - index)) : 0ull;
    unsigned long long wkey = warp_max_u64(key);
    const int lane = threadIdx.x & 31;
    unsigned long long run = 0ull;
    if (lane == 0) {
        unsigned long long old = atomicMax(A.best_key + e, wkey);
        run = old > wkey ? old : wkey;
    }
    run = __shfl_sync(0xffffffffu, run, 0);
    const float S_run = __uint_as_float((uint32_t)(run >> 32));
    // a seed without any match (S = 0 exactly) cannot beat index 0, which ties with it and wins on the index: only
    // index 0 stands in for all of them, so an event (or a neighbourhood) without hits cannot flood the pool
    const bool cand = valid && (Sc >= S_run - A.margin) && (Sc > 0.0f || index == 0u);
    const unsigned ballot = __ballot_sync(0xffffffffu, cand);
    if (ballot) {
        unsigned base = 0;
        if (lane == 0) base = (unsigned)atomicAdd(A.counters + CNT_POOL, (unsigned long long)__popc(ballot));
        base = __shfl_sync(0xffffffffu, base, 0);
        if (cand) {
            unsigned pos = base + __popc(ballot & ((1u << lane) - 1u));
            if (pos < A.pool_cap) {
                PoolEntry pe; pe.event = (uint32_t)e; pe.index = index; pe.S32 = Sc; pe.pad = 0;
                A.pool[pos] = pe;
            }
        }
    }
    unsigned sn = __reduce_add_sync(0xffffffffu, valid ? (unsigned)n : 0u);
    unsigned sm = __reduce_add_sync(0xffffffffu, valid ? (unsigned)m : 0u);
    unsigned st = __reduce_add_sync(0xffffffffu, tests);
    unsigned sl = __reduce_add_sync(0xffffffffu, lookups);
    unsigned sg = __reduce_add_sync(0xffffffffu, cnt & 0xFFFFu);
    unsigned sa = __reduce_add_sync(0xffffffffu, cnt >> 16);
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

cudaError_t launch_seed_scan(const ScanLaunch &L, cudaStream_t s, cudaEvent_t k0, cudaEvent_t k1)
{
    ScanArgs A;
    A.gd = L.gd; A.fd = L.fd; A.grids = L.d_grids; A.axes = L.d_axes; A.axis_stride = L.axis_stride;
    A.drift_tab = L.d_drift_tab; A.bits = L.d_bits;
    const double h = L.h64;
    A.h = (float)h; A.h_half = (float)(h / 2.0); A.h2_8 = (float)(h * h / 8.0); A.h2_2 = (float)(h * h / 2.0);
    A.h_6 = (float)(h / 6.0); A.h2_6 = (float)(h * h / 6.0);
    A.kq = CDC_KAPPA * (double)L.charge; A.h6_64 = h / 6.0;
    A.kq_rel = (float)(A.kq / (double)(float)A.kq - 1.0);
    A.lambda = L.lambda; A.inv_lambda = 1.0f / L.lambda; A.eloss_h = L.eloss_h; A.window = sqrtf(L.lambda) * 1.0001f;
    A.u2_lo = L.u2_lo; A.u2_hi = L.u2_hi; A.uz = L.uz; A.inv_uz = L.inv_uz; A.lookup_every = L.lookup_every; A.lookahead = L.lookahead; A.lookup_every_tight = L.lookup_every_tight; A.tight_curv = L.tight_curv;
    A.delta_max = L.delta_max; A.b_max = L.b_max; A.hold_path = L.hold_path;
    A.k_margin = L.k_margin; A.k_margin0 = L.k_margin0; A.sin_eps = L.sin_eps; A.sep_cap = L.sep_cap;
    A.two_inv_h = (float)(2.0 / h); A.inv_h = (float)(1.0 / h);
    // field reuse: h^3/6 G, B_max^2, half an ulp of B_max (2^-24 B_max; the ulp of values in [B_max / 2, B_max) is 2^-24 times
    // the next power of two >= that)
    A.reuse_c = (float)(h * h * h / 6.0 * (double)L.fd.grad_max); A.reuse_b2 = L.b_max * L.b_max;
    A.reuse_eps = (float)(ldexp(1.0, -24) * (double)L.b_max);
    if (L.variant == 3) A.reuse_eps = -1.0f;          // params.kernel_variant = 3: this kernel with the field reuse off (A / B)
    A.max_steps = L.max_steps; A.margin = L.margin;
    A.n_match = L.d_n_match; A.chi2 = L.d_chi2; A.debug = L.d_debug;
    A.best_key = (unsigned long long *)L.d_best_key;
    A.pool = L.d_pool; A.pool_cap = L.pool_cap; A.counters = L.d_counters;
    if (L.gd.n_bit_words > kMaxBitWords || L.gd.n_layers > CDC_MAX_LAYERS || L.lookup_every < 1) return cudaErrorInvalidValue;
    dim3 grid((unsigned)((L.max_seeds_per_event + kBlock - 1) / kBlock), (unsigned)L.n_events);
    const bool eloss = L.eloss_h != 0.0f;
    if (k0) cudaEventRecord(k0, s);
    // a held wire is scored from vertices at most `back` inside the lookup band's lower edge: if that is still outside
    // R0 the in-gas flag is true whenever it is read (c_0 := true covers the start vertex)
    const double u_lo = sqrt((double)L.u2_lo);
    const double back = (double)L.back;
    const bool track = eloss || L.d_debug != nullptr || !(u_lo - back - 0.5 >= sqrt((double)L.gd.R0sq));
    // comparison variant (params.kernel_variant = 1): two seeds per thread (scan_pair.cu); it has no tabulated-field
    // form with energy loss (per-seed momentum), which stays with the kernel below
    if (L.variant == 1 && !(L.fd.kind != 0 && eloss)) {
        const cudaError_t pe = launch_seed_scan_pair(A, L, eloss, track, s);
        if (k1) cudaEventRecord(k1, s);
        cdc_count_launch();
        return pe;
    }
    // comparison variant (params.kernel_variant = 2): lane refill, a thread runs two seeds in a row (scan_refill.cu)
    if (L.variant == 2) {
        const cudaError_t re = launch_seed_scan_refill(A, L, eloss, track, s);
        if (k1) cudaEventRecord(k1, s);
        cdc_count_launch();
        return re;
    }
    if (L.fd.kind == 0) {
        if (eloss) seed_scan_kernel<0, true, true><<<grid, kBlock, 0, s>>>(A);
        else if (track) seed_scan_kernel<0, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_kernel<0, false, false><<<grid, kBlock, 0, s>>>(A);
    } else {
        if (eloss) seed_scan_kernel<1, true, true><<<grid, kBlock, 0, s>>>(A);
        else if (track) seed_scan_kernel<1, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_kernel<1, false, false><<<grid, kBlock, 0, s>>>(A);
    }
    if (k1) cudaEventRecord(k1, s);
    cdc_count_launch();
    return cudaGetLastError();
}
