// A3-A7 with lane refill (params.kernel_variant = 2): the one-seed-per-thread scan of scan.cu in which a lane whose
// track has ended takes a second seed instead of idling until the slowest track of its warp ends (BJ north_star:
// "warp-level ... ballots cover early termination"; PAPER.md:125 names the divergence of early-exiting seeds).
//
// The lanes of a warp are z0-neighbours (scan.cu, A3) and most tracks end at |z| = z_half, so the step count of a lane
// is close to linear in its z0 index: the refill needs no queue.  A warp owns two consecutive 32-seed chunks; lane l
// runs seed l of the first chunk and then seed 31 - l of the second -- the short track of one chunk is followed by the
// long track of the other and every lane of the warp has about the same total.  One vote per step (__any_sync) ends the
// warp when no lane is live.
//
// What changes against scan.cu is bookkeeping only: the step, the lookup, the live-wire code and the per-seed
// arithmetic are the same functions (scan_one.cuh), so every seed gets bit for bit the n_match, chi2 and final position
// scan.cu gives it.  Three things keep the second seeds from costing more than they save:
//   * the lookup cadence is a warp-uniform clock (kc_u): a lane that starts a second seed looks wires up at once and
//     then joins the common cadence (its first hold is shorter, which the lookup margins cover), so the warp still
//     runs the lookup code once per K steps and not once per lane phase;
//   * a finished seed is written out by its own lane (plain stores); the key of the first seed waits in shared memory
//     and the warp-wide arg max / candidate-pool epilogue runs once, for both seeds, after the loop;
//   * the seed prologue (fp64 divide and square root) runs under divergence for the second seed -- about 16 times per
//     warp instead of once -- which is the price (~1 % of a 1600-step track).
#include "cdc_internal.cuh"
#include "scan_common.cuh"
#include "scan_args.cuh"
#include "pair_math.cuh"
#include "scan_one.cuh"

namespace {

#ifndef REFILL_MB0
#define REFILL_MB0 8
#endif
#ifndef REFILL_MB1
#define REFILL_MB1 0
#endif
#ifndef REFILL_UNROLL
#define REFILL_UNROLL 2
#endif
constexpr int kRefillUnroll = REFILL_UNROLL;

template <int FIELD, bool ELOSS, bool TRACK>
__global__ void __launch_bounds__(kBlock, FIELD == 0 ? REFILL_MB0 : REFILL_MB1) seed_scan_refill_kernel(const ScanArgs A)
{
    __shared__ LayerDev s_layer[CDC_MAX_LAYERS];
    __shared__ uint32_t s_bits[kMaxBitWords];
    __shared__ unsigned long long s_key[2][kBlock];    // packed (S, index) of the thread's first / second seed; 0: none
    __shared__ int s_n0[kBlock], s_m0[kBlock];          // steps / in-gas steps of the thread's finished seeds (counters)

    const int e = blockIdx.y;
    const GridDev G = A.grids[e];
    if ((int64_t)blockIdx.x * (2 * kBlock) >= (int64_t)G.n_seeds) return;
    for (int i = threadIdx.x; i < A.gd.n_layers; i += kBlock) s_layer[i] = A.gd.layers[i];
    for (int i = threadIdx.x; i < A.gd.n_bit_words; i += kBlock)
        s_bits[i] = A.bits[(size_t)e * A.gd.n_bit_words + i];
    s_key[0][threadIdx.x] = 0ull; s_key[1][threadIdx.x] = 0ull; s_n0[threadIdx.x] = 0; s_m0[threadIdx.x] = 0;
    __syncthreads();
    const float *drift_e = A.drift_tab + (size_t)e * A.gd.n_wires_total;

    // ---- A3: thread -> two seeds.  Thread order as in scan.cu (z0 lane-fastest, then theta, px, py, pz); warp w of the
    // grid owns seeds [64 w, 64 w + 64): lane l takes 64 w + l, then 64 w + 32 + (31 - l).
    const int lane = threadIdx.x & 31;
    const int64_t first = ((int64_t)blockIdx.x * (kBlock / 32) + (threadIdx.x >> 5)) * 64;

    f2 xyh, xyl, Txyh, Txyl;
    float zh, zl, Tzh, Tzl, a, epsT, p0h, p0l;
    float ub_h = 0.f, ub_l = 0.f, ue1 = 0.f, up1 = 0.f, up2_h = 0.f, up2_l = 0.f;   // uniform-field step map (FIELD == 0)
    uint32_t index = 0, nm = 0;
    float chi2 = 0.0f;
    int n = 0, m = 0, turn = 0, kcount = 0, max_steps = 0;
    bool cn = true;
    Slots S;
    S.n = 0; S.w0 = S.w1 = S.w2 = S.w3 = 0; S.g0 = S.g1 = S.g2 = S.g3 = 0.0f;

    // the prologue of scan.cu for seed t of the thread order
    auto load_seed = [&](int t) {
        int q = t;
        const int i_z = q % G.n[1]; q /= G.n[1];
        const int i_th = q % G.n[0]; q /= G.n[0];
        const int i_px = q % G.n[2]; q /= G.n[2];
        const int i_py = q % G.n[3];
        const int i_pz = q / G.n[3];
        index = (uint32_t)((((i_th * G.n[1] + i_z) * G.n[2] + i_px) * G.n[3] + i_py) * G.n[4] + i_pz);
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
        epsT = (float)((a64 * A.h6_64) / ((double)a * (double)A.h_6) - 1.0);
        if (ELOSS) epsT = (float)((A.kq * A.h6_64) / ((double)(float)A.kq * (double)A.h_6) - 1.0);
        p0h = (float)p0; p0l = (float)(p0 - (double)p0h);
        if (FIELD == 0) {
            const double h64 = 6.0 * A.h6_64, th = a64 * (double)A.fd.bz * h64, th2 = th * th;
            const double b = th - th * th2 / 6.0, p2 = h64 * (th / 2.0 - th * th2 / 24.0);
            ub_h = (float)b; ub_l = (float)(b - (double)ub_h);
            up2_h = (float)p2; up2_l = (float)(p2 - (double)up2_h);
            ue1 = (float)(-th2 / 2.0 + th2 * th2 / 24.0);
            up1 = (float)(-h64 * th2 / 6.0);
        }
        xyh = pk(xh, yh); xyl = pk(xl, yl); Txyh = pk(Txh, Tyh); Txyl = pk(Txl, Tyl);
        max_steps = (p0h > 1.0f) ? A.max_steps : min(A.max_steps, 1);      // reading C7
        nm = 0; chi2 = 0.0f; n = 0; m = 0; turn = 0; kcount = 0; cn = true; S.n = 0;
    };

    uint32_t tests = 0, cnt = 0, lookups = 0;
    const float h = A.h;

    // a finished seed: per-seed outputs by its own lane; its key waits for the warp-wide epilogue
    auto finish_seed = [&](int pass) {
        const float S32 = fmaf(-chi2, A.inv_lambda, (float)nm);
        const int64_t o = G.out_offset + (int64_t)index;
        if (A.n_match) A.n_match[o] = nm;
        if (A.chi2) A.chi2[o] = chi2;
        if (A.debug) {
            cdc_seed_debug d;
            d.n_steps = n; d.turns = turn; d.m_gas = m; d.pad = 0;
            d.x = (double)lo(xyh) + (double)lo(xyl); d.y = (double)hi(xyh) + (double)hi(xyl); d.z = (double)zh + (double)zl;
            A.debug[o] = d;
        }
        const float Sc = fmaxf(S32, 0.0f);
        s_key[pass][threadIdx.x] = ((unsigned long long)__float_as_uint(Sc) << 32) | (0xFFFFFFFFu - index);
        s_n0[threadIdx.x] += n; s_m0[threadIdx.x] += m;
    };

    int pass = 0;                                      // 0 / 1: running the first / second seed; 2: retired
    bool have = first + lane < (int64_t)G.n_seeds;     // the current pass has a seed
    bool live = false;
    if (have) { load_seed((int)(first + lane)); live = n < max_steps; }
    int kc_u = 0;                                      // warp-uniform lookup clock: the common cadence of the warp's lanes

    // Field reuse as in scan.cu (same decision per seed, so the same arithmetic).  There:  The 4th stage of step n evaluates B at r_n + h T + h^2/2 k3; the
    // start vertex of step n + 1 is r_n + h T + h^2/6 (k1 + k2 + k3), a distance delta = h^2/6 |k1 + k2 - 2 k3| away.
    // With |k| <= |a| B and G a bound of the field's gradient, |k1 - k3| and |k2 - k3| give
    //     delta <= h^3/6 |a| (|a| B^2 + G)      (~1e-5 mm at 105 MeV/c, 1 T, h = 2 mm)
    // so B moves by at most G delta between the two points.  Where that is below HALF AN ULP of B_max in fp32 -- below
    // what the fp32 field value resolves -- the seed takes the carried value instead of a third table look-up per
    // step (decided once per seed from its |a|; soft seeds and steep fields evaluate all three).  Measured: the
    // position error against the oracle is unchanged to three digits.
    bool reuse = false;
    auto decide_reuse = [&]() { reuse = FIELD == 1 && !ELOSS && A.reuse_c * fabsf(a) * fmaf(fabsf(a), A.reuse_b2, A.fd.grad_max) <= A.reuse_eps; };
    f2 Bxy_c = pk(0.f, 0.f);
    float Bz_c = 0.f;
    if (have) decide_reuse();
#pragma unroll kRefillUnroll
    for (;;) {
        if (!live && pass < 2) {                       // this lane's track has ended: write it out, take the next seed
            if (have) finish_seed(pass);
            pass += 1;
            if (pass == 1) {
                const int64_t t1 = first + 32 + (31 - lane);
                have = t1 < (int64_t)G.n_seeds;
                if (have) { load_seed((int)t1); decide_reuse(); live = n < max_steps; }
            }
        }
        if (!__any_sync(0xffffffffu, live)) break;
        if (kc_u == 0) kc_u = A.lookup_every;
        if (live) {
            // ---- A5 (scan.cu): every K steps, the wires near r_n that carry a hit -> slots
            if (kcount == 0) {
                const bool tight = !(fabsf(a) * A.b_max < A.tight_curv);
                kcount = tight ? A.lookup_every_tight : kc_u;          // a second seed joins the warp's cadence
                const float ahead = tight ? 0.0f : A.lookahead;
                S.n = 0;
                const float xh = lo(xyh), yh = hi(xyh), xl = lo(xyl), yl = hi(xyl), Txh = lo(Txyh), Tyh = hi(Txyh);
                const float cx = fmaf(ahead, Txh, xh), cy = fmaf(ahead, Tyh, yh), cz = fmaf(ahead, Tzh, zh);
                const float zeta = cz * A.gd.tan_abs;
                const float u2 = fmaf(cx, cx, fmaf(cy, cy, -zeta * zeta));
                if (u2 > A.u2_lo && u2 < A.u2_hi) {
                    lookups += 1u;
                    const float u = u2 * rsqrt_normal(u2);
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
                        // the bounds of scan.cu with the FULL cadence: a shorter first hold only makes them loose
                        const float kfull = (float)(tight ? A.lookup_every_tight : A.lookup_every);
                        V.g_far = -fmaf(kfull * h, 1.0f + cbend, 0.25f);
                        V.curv = tight ? 0.0f : (ELOSS ? 1.05f : 1.0f) * fabsf(a) * A.b_max;
                        const float hold = kfull * h + 0.5f;
                        V.ptol = fmaf(0.6f * V.curv, hold * hold, A.window + 0.05f);
                        V.hold = hold;
                    }
                    lookup_layer(A, s_layer, s_bits, drift_e, jc, V, S, cnt);
                    lookup_layer(A, s_layer, s_bits, drift_e, j2, V, S, cnt);
                }
            }
            kcount -= 1;
            f2 sdxy;
            float sdz;

            // ---- A4: one Nystroem-RK4 step (scan.cu: closed-form map in the uniform field, packed stages in the table)
            if (FIELD == 0) {
                if (ELOSS) {
                    const float th = a * A.fd.bz * h, th2 = th * th;
                    ub_h = fmaf(-th * th2, 0.166666672f, th); ub_l = ub_h * A.kq_rel;
                    ue1 = th2 * fmaf(th2, 0.0416666679f, -0.5f);
                    up1 = -h * th2 * 0.166666672f;
                    up2_h = h * th * fmaf(th2, -0.0416666679f, 0.5f); up2_l = up2_h * A.kq_rel;
                }
                const f2 JT = pk(hi(Txyh), -lo(Txyh));
                const f2 dTxy = fma2(bc(ue1), Txyh, fma2(bc(ub_h), JT, mul2(bc(ub_l), JT)));
                const f2 dxy = fma2(bc(up1), Txyh, fma2(bc(up2_h), JT, fma2(bc(up2_l), JT, mul2(h, Txyh))));
                sdxy = fma2(bc(h), Txyl, dxy); sdz = fmaf(h, Tzl, h * Tzh);
                comp_add2(xyh, xyl, sdxy);
                comp_add(zh, zl, sdz);
                comp_add2(Txyh, Txyl, dTxy);
            } else {
                f2 Bxy;
                float Bz;
                if (n == 0 || !reuse) field_at_p(A.fd, a, xyh, zh, Bxy_c, Bz_c);     // else: carried from the last 4th stage
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
                comp_add(zh, zl, sdz);
                comp_add2(Txyh, Txyl, fma2(dTxy, bc(epsT), dTxy));
                comp_add(Tzh, Tzl, fmaf(dTz, epsT, dTz));
            }

            // ---- A6: live wires over interval n
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

            // ---- advance, energy loss (C6), turn counter and termination (C7): a track that ends clears `live`
            n += 1;
            float rho2 = fmaf(lo(xyh), lo(xyh), hi(xyh) * hi(xyh));
            if (TRACK) {
                bool cnext = rho2 >= A.gd.R0sq;
                if (!cn && cnext) turn += 1;
                cn = cnext;
            }
            live = n < max_steps && fabsf(zh) <= A.gd.z_half && rho2 <= A.gd.r_out_sq;
            if (ELOSS) {
                float p = fmaf(-A.eloss_h, (float)m, p0h) + p0l;
                a = (float)A.kq / p;      // IEEE division
                live = live && p > 1.0f;
            }
        }
        kc_u -= 1;
    }

    // ---- A7: per-event arg max and candidate pool, once for the two seeds of every lane (scan.cu's epilogue)
    const unsigned long long key0 = s_key[0][threadIdx.x], key1 = s_key[1][threadIdx.x];
    const unsigned long long wkey = warp_max_u64(key0 > key1 ? key0 : key1);
    unsigned long long run = 0ull;
    if (lane == 0) {
        unsigned long long old = atomicMax(A.best_key + e, wkey);
        run = old > wkey ? old : wkey;
    }
    run = __shfl_sync(0xffffffffu, run, 0);
    const float S_run = __uint_as_float((uint32_t)(run >> 32));
#pragma unroll
    for (int k = 0; k < 2; ++k) {
        const unsigned long long key = k ? key1 : key0;
        const float Sc = __uint_as_float((uint32_t)(key >> 32));
        const uint32_t idx = 0xFFFFFFFFu - (uint32_t)key;
        // key == 0: no seed (a real key has a non-zero low word: indices stay below 2^31)
        const bool cand = key != 0ull && (Sc >= S_run - A.margin) && (Sc > 0.0f || idx == 0u);
        const unsigned ballot = __ballot_sync(0xffffffffu, cand);
        if (ballot) {
            unsigned base = 0;
            if (lane == 0) base = (unsigned)atomicAdd(A.counters + CNT_POOL, (unsigned long long)__popc(ballot));
            base = __shfl_sync(0xffffffffu, base, 0);
            if (cand) {
                unsigned pos = base + __popc(ballot & ((1u << lane) - 1u));
                if (pos < A.pool_cap) {
                    PoolEntry pe; pe.event = (uint32_t)e; pe.index = idx; pe.S32 = Sc; pe.pad = 0;
                    A.pool[pos] = pe;
                }
            }
        }
    }
    unsigned sn = __reduce_add_sync(0xffffffffu, (unsigned)s_n0[threadIdx.x]);
    unsigned sm = __reduce_add_sync(0xffffffffu, (unsigned)s_m0[threadIdx.x]);
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

cudaError_t launch_seed_scan_refill(const ScanArgs &A, const ScanLaunch &L, bool eloss, bool track, cudaStream_t s)
{
    dim3 grid((unsigned)((L.max_seeds_per_event + 2 * kBlock - 1) / (2 * kBlock)), (unsigned)L.n_events);
    if (L.fd.kind == 0) {
        if (eloss) seed_scan_refill_kernel<0, true, true><<<grid, kBlock, 0, s>>>(A);
        else if (track) seed_scan_refill_kernel<0, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_refill_kernel<0, false, false><<<grid, kBlock, 0, s>>>(A);
    } else {
        if (eloss) seed_scan_refill_kernel<1, true, true><<<grid, kBlock, 0, s>>>(A);
        else if (track) seed_scan_refill_kernel<1, false, true><<<grid, kBlock, 0, s>>>(A);
        else seed_scan_refill_kernel<1, false, false><<<grid, kBlock, 0, s>>>(A);
    }
    return cudaGetLastError();
}
