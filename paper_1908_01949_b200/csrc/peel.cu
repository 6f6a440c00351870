// Kernels of cdc_peel_turns (reading C18).  Compiled with -fmad=false:
// the extrapolation to the next entrance is fp64 IEEE arithmetic in the order reading C18 writes it.
#include "eval64.cuh"
#include "peel.cuh"

namespace {

// hits of the partition under investigation: unclassified hits the best seed matches in its first gas passage
__global__ void peel_count_kernel(const int32_t *offsets, const int32_t *labels, const int32_t *partition,
                                  const int32_t *active, int32_t *counts)
{
    const int e = blockIdx.y;
    if (!active[e]) return;
    const int i = offsets[e] + blockIdx.x * blockDim.x + threadIdx.x;
    const bool in = i < offsets[e + 1];
    const bool open = in && partition[i] < 0;
    const bool mine = open && labels[i] == 0;
    const unsigned m_open = __ballot_sync(0xffffffffu, open), m_mine = __ballot_sync(0xffffffffu, mine);
    if ((threadIdx.x & 31) == 0) {
        if (m_mine) atomicAdd(counts + 2 * e, __popc(m_mine));
        if (m_open) atomicAdd(counts + 2 * e + 1, __popc(m_open));
    }
}

// the partition is kept iff it has at least min_classified hits: label them k and take their wires out of the event
__global__ void peel_apply_kernel(int k, int min_classified, int32_t n_bit_words, const int32_t *offsets,
                                  const int32_t *wire_id, const int32_t *labels, const int32_t *active,
                                  const int32_t *counts, int32_t *partition, uint32_t *bits)
{
    const int e = blockIdx.y;
    if (!active[e] || counts[2 * e] < min_classified) return;
    const int i = offsets[e] + blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= offsets[e + 1]) return;
    if (partition[i] >= 0 || labels[i] != 0) return;
    partition[i] = k;
    const int w = wire_id[i];
    atomicAnd(bits + (size_t)e * n_bit_words + (w >> 5), ~(1u << (w & 31)));
}

__device__ __forceinline__ void crossing64(const double *r, const double *T, const double *rn, const double *Tn, double p,
                                           double R0, double *out)
{
    const double dx = rn[0] - r[0], dy = rn[1] - r[1], dz = rn[2] - r[2];
    const double A = dx * dx + dy * dy;
    const double B = r[0] * dx + r[1] * dy;
    const double Cc = r[0] * r[0] + r[1] * r[1] - R0 * R0;
    const double tau = (-B + sqrt(B * B - A * Cc)) / A;
    out[0] = r[0] + tau * dx; out[1] = r[1] + tau * dy; out[2] = r[2] + tau * dz;
    const double Ux = T[0] + tau * (Tn[0] - T[0]), Uy = T[1] + tau * (Tn[1] - T[1]), Uz = T[2] + tau * (Tn[2] - T[2]);
    const double nU = sqrt(Ux * Ux + Uy * Uy + Uz * Uz);
    out[3] = p * (Ux / nU); out[4] = p * (Uy / nU); out[5] = p * (Uz / nU);
}

// reading C18, step 6: the best seed's track to its next outward crossing of rho = R0 (same loop as eval_seed64:
// C4-C7), then the point of the chord on the cylinder.  One thread per event.
template <bool UNI>
__device__ bool next_entrance64(const PeelLaunch &L, int e, uint32_t index, double *out)
{
    const GridDev G = L.d_grids[e];
    uint32_t q = index;
    const int i_pz = q % G.n[4]; q /= G.n[4];
    const int i_py = q % G.n[3]; q /= G.n[3];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_z = q % G.n[1];
    const int i_th = q / G.n[1];
    const int st = L.axis_stride;
    const double *ax = L.d_axes + (size_t)e * 6 * st;
    const double px = ax[3 * st + i_px], py = ax[4 * st + i_py], pz = ax[5 * st + i_pz];
    double r[3] = {ax[i_th], ax[st + i_th], ax[2 * st + i_z]};                                    // C4
    const double p0 = sqrt(px * px + py * py + pz * pz);
    double T[3] = {px / p0, py / p0, pz / p0};
    const double eloss_h = L.eloss * L.h, R0 = L.g.R0;
    double p = p0;
    int n = 0, m = 0;
    bool cn = true;
    while (n < L.extrap_max_steps) {
        const double a = L.kq / p;
        double rn[3], Tn[3];
        rkn_step64<UNI>(L.g, a, L.h, r, T, rn, Tn);
        if (cn) m += 1;                                                                         // C6
        const double p_next = p0 - eloss_h * (double)m;
        const bool cnext = rn[0] * rn[0] + rn[1] * rn[1] >= R0 * R0;
        if (!cn && cnext) {                                                                     // C7: a new turn
            crossing64(r, T, rn, Tn, p_next, R0, out);
            return true;
        }
#pragma unroll
        for (int i = 0; i < 3; ++i) { r[i] = rn[i]; T[i] = Tn[i]; }
        n += 1;
        p = p_next;
        cn = cnext;
        if (fabs(r[2]) > L.g.z_half) break;
        if (r[0] * r[0] + r[1] * r[1] > L.g.r_out * L.g.r_out) break;
        if (!(p > 1.0)) break;
        if (!(isfinite(r[0]) && isfinite(r[1]) && isfinite(r[2]) && isfinite(T[0]) && isfinite(T[1]) && isfinite(T[2])))
            break;
    }
    return false;
}

// reading C19: the same extrapolation with the step-doubling controller on the error estimate of the paper's
// ref. [5]: step lengths h 2^j in [h, h_max]; halve and repeat on err > tol or on an outward crossing taken with more
// than h; double after an accepted step with err <= tol / 32.
__device__ bool next_entrance64_adaptive(const PeelLaunch &L, int e, uint32_t index, double *out)
{
    const GridDev G = L.d_grids[e];
    uint32_t q = index;
    const int i_pz = q % G.n[4]; q /= G.n[4];
    const int i_py = q % G.n[3]; q /= G.n[3];
    const int i_px = q % G.n[2]; q /= G.n[2];
    const int i_z = q % G.n[1];
    const int i_th = q / G.n[1];
    const int st = L.axis_stride;
    const double *ax = L.d_axes + (size_t)e * 6 * st;
    const double px = ax[3 * st + i_px], py = ax[4 * st + i_py], pz = ax[5 * st + i_pz];
    double r[3] = {ax[i_th], ax[st + i_th], ax[2 * st + i_z]};                                    // C4
    const double p0 = sqrt(px * px + py * py + pz * pz);
    double T[3] = {px / p0, py / p0, pz / p0};
    const double R0 = L.g.R0, h0 = L.h, tol = L.extrap_tol;
    double p = p0, s_gas = 0.0, hc = h0;
    int n = 0;
    bool cn = true;
    while (n < L.extrap_max_steps) {
        const double a = L.kq / p;
        double rn[3], Tn[3], err;
        rkn_step64_err(L.g, a, hc, r, T, rn, Tn, &err);
        if (err > tol && hc > h0) { hc = hc / 2.0; continue; }
        const bool cnext = rn[0] * rn[0] + rn[1] * rn[1] >= R0 * R0;
        if (!cn && cnext && hc > h0) { hc = hc / 2.0; continue; }
        const double s_next = cn ? s_gas + hc : s_gas;                                          // C6
        const double p_next = p0 - L.eloss * s_next;
        if (!cn && cnext) { crossing64(r, T, rn, Tn, p_next, R0, out); return true; }           // C7: a new turn
#pragma unroll
        for (int i = 0; i < 3; ++i) { r[i] = rn[i]; T[i] = Tn[i]; }
        n += 1;
        p = p_next; s_gas = s_next;
        cn = cnext;
        if (fabs(r[2]) > L.g.z_half) break;
        if (r[0] * r[0] + r[1] * r[1] > L.g.r_out * L.g.r_out) break;
        if (!(p > 1.0)) break;
        if (!(isfinite(r[0]) && isfinite(r[1]) && isfinite(r[2]) && isfinite(T[0]) && isfinite(T[1]) && isfinite(T[2])))
            break;
        if (err <= tol / 32.0 && hc * 2.0 <= L.extrap_h_max) hc = hc * 2.0;
    }
    return false;
}

__global__ void next_entrance_kernel(const PeelLaunch L)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= L.n_events) return;
    double out[6] = {0.0, 0.0, 0.0, 0.0, 0.0, 0.0};
    bool ok = false;
    const int64_t b = L.d_best_seed[e];
    if (L.d_active[e] && b >= 0 && L.extrap_tol > 0.0)
        ok = next_entrance64_adaptive(L, e, (uint32_t)b, out);
    else if (L.d_active[e] && b >= 0)
        ok = L.g.field_kind == 0 ? next_entrance64<true>(L, e, (uint32_t)b, out) : next_entrance64<false>(L, e, (uint32_t)b, out);
#pragma unroll
    for (int i = 0; i < 6; ++i) L.d_next[(size_t)e * 6 + i] = out[i];
    L.d_next_ok[e] = ok ? 1 : 0;
}

}  // namespace

cudaError_t peel_partition(const PeelLaunch &L, int k, int min_classified, cudaStream_t s)
{
    cudaError_t e;
    if ((e = cudaMemsetAsync(L.d_counts, 0, sizeof(int32_t) * 2 * (size_t)L.n_events, s)) != cudaSuccess) return e;
    if (L.max_hits_per_event > 0) {
        dim3 grid((unsigned)((L.max_hits_per_event + 127) / 128), (unsigned)L.n_events);
        peel_count_kernel<<<grid, 128, 0, s>>>(L.d_offsets, L.d_labels, L.d_partition, L.d_active, L.d_counts);
        peel_apply_kernel<<<grid, 128, 0, s>>>(k, min_classified, L.n_bit_words, L.d_offsets, L.d_wire_id, L.d_labels,
                                               L.d_active, L.d_counts, L.d_partition, L.d_bits);
        cdc_count_launch(2);
    }
    next_entrance_kernel<<<(L.n_events + 31) / 32, 32, 0, s>>>(L);
    cdc_count_launch();
    return cudaGetLastError();
}
