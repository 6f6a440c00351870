// A2: Hough circle pre-vote (PAPER.md:51 "circle finding method, namely the Hough transform", :61 Fig. 4;
// parametrisation = reading C13).
//
// Definition (gather form): acc[iR][icy][icx] = #{hits : | |c - x_hit| - R | < tol} at the bin centres, bins
// with | |c| - R | > origin + tol are ineligible (count 0); peak = max count, ties -> lowest linear index.
//
// Mapping: one thread owns one centre bin (icx, icy) and ALL its radius bins: the distance |c - x_hit| is
// computed once per (centre, hit) and fans out to the <= ceil(2 tol / bin_R) + 1 radius bins it can vote for.
// The per-thread radius histogram lives in shared memory, [iR][thread] u16 (bank-conflict free, no atomics:
// each column has one owner, so the accumulator is deterministic).  Hit (x, y) at z_ref are staged through
// shared memory in chunks.  The peak is reduced by warp shuffles and one atomicMax per warp on a packed
// (votes << 32 | ~linear index) key.
#include "cdc_internal.cuh"

namespace {

constexpr int kHBlock = 256;
constexpr int kChunk = 1024;

__device__ __forceinline__ unsigned long long warp_max_u64(unsigned long long v)
{
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        unsigned long long other = __shfl_xor_sync(0xffffffffu, v, o);
        v = other > v ? other : v;
    }
    return v;
}

struct HoughArgs {
    int32_t nR, ncy, ncx, nspan;
    float bin_xy, bin_R, inv_bin_R, tol, R_lo, half_xy, origin;
    const float *wire5;
    const int32_t *offsets, *wire_id;
    const float *zref;
    uint32_t *accum;
    unsigned long long *peak_key;
};

__global__ void __launch_bounds__(kHBlock) hough_vote_kernel(const HoughArgs A)
{
    extern __shared__ unsigned char smem_raw[];
    float2 *s_xy = reinterpret_cast<float2 *>(smem_raw);                          // [kChunk]
    unsigned short *s_hist = reinterpret_cast<unsigned short *>(s_xy + kChunk);   // [nR][kHBlock]

    const int e = blockIdx.y;
    const int col = blockIdx.x * kHBlock + threadIdx.x;
    const int n_col = A.ncy * A.ncx;
    const bool valid = col < n_col;
    const int icy = valid ? col / A.ncx : 0, icx = valid ? col - icy * A.ncx : 0;
    const float cx = fmaf((float)icx + 0.5f, A.bin_xy, -A.half_xy);
    const float cy = fmaf((float)icy + 0.5f, A.bin_xy, -A.half_xy);
    for (int r = 0; r < A.nR; ++r) s_hist[r * kHBlock + threadIdx.x] = 0;

    const int h0 = A.offsets[e], h1 = A.offsets[e + 1];
    const float zr = A.zref[e];
    for (int base = h0; base < h1; base += kChunk) {
        const int cnt = min(kChunk, h1 - base);
        __syncthreads();
        for (int i = threadIdx.x; i < cnt; i += kHBlock) {
            const float *w = A.wire5 + (size_t)A.wire_id[base + i] * 5;
            const float t = zr / w[4];                         // wire (x, y) at z = z_ref
            s_xy[i] = make_float2(fmaf(t, w[2], w[0]), fmaf(t, w[3], w[1]));
        }
        __syncthreads();
        if (valid) {
            for (int i = 0; i < cnt; ++i) {
                const float2 p = s_xy[i];                      // broadcast read
                const float ex = cx - p.x, ey = cy - p.y;
                const float d = sqrtf(fmaf(ex, ex, ey * ey));
                int r = __float2int_rd((d - A.tol - A.R_lo) * A.inv_bin_R - 0.5f);   // one below the first possible bin
                for (int k = 0; k < A.nspan; ++k, ++r) {
                    if ((unsigned)r < (unsigned)A.nR) {
                        const float Rc = fmaf((float)r + 0.5f, A.bin_R, A.R_lo);
                        if (fabsf(d - Rc) < A.tol) s_hist[r * kHBlock + threadIdx.x] += 1;
                    }
                }
            }
        }
    }

    unsigned long long best = 0ull;
    if (valid) {
        const float cn = sqrtf(fmaf(cx, cx, cy * cy));
        for (int r = 0; r < A.nR; ++r) {
            const float Rc = fmaf((float)r + 0.5f, A.bin_R, A.R_lo);
            const bool eligible = fabsf(cn - Rc) <= A.origin + A.tol;
            const uint32_t votes = eligible ? (uint32_t)s_hist[r * kHBlock + threadIdx.x] : 0u;
            const uint32_t lin = (uint32_t)((r * A.ncy + icy) * A.ncx + icx);
            if (A.accum) A.accum[(size_t)e * A.nR * n_col + lin] = votes;
            const unsigned long long key = ((unsigned long long)votes << 32) | (0xFFFFFFFFu - lin);
            best = key > best ? key : best;
        }
    }
    best = warp_max_u64(best);
    if ((threadIdx.x & 31) == 0) atomicMax(A.peak_key + e, best);   // all-zero accumulator -> bin 0 wins
}

// Peak bin -> circle -> transverse seed at R0 and its ranges (Fig. 4; reading C13), fp64.
__global__ void hough_finalize_kernel(int n_events, int nR, int ncy, int ncx, double bin_xy, double bin_R,
                                      double R_lo, double half_xy, double R0, double half_theta, double half_pt,
                                      double bz, int charge, const unsigned long long *peak_key, double *ranges,
                                      int32_t *peak)
{
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e >= n_events) return;
    const unsigned long long key = peak_key[e];
    const uint32_t lin = 0xFFFFFFFFu - (uint32_t)(key & 0xFFFFFFFFull);
    const int votes = (int)(key >> 32);
    const int icx = (int)(lin % (uint32_t)ncx), icy = (int)((lin / (uint32_t)ncx) % (uint32_t)ncy);
    const int iR = (int)(lin / ((uint32_t)ncx * (uint32_t)ncy));
    peak[4 * e + 0] = iR; peak[4 * e + 1] = icy; peak[4 * e + 2] = icx; peak[4 * e + 3] = votes;
    const double R = R_lo + ((double)iR + 0.5) * bin_R;
    const double cy = -half_xy + ((double)icy + 0.5) * bin_xy;
    const double cx = -half_xy + ((double)icx + 0.5) * bin_xy;
    const double cn = sqrt(cx * cx + cy * cy);
    const double gamma = atan2(cy, cx);
    double cb = (R0 * R0 + cn * cn - R * R) / (2.0 * R0 * cn);   // law of cosines: |R0 e(theta) - c| = R
    cb = fmin(1.0, fmax(-1.0, cb));
    const double beta = acos(cb);
    const double sgn = ((double)charge * bz < 0.0) ? 1.0 : -1.0;  // q Bz < 0: counter-clockwise, entrance at gamma - beta
    const double th = gamma - sgn * beta;
    const double ex = R0 * cos(th), ey = R0 * sin(th);
    const double pt = CDC_KAPPA * fabs(bz) * R;
    const double px = sgn * pt * (-(ey - cy)) / R;
    const double py = sgn * pt * (ex - cx) / R;
    double *o = ranges + 6 * (size_t)e;
    o[0] = th - half_theta; o[1] = th + half_theta;
    o[2] = px - half_pt;    o[3] = px + half_pt;
    o[4] = py - half_pt;    o[5] = py + half_pt;
}

}  // namespace

cudaError_t launch_hough(const HoughLaunch &L, cudaStream_t s)
{
    HoughArgs A;
    A.nR = L.nR; A.ncy = L.ncy; A.ncx = L.ncx;
    A.nspan = (int)ceil(2.0 * (double)L.tol / (double)L.bin_R) + 2;
    A.bin_xy = L.bin_xy; A.bin_R = L.bin_R; A.inv_bin_R = 1.0f / L.bin_R; A.tol = L.tol; A.R_lo = L.R_lo;
    A.half_xy = L.half_xy; A.origin = L.origin;
    A.wire5 = L.d_wire5; A.offsets = L.d_offsets; A.wire_id = L.d_wire_id; A.zref = L.d_zref;
    A.accum = L.d_accum; A.peak_key = L.d_peak_key;
    cudaError_t e = cudaMemsetAsync(L.d_peak_key, 0, sizeof(unsigned long long) * (size_t)L.n_events, s);
    if (e != cudaSuccess) return e;
    const size_t smem = sizeof(float2) * kChunk + sizeof(unsigned short) * (size_t)L.nR * kHBlock;
    if (smem > 200 * 1024) return cudaErrorInvalidValue;
    if (smem > 48 * 1024) {
        e = cudaFuncSetAttribute(hough_vote_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
        if (e != cudaSuccess) return e;
    }
    dim3 grid((unsigned)((L.ncy * L.ncx + kHBlock - 1) / kHBlock), (unsigned)L.n_events);
    hough_vote_kernel<<<grid, kHBlock, smem, s>>>(A);
    cdc_count_launch(2);
    e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    hough_finalize_kernel<<<(L.n_events + 63) / 64, 64, 0, s>>>(L.n_events, L.nR, L.ncy, L.ncx, L.bin_xy64, L.bin_R64,
                                                                 L.R_lo64, L.half_xy64, L.R0, L.half_theta, L.half_pt,
                                                                 L.bz, L.charge, L.d_peak_key, L.d_ranges, L.d_peak);
    return cudaGetLastError();
}
