// Register-only FFMA chains: the empirical FP32 peak that the scan's roofline fraction is quoted against.
// 8 independent accumulators per thread (enough ILP to cover the 4-cycle FFMA latency at any occupancy),
// 1024 threads per block, 2 blocks per SM.
#include "cdc_internal.cuh"

namespace {

__global__ void __launch_bounds__(1024) ffma_chain_kernel(int iters, float seed, float *sink)
{
    float a0 = seed + threadIdx.x, a1 = a0 + 1.f, a2 = a0 + 2.f, a3 = a0 + 3.f;
    float a4 = a0 + 4.f, a5 = a0 + 5.f, a6 = a0 + 6.f, a7 = a0 + 7.f;
    const float m = 0.9999f, c = 1e-3f * seed;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            a0 = fmaf(a0, m, c); a1 = fmaf(a1, m, c); a2 = fmaf(a2, m, c); a3 = fmaf(a3, m, c);
            a4 = fmaf(a4, m, c); a5 = fmaf(a5, m, c); a6 = fmaf(a6, m, c); a7 = fmaf(a7, m, c);
        }
    }
    const float r = ((a0 + a1) + (a2 + a3)) + ((a4 + a5) + (a6 + a7));
    if (r == 123.456f) sink[0] = r;       // never true; keeps the chains alive
}

// Issue rates of the packed fp32 instructions of sm_100a (FFMA2 / FADD2 / FMUL2) against the scalar ones, alone and mixed
// with integer-pipe work: the measurement behind the choice of packed pairs in the scan kernel.
// 8 independent chains per thread, 256 threads, 8 blocks per SM.  MODE: 0 FFMA, 1 FFMA2, 2 FADD, 3 FADD2, 4 FMUL2,
// 5 FFMA2 + LOP3, 6 FFMA + LOP3, 7 FFMA2 + FFMA.
#define PK(d, a, b) asm volatile("mov.b64 %0, {%1, %2};" : "=l"(d) : "f"(a), "f"(b))
#define FMA2(d, a, b, c) asm volatile("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c))
#define ADD2(d, a, b) asm volatile("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b))
#define MUL2(d, a, b) asm volatile("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b))
#define FMA1(d, a, b, c) asm volatile("fma.rn.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c))
#define ADD1(d, a, b) asm volatile("add.rn.f32 %0, %1, %2;" : "=f"(d) : "f"(a), "f"(b))
#define LOP(d, a, b) asm volatile("xor.b32 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b))

template <int MODE>
__global__ void __launch_bounds__(256) issue_probe_kernel(int iters, float s, float *sink)
{
    float x[8];
    unsigned long long X[8], Bp, Cp;
    unsigned q[8];
    for (int i = 0; i < 8; ++i) { x[i] = threadIdx.x * 0.001f + i; PK(X[i], x[i], x[i] + 0.5f); q[i] = threadIdx.x + i; }
    const float b = s, c = 1.0f - s;
    PK(Bp, b, b); PK(Cp, c, c);
    for (int it = 0; it < iters; ++it) {
#pragma unroll
        for (int r = 0; r < 4; ++r) {
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                if (MODE == 0) FMA1(x[i], x[i], b, c);
                if (MODE == 1) FMA2(X[i], X[i], Bp, Cp);
                if (MODE == 2) ADD1(x[i], x[i], c);
                if (MODE == 3) ADD2(X[i], X[i], Cp);
                if (MODE == 4) MUL2(X[i], X[i], Bp);
                if (MODE == 5) { FMA2(X[i], X[i], Bp, Cp); LOP(q[i], q[i], q[(i + 1) & 7]); }
                if (MODE == 6) { FMA1(x[i], x[i], b, c); LOP(q[i], q[i], q[(i + 1) & 7]); }
                if (MODE == 7) { FMA2(X[i], X[i], Bp, Cp); FMA1(x[i], x[i], b, c); }
            }
        }
    }
    float acc = 0.f;
    for (int i = 0; i < 8; ++i) acc += x[i] + (float)(X[i] & 0xFFFF) + (float)q[i];
    if (acc == 123.456f) sink[0] = acc;
}

}  // namespace

cudaError_t run_fp32_issue_probe(int32_t mode, int32_t iters, double *ms_out, double *warp_inst, double *flops, cudaStream_t s)
{
    int dev = 0, n_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    float *sink = nullptr;
    if ((e = cudaMalloc(&sink, sizeof(float))) != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int blocks = 8 * n_sm;
    auto launch = [&](int it) {
        switch (mode) {
        case 0: issue_probe_kernel<0><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 1: issue_probe_kernel<1><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 2: issue_probe_kernel<2><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 3: issue_probe_kernel<3><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 4: issue_probe_kernel<4><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 5: issue_probe_kernel<5><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        case 6: issue_probe_kernel<6><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        default: issue_probe_kernel<7><<<blocks, 256, 0, s>>>(it, 0.5f, sink); break;
        }
    };
    launch(iters / 8 + 1);
    cudaEventRecord(t0, s);
    launch(iters);
    cudaEventRecord(t1, s);
    cdc_count_launch(2);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    static const double inst_per_inner[8] = {1, 1, 1, 1, 1, 2, 2, 2}, flops_per_inner[8] = {2, 4, 1, 2, 2, 4, 2, 6};
    const double inner = (double)blocks * 256.0 * (double)iters * 32.0;          // 4 x 8 per iteration
    if (ms_out) *ms_out = (double)ms;
    if (warp_inst) *warp_inst = inner * inst_per_inner[mode & 7] / 32.0;
    if (flops) *flops = inner * flops_per_inner[mode & 7];
    return cudaGetLastError();
}

cudaError_t run_fp32_peak_probe(int32_t iters, double *flops_per_s, double *ms_out, cudaStream_t s)
{
    int dev = 0, n_sm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&n_sm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    float *sink = nullptr;
    if ((e = cudaMalloc(&sink, sizeof(float))) != cudaSuccess) return e;
    cudaEvent_t t0, t1;
    cudaEventCreate(&t0); cudaEventCreate(&t1);
    const int blocks = 2 * n_sm;
    ffma_chain_kernel<<<blocks, 1024, 0, s>>>(iters / 8 + 1, 1.0f, sink);     // warm-up
    cudaEventRecord(t0, s);
    ffma_chain_kernel<<<blocks, 1024, 0, s>>>(iters, 1.0f, sink);
    cudaEventRecord(t1, s);
    cdc_count_launch(2);
    e = cudaEventSynchronize(t1);
    float ms = 0.f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, t0, t1);
    cudaEventDestroy(t0); cudaEventDestroy(t1);
    cudaFree(sink);
    if (e != cudaSuccess) return e;
    const double flops = 2.0 * 8.0 * 16.0 * (double)iters * 1024.0 * (double)blocks;
    if (flops_per_s) *flops_per_s = flops / ((double)ms * 1e-3);
    if (ms_out) *ms_out = (double)ms;
    return cudaGetLastError();
}
