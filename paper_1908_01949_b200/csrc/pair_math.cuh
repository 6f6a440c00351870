// Packed fp32 pairs for sm_100a: one 64-bit register pair holds the same quantity of TWO seeds (A in the low half,
// B in the high half) and every arithmetic instruction on it is one issue slot for both -- FFMA2 / FADD2 / FMUL2 in SASS
// (PTX fma.rn.f32x2, add.rn.f32x2, sub.rn.f32x2, mul.rn.f32x2; ISA 8.6, sm_100+).  Each half is rounded to nearest
// exactly like the scalar instruction, so a packed seed computes bit for bit what a scalar seed computes.
// An operand built as pk(s, s) compiles to the broadcast form (R.F32 / UR.F32): no register pair is materialised.
// Measured on B200 (profiles/r2_f32x2_issue_rates.md): FFMA2 issues every second cycle per SM sub-partition -- the FP32
// pipe delivers the same 128 lanes x 2 flops per clock either way -- but it takes ONE issue slot for 64 lane-operations,
// which leaves the other slot to the integer / memory / branch instructions this kernel is full of.
#pragma once
#include <cuda_runtime.h>

namespace {

struct f2 { unsigned long long v; };

__device__ __forceinline__ f2 pk(float a, float b)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(a), "f"(b));
    return r;
}
__device__ __forceinline__ f2 bc(float s) { return pk(s, s); }
__device__ __forceinline__ float lo(f2 a)
{
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
    (void)y;
    return x;
}
__device__ __forceinline__ float hi(f2 a)
{
    float x, y;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(x), "=f"(y) : "l"(a.v));
    (void)x;
    return y;
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 sub2(f2 a, f2 b)
{
    f2 r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
// exact negation of both halves: ptxas folds the two scalar negations into the consumer's operand modifier
// (-R.F32x2.HI_LO), so it costs no instruction
__device__ __forceinline__ f2 neg2(f2 a) { return pk(-lo(a), -hi(a)); }
// scalar-broadcast shorthands
__device__ __forceinline__ f2 fma2(float a, f2 b, f2 c) { return fma2(bc(a), b, c); }
__device__ __forceinline__ f2 fma2(f2 a, float b, f2 c) { return fma2(a, bc(b), c); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, float c) { return fma2(a, b, bc(c)); }
__device__ __forceinline__ f2 fma2(float a, f2 b, float c) { return fma2(bc(a), b, bc(c)); }
__device__ __forceinline__ f2 mul2(float a, f2 b) { return mul2(bc(a), b); }
__device__ __forceinline__ f2 mul2(f2 a, float b) { return mul2(a, bc(b)); }
__device__ __forceinline__ f2 add2(f2 a, float b) { return add2(a, bc(b)); }
__device__ __forceinline__ f2 sub2(f2 a, float b) { return sub2(a, bc(b)); }

// Kahan-compensated accumulation of both halves: (hi, lo) += d (the scalar comp_add of scan_common.cuh, packed)
__device__ __forceinline__ void comp_add2(f2 &h, f2 &l, f2 d)
{
    const f2 y = add2(d, l);
    const f2 t = add2(h, y);
    l = sub2(y, sub2(t, h));
    h = t;
}

}  // namespace
