// jp_f32x2.cuh -- packed FP32 pairs (sm_100 FFMA2 / FADD2: one instruction, two lanes of a 64-bit register pair).
// The plane loops of the tiled kernels are bound by instruction issue; two consecutive planes of one LOR share their
// coefficients, so the coordinate arithmetic of both (u = a2 + b2 k, the magic-number floor, the fractional part, the
// fixed-point rounding) is done on pairs.  The halves of a pair are ordinary registers: no moves to unpack.
#pragma once
#include <cuda_runtime.h>

namespace jp {

struct F2 {
    unsigned long long v;
};

__device__ __forceinline__ F2 f2(float lo, float hi)
{
    F2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ F2 f2(float x) { return f2(x, x); }
__device__ __forceinline__ float f2_lo(F2 a)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v));
    return lo;
}
__device__ __forceinline__ float f2_hi(F2 a)
{
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v));
    return hi;
}
__device__ __forceinline__ F2 fma2(F2 a, F2 b, F2 c)
{
    F2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ F2 add2(F2 a, F2 b)
{
    F2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ F2 add2_rm(F2 a, F2 b) // round towards minus infinity (the magic-number floor)
{
    F2 r;
    asm("add.rm.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}

} // namespace jp
