// Packed pair arithmetic (device code): two reals in one aligned register pair.
#pragma once

#include <cuda_runtime.h>

namespace nmp {

// fp32: add.f32x2 / mul.f32x2 / fma.f32x2 (FADD2 / FMUL2 / FFMA2 of sm_100a).  A pair of fp32
// values (a complex number, or the same quantity on two mesh rows) is one aligned register pair;
// the packed instructions work on both halves with one issue slot, and ptxas folds half swaps, per-half negation and scalar broadcast
// into their operand modifiers (.LO_HI, .NP, .F32), so a rotation by +-i or a complex product costs
// no extra instruction.  Same rounding per element as the scalar forms.
// fp64 pairs use the scalar instructions (same names, so that kernels are written once).
__device__ __forceinline__ unsigned long long pk2(float x, float y)
{
    unsigned long long v;
    asm("mov.b64 %0, {%1, %2};" : "=l"(v) : "f"(x), "f"(y));
    return v;
}
__device__ __forceinline__ float2 up2(unsigned long long v)
{
    float2 r;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(r.x), "=f"(r.y) : "l"(v));
    return r;
}
__device__ __forceinline__ float2 padd(float2 a, float2 b)
{
    unsigned long long r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)));
    return up2(r);
}
__device__ __forceinline__ float2 psub(float2 a, float2 b)
{
    unsigned long long r;
    asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)));
    return up2(r);
}
__device__ __forceinline__ float2 pmul(float2 a, float2 b)
{
    unsigned long long r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)));
    return up2(r);
}
__device__ __forceinline__ float2 pfma(float2 a, float2 b, float2 c)
{
    unsigned long long r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(pk2(a.x, a.y)), "l"(pk2(b.x, b.y)), "l"(pk2(c.x, c.y)));
    return up2(r);
}
__device__ __forceinline__ double2 padd(double2 a, double2 b) { a.x += b.x; a.y += b.y; return a; }
__device__ __forceinline__ double2 psub(double2 a, double2 b) { a.x -= b.x; a.y -= b.y; return a; }
__device__ __forceinline__ double2 pmul(double2 a, double2 b) { a.x *= b.x; a.y *= b.y; return a; }
__device__ __forceinline__ double2 pfma(double2 a, double2 b, double2 c)
{
    c.x = fma(a.x, b.x, c.x);
    c.y = fma(a.y, b.y, c.y);
    return c;
}

} // namespace nmp
