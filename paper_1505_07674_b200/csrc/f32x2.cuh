// f32x2.cuh -- packed FP32 pairs for sm_100a (FFMA2 / FMUL2 / FADD2).
//
// Blackwell issues one packed instruction for two FP32 lanes held in an aligned 64-bit
// register pair; the FMA pipe still does 128 lanes per SM per clock, but a warp spends ONE
// issue slot per two results.  Both kernels of this library are issue-slot bound with
// scalar FP32 (profiles/r1a.md), so their inner loops are written on pairs.
//
// ptxas folds a pair built from one scalar (`bc(s)`), an immediate or a uniform register
// into the instruction's broadcast operand form (`R7.F32`, `0.5`, `UR6.F32`): no MOV.
#pragma once

namespace lensed {

struct f2 { unsigned long long v; };

__device__ __forceinline__ f2 mk2(float lo, float hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r.v) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ f2 bc(float s) { return mk2(s, s); }
__device__ __forceinline__ void un2(f2 a, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(a.v));
}
__device__ __forceinline__ float lo2(f2 a) { float x, y; un2(a, x, y); return x; }
__device__ __forceinline__ float hi2(f2 a) { float x, y; un2(a, x, y); return y; }

__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r.v) : "l"(a.v), "l"(b.v), "l"(c.v));
    return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r.v) : "l"(a.v), "l"(b.v));
    return r;
}

// apply a scalar function to both halves (MUFU and ALU-pipe operations have no packed form)
template <class F>
__device__ __forceinline__ f2 map2(f2 a, F f)
{
    float x, y;
    un2(a, x, y);
    return mk2(f(x), f(y));
}
template <class F>
__device__ __forceinline__ f2 map2(f2 a, f2 b, F f)
{
    float ax, ay, bx, by;
    un2(a, ax, ay);
    un2(b, bx, by);
    return mk2(f(ax, bx), f(ay, by));
}

}  // namespace lensed
