// f32x2.cuh -- packed fp32x2 arithmetic of sm_100 (FFMA2 / FADD2 / FMUL2: one issue slot, two IEEE fp32 operations), used
// by the step kernels (step_site.cuh) and the fused diagnostics sweep (diag_fused.cu).
#pragma once
#include <cuda_runtime.h>

namespace u1u1 {

// A pair holds the SAME quantity of the two sectors (p in .x, q in .y): the two sectors obey the same equations
// (PAPER.md:79), and the layout of common.cuh puts such pairs in the aligned 64-bit halves of every vector load.
// Negations fold into the operand modifiers of the packed instructions; scalars broadcast from uniform registers.
typedef float2 f2;
__device__ __forceinline__ f2 lo(const float4 &v) { return make_float2(v.x, v.y); }
__device__ __forceinline__ f2 hi(const float4 &v) { return make_float2(v.z, v.w); }
__device__ __forceinline__ f2 bc(float a) { return make_float2(a, a); }
__device__ __forceinline__ f2 neg(f2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ f2 add2(f2 a, f2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ f2 sub2(f2 a, f2 b) { return __fadd2_rn(a, neg(b)); }
__device__ __forceinline__ f2 mul2(f2 a, f2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ f2 plaq2(f2 a, f2 b, f2 c, f2 d) { return sub2(sub2(add2(a, b), c), d); }

// Range reduction in front of the SFU sine / cosine (MUFU takes the angle times 1/(2 pi) rounded to fp32, an absolute
// error of 6e-8 |theta| for the non-compact link phases of reading R-9): r = theta - n 2 pi with n = rint(theta / 2 pi) by
// the magic-number addition and 2 pi split into its fp32 value and the remainder (Cody-Waite; |theta| < 2^22 * 2 pi).
// For |theta| < pi (every production run) n = 0 and r is theta itself, bit for bit.
constexpr float RR_INV_2PI = 0.15915494309189535f, RR_MAGIC = 12582912.f;
constexpr float RR_2PI_HI = 6.2831854820251465f, RR_2PI_LO = -1.7484555e-07f;       // 2 pi = HI + LO
__device__ __forceinline__ f2 reduce_2pi2(f2 th)
{
    const f2 n = add2(fma2(th, bc(RR_INV_2PI), bc(RR_MAGIC)), bc(-RR_MAGIC));
    return fma2(n, bc(-RR_2PI_LO), fma2(n, bc(-RR_2PI_HI), th));
}

}  // namespace u1u1
