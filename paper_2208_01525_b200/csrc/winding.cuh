// winding.cuh -- per-site phase and per-link wrap count of the winding sweep; see the header comment of diag_fused.cu
// for the method.
#pragma once
#include "f32x2.cuh"

namespace u1u1 {

constexpr float INV_2PI = 0.15915494309189535f;
constexpr float NEAR_T = 0.5f - 1.5915494e-6f;             // pi - |chi| < 1e-5  <=>  |t - rint t| > 1/2 - 1e-5 / 2 pi
constexpr unsigned FLAG_LANES = 0xff00ff00u, VAL_LANES = 0x00ff00ffu;   // lanes 0 / 2: p / q values, lanes 1 / 3: their flags

// atan2 in ~20 instructions: octant reduction to t = min/max in [0, 1] and the degree-8 (in t^2) polynomial of
// Abramowitz & Stegun 4.4.49 (|error| <= 2e-8 in exact arithmetic; ~4e-7 in fp32 with the SFU reciprocal).
// A field that is exactly zero has no phase: NaN, which marks the links that touch it as degenerate.
__device__ inline float site_phase(float x, float y)
{
    const float ax = fabsf(x), ay = fabsf(y), mx = fmaxf(ax, ay);
    float inv;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv) : "f"(mx));
    const float t = fminf(ax, ay) * inv, s = t * t;
    float p = 0.0028662257f;
    p = fmaf(p, s, -0.0161657367f);
    p = fmaf(p, s, 0.0429096138f);
    p = fmaf(p, s, -0.0752896400f);
    p = fmaf(p, s, 0.1065626393f);
    p = fmaf(p, s, -0.1420889944f);
    p = fmaf(p, s, 0.1999355085f);
    p = fmaf(p, s, -0.3333314528f);
    float r = fmaf(p * s, t, t);
    r = ay > ax ? 1.57079637f - r : r;
    r = x < 0.f ? 3.14159274f - r : r;
    r = copysignf(r, y);
    return mx == 0.f ? __int_as_float(0x7fc00000) : r;
}

// Both sectors' phases at once: the same operations per lane as site_phase (so the slow path, which re-evaluates single
// phases with site_phase, sees the same bits), the multiplications and the polynomial in packed fp32x2 instructions.
__device__ inline f2 site_phase2(f2 x, f2 y)
{
    const f2 ax = make_float2(fabsf(x.x), fabsf(x.y)), ay = make_float2(fabsf(y.x), fabsf(y.y));
    const f2 mx = make_float2(fmaxf(ax.x, ay.x), fmaxf(ax.y, ay.y)), mn = make_float2(fminf(ax.x, ay.x), fminf(ax.y, ay.y));
    f2 inv;
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv.x) : "f"(mx.x));
    asm("rcp.approx.ftz.f32 %0, %1;" : "=f"(inv.y) : "f"(mx.y));
    const f2 t = mul2(mn, inv), s = mul2(t, t);
    f2 p = bc(0.0028662257f);
    p = fma2(p, s, bc(-0.0161657367f));
    p = fma2(p, s, bc(0.0429096138f));
    p = fma2(p, s, bc(-0.0752896400f));
    p = fma2(p, s, bc(0.1065626393f));
    p = fma2(p, s, bc(-0.1420889944f));
    p = fma2(p, s, bc(0.1999355085f));
    p = fma2(p, s, bc(-0.3333314528f));
    const f2 r0 = fma2(mul2(p, s), t, t);
    f2 r;
    r.x = ay.x > ax.x ? 1.57079637f - r0.x : r0.x;
    r.y = ay.y > ax.y ? 1.57079637f - r0.y : r0.y;
    r.x = x.x < 0.f ? 3.14159274f - r.x : r.x;
    r.y = x.y < 0.f ? 3.14159274f - r.y : r.y;
    r.x = copysignf(r.x, y.x);
    r.y = copysignf(r.y, y.y);
    r.x = mx.x == 0.f ? __int_as_float(0x7fc00000) : r.x;
    r.y = mx.y == 0.f ? __int_as_float(0x7fc00000) : r.y;
    return r;
}

// One link as a byte lane: wrap count n = rint(t) stored as n + 32 (|n| <= 31, i.e. |theta| < 190: the host checks the
// largest |theta| of the sweep), plus 0x100 in the next lane if the link needs the slow path: its angle is within 1e-5
// of the cut, or an end point is exactly zero (t is NaN, which fails the <=).  rint by the magic-number addition
// (exact for |t| < 2^22, ties to even like rintf): the low mantissa byte of t + 1.5 * 2^23 + 32 IS (n + 32) & 0xff, so
// no float <-> int conversion (XU pipe) is needed.
__device__ inline unsigned link_lane(float alpha_a, float alpha_b, float theta)
{
    constexpr float MAGIC = 12582912.f + 32.f;
    const float t = ((alpha_b - alpha_a) - theta) * INV_2PI;
    const float tm = t + MAGIC;
    const float d = t - (tm - MAGIC);
    return (__float_as_uint(tm) & 0xffu) + (fabsf(d) <= NEAR_T ? 0u : 256u);
}

// The same link of both sectors: the p lane in byte 0 (+ flag in byte 1), the q lane in byte 2 (+ flag in byte 3).
__device__ inline unsigned link_lane2(f2 alpha_a, f2 alpha_b, f2 theta)
{
    constexpr float MAGIC = 12582912.f + 32.f;
    const f2 t = mul2(sub2(sub2(alpha_b, alpha_a), theta), bc(INV_2PI));
    const f2 tm = add2(t, bc(MAGIC));
    const f2 d = sub2(t, sub2(tm, bc(MAGIC)));
    const unsigned lp = (__float_as_uint(tm.x) & 0xffu) + (fabsf(d.x) <= NEAR_T ? 0u : 256u);
    const unsigned lq = (__float_as_uint(tm.y) & 0xffu) + (fabsf(d.y) <= NEAR_T ? 0u : 256u);
    return __byte_perm(lp, lq, 0x5410);
}

}  // namespace u1u1
