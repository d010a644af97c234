// winding.cuh -- per-site phase and per-link wrap count of the winding sweep; see the header comment of diag_fused.cu
// for the method.
#pragma once

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

}  // namespace u1u1
