// step_site.cuh -- one site of the fused kick + drift step (Eq. 17-26) for BOTH sectors at once in the
// packed fp32x2 instructions of sm_100, as a function of accessors into staged planes: shared by the one-step kernel
// (step_tiled.cu) and the two-steps-per-pass kernel (step_tb.cu), so that the two produce the same bits.
#pragma once
#include "common.cuh"
#include "f32x2.cuh"

namespace u1u1 {

// difference-form phasors of both sectors' link: the two MUFU pairs stay scalar, everything around them is packed
// RR: explicit range reduction of the half angle in front of the SFU (f32x2.cuh): keeps the phasor error at 5e-7 for
// non-compact phases of any size instead of 6e-8 |theta|; the identity, bit for bit, while |theta| < 2 pi.
template <bool RR>
__device__ __forceinline__ void phasor_diff2(f2 th, f2 &sn, f2 &c1)
{
    const f2 h0 = mul2(th, bc(0.5f)), h = RR ? reduce_2pi2(h0) : h0;
    f2 sh, ch;
    __sincosf(h.x, &sh.x, &ch.x);
    __sincosf(h.y, &sh.y, &ch.y);
    const f2 sh2 = add2(sh, sh);
    sn = mul2(sh2, ch);
    c1 = mul2(sh2, sh);
}


// What a site needs from plane z-1, computed by the same thread one plane earlier: the backward z difference
// conj(U_z(x-z)) f(x-z) - f(x) and the two plaquettes that contain theta_z(x-z) (bit-identical to the neighbour's own).
struct PkCarry {
    f2 bzr, bzi, Pyz, Pzx;
    float4 Ac, Bc;          // OWN: the site's own packs A and B, loaded one plane earlier as its z+1 neighbour's
};

// Accessors: A(p, dx, dy), B(p, dx, dy) return the float4 of pack A / B and C(p, dx, dy) the float2 of pack C of the site
// displaced by (dx, dy) in plane p (0 = the site's own plane z, 1 = plane z+1); the displacements are literals, so every
// address is base + immediate.  Operation order = the scalar difference-form chain of step_tiled.cu.
template <bool RR, bool OWN = false, class FA, class FB, class FC>
__device__ __forceinline__ void pk_carry_init(PkCarry &cy, FA A, FB B, FC C)       // here plane 0 = z-1, plane 1 = z
{
    const float4 Ac = A(0, 0, 0), Bc = B(0, 0, 0), Bzp = B(1, 0, 0), Azp = A(1, 0, 0);
    const f2 thz = C(0, 0, 0), Cxp = C(0, 1, 0), Cyp = C(0, 0, 1);
    const f2 fr = lo(Ac), fi = hi(Ac);
    f2 sn, c1;
    phasor_diff2<RR>(thz, sn, c1);
    cy.bzr = fma2(neg(sn), fi, fma2(neg(c1), fr, sub2(fr, lo(Azp))));
    cy.bzi = fma2(sn, fr, fma2(neg(c1), fi, sub2(fi, hi(Azp))));
    cy.Pyz = plaq2(hi(Bc), Cyp, hi(Bzp), thz);
    cy.Pzx = plaq2(thz, lo(Bzp), Cxp, lo(Bc));
    if (OWN) {
        cy.Ac = Azp;
        cy.Bc = Bzp;
    }
}

// MA, MB, MC: the site's momenta, updated in place; OA, OB, OC: its new positions.
// OWN: the site's own packs A and B of plane z come from the carry (two fewer 128-bit shared-memory reads, eight more
// carried registers).
template <bool RR, bool OWN = false, class FA, class FB, class FC>
__device__ __forceinline__ void pk_site_update(PkCarry &cy, FA A, FB B, FC C, const StepCoef &k, float4 &MA, float4 &MB,
                                               float2 &MC, float4 &OA, float4 &OB, float2 &OC)
{
    const float4 Ac = OWN ? cy.Ac : A(0, 0, 0), Axp = A(0, 1, 0), Axm = A(0, -1, 0), Ayp = A(0, 0, 1), Aym = A(0, 0, -1), Azp = A(1, 0, 0);
    const float4 Bc = OWN ? cy.Bc : B(0, 0, 0), Bxp = B(0, 1, 0), Bxm = B(0, -1, 0), Byp = B(0, 0, 1), Bym = B(0, 0, -1);
    const float4 Bxmyp = B(0, -1, 1), Bxpym = B(0, 1, -1), Bzp = B(1, 0, 0), Bxmzp = B(1, -1, 0), Bymzp = B(1, 0, -1);
    const f2 Cc = C(0, 0, 0), Cxp = C(0, 1, 0), Cxm = C(0, -1, 0), Cyp = C(0, 0, 1), Cym = C(0, 0, -1);
    const f2 fr = lo(Ac), fi = hi(Ac);
    const f2 thx = lo(Bc), thy = hi(Bc), thz = Cc;
    const f2 thmx = lo(Bxm), thmy = hi(Bym);                             // theta_i(x - i), i = x, y
    f2 lap_re = cy.bzr, lap_im = cy.bzi, J0, J1, J2, sn, c1, dr, di;
    // x: forward hop, current, backward hop
    phasor_diff2<RR>(thx, sn, c1);
    dr = fma2(sn, hi(Axp), fma2(neg(c1), lo(Axp), sub2(lo(Axp), fr)));
    di = fma2(neg(sn), lo(Axp), fma2(neg(c1), hi(Axp), sub2(hi(Axp), fi)));
    lap_re = add2(lap_re, dr);
    lap_im = add2(lap_im, di);
    J0 = fma2(fr, di, neg(mul2(fi, dr)));
    phasor_diff2<RR>(thmx, sn, c1);
    lap_re = add2(lap_re, fma2(neg(sn), hi(Axm), fma2(neg(c1), lo(Axm), sub2(lo(Axm), fr))));
    lap_im = add2(lap_im, fma2(sn, lo(Axm), fma2(neg(c1), hi(Axm), sub2(hi(Axm), fi))));
    // y
    phasor_diff2<RR>(thy, sn, c1);
    dr = fma2(sn, hi(Ayp), fma2(neg(c1), lo(Ayp), sub2(lo(Ayp), fr)));
    di = fma2(neg(sn), lo(Ayp), fma2(neg(c1), hi(Ayp), sub2(hi(Ayp), fi)));
    lap_re = add2(lap_re, dr);
    lap_im = add2(lap_im, di);
    J1 = fma2(fr, di, neg(mul2(fi, dr)));
    phasor_diff2<RR>(thmy, sn, c1);
    lap_re = add2(lap_re, fma2(neg(sn), hi(Aym), fma2(neg(c1), lo(Aym), sub2(lo(Aym), fr))));
    lap_im = add2(lap_im, fma2(sn, lo(Aym), fma2(neg(c1), hi(Aym), sub2(hi(Aym), fi))));
    // z: forward hop, current, and the backward z difference of the NEXT plane
    phasor_diff2<RR>(thz, sn, c1);
    dr = fma2(sn, hi(Azp), fma2(neg(c1), lo(Azp), sub2(lo(Azp), fr)));
    di = fma2(neg(sn), lo(Azp), fma2(neg(c1), hi(Azp), sub2(hi(Azp), fi)));
    lap_re = add2(lap_re, dr);
    lap_im = add2(lap_im, di);
    J2 = fma2(fr, di, neg(mul2(fi, dr)));
    cy.bzr = fma2(neg(sn), fi, fma2(neg(c1), fr, sub2(fr, lo(Azp))));
    cy.bzi = fma2(sn, fr, fma2(neg(c1), fi, sub2(fi, hi(Azp))));
    // potential force (Eq. 17-18): bracket_s = c lambda_s/2 (|f_s|^2 - sigma_s^2) - c kappa (|f_o|^2 - sigma_o^2)
    const f2 u = sub2(fma2(fr, fr, mul2(fi, fi)), make_float2(k.sig1sq, k.sig2sq));
    const f2 ku = mul2(bc(k.kap), u);
    const f2 bracket = fma2(make_float2(k.lamh1, k.lamh2), u, make_float2(-ku.y, -ku.x));
    const f2 m0 = lo(MA), m1 = hi(MA);
    const f2 pr = add2(m0, fma2(bc(k.aSm1), m0, mul2(bc(k.bS), fma2(lap_re, bc(k.inv_dx2), neg(mul2(fr, bracket))))));
    const f2 pi = add2(m1, fma2(bc(k.aSm1), m1, mul2(bc(k.bS), fma2(lap_im, bc(k.inv_dx2), neg(mul2(fi, bracket))))));
    MA = make_float4(pr.x, pr.y, pi.x, pi.y);
    const f2 or_ = fma2(bc(k.dtau), pr, fr), oi_ = fma2(bc(k.dtau), pi, fi);
    OA = make_float4(or_.x, or_.y, oi_.x, oi_.y);
    // lattice curl of the plaquettes (Eq. 20-21)
    const f2 Pxy = plaq2(thx, hi(Bxp), lo(Byp), thy);
    const f2 Pxy_my = plaq2(lo(Bym), hi(Bxpym), thx, thmy);
    const f2 Pxy_mx = plaq2(thmx, thy, lo(Bxmyp), hi(Bxm));
    const f2 Pyz = plaq2(thy, Cyp, hi(Bzp), thz);
    const f2 Pyz_my = plaq2(thmy, thz, hi(Bymzp), Cym);
    const f2 Pzx = plaq2(thz, lo(Bzp), Cxp, thx);
    const f2 Pzx_mx = plaq2(Cxm, lo(Bxmzp), thz, thmx);
    const f2 cc0 = sub2(sub2(Pxy, Pxy_my), sub2(Pzx, cy.Pzx));
    const f2 cc1 = sub2(sub2(Pyz, cy.Pyz), sub2(Pxy, Pxy_mx));
    const f2 cc2 = sub2(sub2(Pzx, Pzx_mx), sub2(Pyz, Pyz_my));
    cy.Pyz = Pyz;
    cy.Pzx = Pzx;
    if (OWN) {
        cy.Ac = Azp;
        cy.Bc = Bzp;
    }
    const f2 cur = make_float2(k.cur1, k.cur2);
    const f2 g0 = lo(MB), g1 = hi(MB), g2 = MC;
    const f2 e0 = add2(g0, fma2(bc(k.aGm1), g0, mul2(bc(k.bG), fma2(cur, J0, neg(mul2(cc0, bc(k.inv_dx3)))))));
    const f2 e1 = add2(g1, fma2(bc(k.aGm1), g1, mul2(bc(k.bG), fma2(cur, J1, neg(mul2(cc1, bc(k.inv_dx3)))))));
    const f2 e2 = add2(g2, fma2(bc(k.aGm1), g2, mul2(bc(k.bG), fma2(cur, J2, neg(mul2(cc2, bc(k.inv_dx3)))))));
    MB = make_float4(e0.x, e0.y, e1.x, e1.y);
    MC = e2;
    const f2 ox = fma2(bc(k.dtau_dx), e0, thx), oy = fma2(bc(k.dtau_dx), e1, thy);
    OB = make_float4(ox.x, ox.y, oy.x, oy.y);
    OC = fma2(bc(k.dtau_dx), e2, thz);
}

}  // namespace u1u1
