// diag_fused.cu -- ONE read-only sweep over the 80 B/site state for all in-loop diagnostics:
//   Gauss-law residual (Eq. 9-10), per-plaquette windings with near-branch-cut flags (:183-188, readings
//   R-12, R-15), pierced-cell arrays and the fast-method overlap count (:234, :252), Lagrangian / velocity-estimator /
//   energy sums (:196-224 Eq. 33, 36-37), largest link phase.
// Same tiling as the fused step kernel (stage.cuh): a CTA owns a 32 x 8 xy tile and marches through a z chunk; the
// position planes z, z+1 (+ halo) and the momentum plane z (+ halo, for div E) arrive in shared-memory rings by TMA box
// loads (interior tiles) or cp.async / direct loads (boundary tiles).  Persistent CTAs walk the (tile, chunk) items in
// the band order of the step kernel, so the per-CTA partial sums are few and their fold is deterministic.
//
// Windings.  With alpha = arg f per site and t_l = (alpha(x+l) - alpha(x) - theta_l(x)) / 2 pi per link, the link angle
// of reading R-12 is chi_l = 2 pi (t_l - n_l), n_l = rint(t_l), and around a plaquette the alpha's telescope and the
// theta's add up to -P_ij, so
//     W_ij(x) = rint((chi_i(x) + chi_j(x+i) - chi_i(x+j) - chi_j(x) + P_ij(x)) / 2 pi) = -(n_i(x) + n_j(x+i) - n_i(x+j) - n_j(x))
// EXACTLY: one atan2 per site and sector, one rint per link, integer adds per plaquette.  The wrap counts n_l of both
// sectors travel through shared memory as byte lanes of 32-bit words (lane 0 = p, lane 2 = q, lane 1 = flags), so a
// plaquette of both sectors is two integer adds and one VABSDIFF4.  Links with an end point that is exactly zero
// (atan2(0,0) = 0, R-15: chi = 0) or within 1e-5 of the cut are flagged and take a slow path that evaluates the
// printed formula.
#include <cstring>
#include <type_traits>

#include "common.cuh"
#include "kernels.h"
#include "stage.cuh"
#include "f32x2.cuh"
#include "winding.cuh"

namespace u1u1 {

namespace {

constexpr int NSLOT = 3;                                   // position ring: planes z, z+1 in use, z+2 in flight
constexpr int MSLOT_BYTES = 5504;                          // momentum ring slot: pack B (E_x, E_y, H_x, H_y) with halo
constexpr int OFF_MRING = NSLOT * SLOT_BYTES;
constexpr int OFF_ALPHA = OFF_MRING + 2 * MSLOT_BYTES;     // float2 [2 planes][NELEM]: the phases (alpha_p, alpha_q) of a site
constexpr int OFF_XY = OFF_ALPHA + 2 * 2 * NELEM * 4;      // uint2 [2 planes][NELEM]: wrap counts of the x and y links
constexpr int OFF_Z = OFF_XY + 2 * NELEM * 8;              // uint  [NELEM]: wrap counts of the z links of plane z
constexpr int OFF_RED = OFF_Z + NELEM * 4;                 // double [FUSED_NRES][NTHREADS / 32]: per-warp accumulators
constexpr int OFF_BARS = OFF_RED + FUSED_NRES * (NTHREADS / 32) * 8;
constexpr int SMEM_BYTES = OFF_BARS + 64;                  // 66.6 KB -> 3 CTAs per SM
static_assert(NELEM * 16 <= MSLOT_BYTES && MSLOT_BYTES % 128 == 0, "momentum slot");
static_assert(OFF_ALPHA % 16 == 0 && OFF_XY % 16 == 0 && OFF_RED % 8 == 0 && OFF_BARS % 8 == 0, "alignment");

#ifndef FUSED_CTAS
#define FUSED_CTAS 3
#endif
template <bool EXPORT>
__global__ void __launch_bounds__(NTHREADS, FUSED_CTAS)
diag_fused_kernel(const float *__restrict__ posp, const float *__restrict__ momp, size_t V, int N, FusedCoef k, int zchunk,
                  int band, uint8_t *__restrict__ cells, uint8_t *__restrict__ codes, double *__restrict__ partials,
                  const __grid_constant__ DiagMaps maps)
{
    extern __shared__ __align__(128) char smem[];
    const unsigned sbase = smem_u32(smem), bars = sbase + OFF_BARS;
    float2 *alpha = reinterpret_cast<float2 *>(smem + OFF_ALPHA);
    uint2 *XY = reinterpret_cast<uint2 *>(smem + OFF_XY);
    unsigned *ZW = reinterpret_cast<unsigned *>(smem + OFF_Z);
    double *red = reinterpret_cast<double *>(smem + OFF_RED);
    const size_t NN = (size_t)N * N;
    const int tid = threadIdx.x, tx = tid & (TX - 1), ty = tid / TX, warp = tid >> 5, lane = tid & 31;
    const char *pos = reinterpret_cast<const char *>(posp);
    const unsigned long long pol_stream = (k.flags & 32) ? policy_evict_last() : policy_evict_first();
    const unsigned long long pol_keep = (k.flags & 16) ? policy_evict_first() : policy_evict_last();
    // z extent: the whole periodic lattice, or the own planes 1 .. nz_own of a z slab (halo planes 0 and nz_own + 1 are
    // only read: positions above for the forward z neighbours, momentum pack C below for div E)
    const int NZO = k.nz_own ? k.nz_own : N, ZB = k.nz_own ? 1 : 0;
    const bool zwrap = k.nz_own == 0;
    const int ntx = (N + TX - 1) / TX, nty = (N + TY - 1) / TY, nzc = (NZO + zchunk - 1) / zchunk;
    const int items = ntx * nty * nzc;
    const float4 *gMA = reinterpret_cast<const float4 *>(momp);
    const float2 *gMC = reinterpret_cast<const float2 *>(momp + 8 * V);

    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < NSLOT + 2; b++) mbar_init(bars + 8 * b, 1);
        mbar_fence_init();
    }
    for (int i = tid; i < FUSED_NRES * (NTHREADS / 32); i += NTHREADS) red[i] = 0.0;
    __syncthreads();
    unsigned gpos = 0, gmom = 0;          // planes staged by TMA so far (ring slot and mbarrier phase bookkeeping)

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        // item -> (tile, chunk) in band order (see step_tiled.cu)
        const int full = ntx * band * nzc, bnd = item / full, rem = item - bnd * full;
        const int rows = min(band, nty - bnd * band), bzc = rem / (ntx * rows), tl = rem - bzc * (ntx * rows);
        const int x0 = (tl % ntx) * TX, y0 = (bnd * band + tl / ntx) * TY, z0 = ZB + bzc * zchunk;
        const int nz = min(zchunk, ZB + NZO - z0);
        // Two instances of the item body: interior tiles (full 32 x 8 tile, TMA staging: every tile predicate and the
        // cp.async path fold away at compile time -- 92 % of the tiles at 1024^3) and boundary / ragged tiles.
        auto run_item = [&](auto interior) {
        constexpr bool tma = decltype(interior)::value;
        const int wx = tma ? TX : min(TX, N - x0), wy = tma ? TY : min(TY, N - y0);
        const bool active = tma || (tx < wx && ty < wy);

        // this item's partial sums in fp32 (at most zchunk terms each), folded into the per-warp fp64 accumulators at its end
        f2 gf[3] = {bc(0.f), bc(0.f), bc(0.f)};     // Gauss: sum g^2, rho^2, div^2, (p, q) pairs
        float df[11] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
        float gmax[2] = {0.f, 0.f}, maxth = 0.f;
        unsigned wsum = 0, csum = 0;          // sum |W| (lanes p: bits 0..15, q: 16..31); pierced cells p, q (same lanes)
        int npq = 0, nnear = 0, maxw = 0;     // cells pierced by both; near-cut plaquettes (p: bits 0..15, q: 16..31)
        unsigned wany = 0;                    // OR of all |W| lanes: tells max|W| = 0 from 1

        // ---- staging: relative position plane j = 0 .. nz (slot = running plane count mod 3), momentum pack B (with
        // halo) of plane m = 0 .. nz-1 (slot = running count mod 2).  TMA tiles: one thread issues box loads that
        // complete on mbarriers; boundary tiles: every thread issues its cp.async copies.
        CpPlan plan;
        if (!tma) make_cp_plan(plan, tid, x0, y0, wx, wy, N);
        const unsigned pb = tma ? gpos : 0u, mb = tma ? gmom : 0u;
        auto stage_pos = [&](int j, unsigned slot) {
            const int z = zwrap ? wrapi(z0 + j, N) : z0 + j;
            if (tma) stage_plane_tma(maps.pos, x0, y0, z, sbase + slot * SLOT_BYTES, bars + 8 * slot, pol_keep);
            else stage_plane_cp(plan, tid, pos, V, (size_t)z * NN, sbase + slot * SLOT_BYTES);
        };
        auto stage_mom = [&](int m) {
            const unsigned sl = (mb + (unsigned)m) & 1u;
            if (tma) {
                const unsigned bar = bars + 8 * (NSLOT + sl);
                mbar_expect_tx(bar, NELEM * 16);
                tma_load_3d_hint(sbase + OFF_MRING + sl * MSLOT_BYTES, &maps.mom.B, 4 * (x0 - 1), y0 - 1, z0 + m, bar, pol_stream);
            } else {
                stage_packB_cp(plan, tid, reinterpret_cast<const char *>(momp), V, (size_t)(z0 + m) * NN, sbase + OFF_MRING + sl * MSLOT_BYTES);
            }
        };

        __syncthreads();                      // the previous item's readers are done with every buffer
        unsigned s_n = pb % 3u, par_n = (pb / 3u) & 1u;       // ring slot and mbarrier parity of plane iz+1 (here: plane 0)
        {
            unsigned sl = s_n;
            if (!tma || tid == 0) {
                for (int j = 0; j <= 2; j++) {
                    if (j <= nz) stage_pos(j, sl);
                    sl = sl == 2u ? 0u : sl + 1u;
                }
                stage_mom(0);
                if (nz > 1) stage_mom(1);
            }
            if (!tma) cp_async_commit();
        }

        // element indices of this thread's own site inside a staged plane
        const int e_own = (ty + 1) * COLS + tx + 1, e_ownC = (ty + 1) * CCOLS + tx + 2;
        const size_t gsite = (size_t)(y0 + ty) * N + (size_t)(x0 + tx);
        size_t lin = (size_t)z0 * NN + gsite;
        // E_z, H_z of plane z0 - 1 (for div E of the first plane)
        float2 ez_prev = make_float2(0.f, 0.f);
        if (active) ez_prev = __ldg(gMC + (size_t)(zwrap ? wrapi(z0 - 1, N) : z0 - 1) * NN + gsite);

        // extended sites: the tile plus its +x column and +y row (the cells of the last column / row need their
        // plaquettes).  Pass 1 = own element of every thread; pass 2 = the extra row (32 lanes of one warp) and the
        // extra column (9 lanes of the next warp), rotated over the warps from plane to plane to spread the load.
        const bool own_ext = tma || (tx <= wx && ty <= wy);
        const int e_row = (TY + 1) * COLS + lane + 1, e_col = (lane + 1) * COLS + TX + 1;
        auto do_alpha = [&](int e, const char *sn, int nxt) {          // phases of one site of plane `sn` into alpha[nxt]
            const float4 a = *reinterpret_cast<const float4 *>(sn + e * 16);
            alpha[nxt * NELEM + e] = site_phase2(lo(a), hi(a));
        };
        // wrap counts of the x and y links of one site of plane `sn` (links that leave the extended tile -- x links of
        // the extra column, y links of the extra row -- are evaluated on whatever the neighbouring shared-memory words
        // hold and never read), returns the site's two phases for the z links
        auto do_links_xy = [&](int e, const char *sn, int nxt, f2 &a0) {
            const float4 Bn = *reinterpret_cast<const float4 *>(sn + OFF_B + e * 16);
            const float2 *ap = alpha + nxt * NELEM + e;
            a0 = ap[0];
            XY[nxt * NELEM + e] = make_uint2(link_lane2(a0, ap[1], lo(Bn)), link_lane2(a0, ap[COLS], hi(Bn)));
        };
        auto do_links = [&](int e, const char *sc, const char *sn, int cur) {      // + the z links of plane `sc`
            f2 a0;
            do_links_xy(e, sn, cur ^ 1, a0);
            const int r = e / COLS;
            const float2 Cz = *reinterpret_cast<const float2 *>(sc + OFF_C + (e + 2 * r + 1) * 8);
            ZW[e] = link_lane2(alpha[cur * NELEM + e], a0, Cz);
        };
        auto wait_plane = [&]() {             // plane iz+1 (slot s_n) has landed
            if (tma) mbar_wait(bars + 8 * s_n, par_n);
            else {
                cp_async_wait<0>();
                __syncthreads();
            }
        };

        // ---- prologue: phases and in-plane links of plane 0, W_xy of plane 0 ----
        unsigned Pxy = 0, Qxy = 0;            // W_xy of the current plane, carried from one iteration to the next
        {
            wait_plane();
            const char *sn = smem + s_n * SLOT_BYTES;
            const bool xrow = warp == 0 && wy == TY, xcol = warp == 1 && wx == TX && lane <= TY;
            if (own_ext) do_alpha(e_own, sn, 0);
            if (xrow || xcol) do_alpha(xrow ? e_row : e_col, sn, 0);
            __syncthreads();
            f2 u;
            if (own_ext) do_links_xy(e_own, sn, 0, u);
            if (xrow || xcol) do_links_xy(xrow ? e_row : e_col, sn, 0, u);
            __syncthreads();
            if (active) {
                const uint2 Ln = XY[e_own], Lnx = XY[e_own + 1], Lny = XY[e_own + COLS];
                Pxy = Ln.x + Lnx.y;
                Qxy = Lny.x + Ln.y;
            }
        }

        unsigned s_c = s_n;                   // slot of plane iz
        for (int iz = 0; iz < nz; iz++) {
            // momenta of this thread's site: the own-site packs straight from global memory (pack B, whose -x / -y
            // neighbours div E needs, comes through the shared-memory ring)
            float4 MA = make_float4(0.f, 0.f, 0.f, 0.f);
            float2 MC = make_float2(0.f, 0.f);
            if (active) {
                MA = __ldcs(gMA + lin);
                MC = __ldcs(gMC + lin);
            }
            s_n = s_c == 2u ? 0u : s_c + 1u;
            par_n ^= s_n == 0u ? 1u : 0u;
            wait_plane();                     // plane iz+1; on boundary tiles also the momenta of plane iz
            if (tma) {
                const unsigned h = mb + (unsigned)iz;
                mbar_wait(bars + 8 * (NSLOT + (h & 1u)), (h >> 1) & 1u);
            }
            const int cur = iz & 1, nxt = cur ^ 1;
            const char *sc = smem + s_c * SLOT_BYTES, *sn = smem + s_n * SLOT_BYTES;
            const int rot = (warp - iz - 1) & 7;
            const bool xrow = rot == 0 && wy == TY, xcol = rot == 1 && wx == TX && lane <= TY;
            const bool has_extra = xrow || xcol;
            const int e_ext = xrow ? e_row : e_col;

            // ---- phase A: phases alpha of plane iz+1 on the extended tile ----
            if (own_ext) do_alpha(e_own, sn, nxt);
            if (has_extra) do_alpha(e_ext, sn, nxt);

            // ---- Gauss residual and densities of this thread's site in plane iz (independent of the windings) ----
            if (active) {
                auto A = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + (e_own + d) * 16); };
                auto B = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + OFF_B + (e_own + d) * 16); };
                auto C = [&](const char *s, int d) { return *reinterpret_cast<const float2 *>(s + OFF_C + (e_ownC + d) * 8); };
                const float4 *ms = reinterpret_cast<const float4 *>(smem + OFF_MRING + ((mb + (unsigned)iz) & 1u) * MSLOT_BYTES);
                const float4 MB = ms[e_own], MBxm = ms[e_own - 1], MBym = ms[e_own - COLS];
                const float4 Ac = A(sc, 0), Axp = A(sc, 1), Ayp = A(sc, COLS), Azp = A(sn, 0);
                const float4 Bc = B(sc, 0), Bxp = B(sc, 1), Byp = B(sc, COLS), Bzp = B(sn, 0);
                const float2 Cc = C(sc, 0), Cxp = C(sc, 1), Cyp = C(sc, CCOLS);
                // both sectors at once: a pair is (p, q) of one quantity, the 64-bit halves of the vector loads (common.cuh)
                const f2 fr = lo(Ac), fi = hi(Ac), pr = lo(MA), pi = hi(MA);
                const f2 E[3] = {lo(MB), hi(MB), MC}, Em[3] = {lo(MBxm), hi(MBym), ez_prev};
                // Gauss (Eq. 9-10): differences and the charge density in fp64 (g is a 1e-6 cancellation), per sector
                f2 gl, rl, dl;
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const double div = (((double)pkc(E[0], s) - (double)pkc(Em[0], s)) + ((double)pkc(E[1], s) - (double)pkc(Em[1], s)) +
                                        ((double)pkc(E[2], s) - (double)pkc(Em[2], s))) * k.inv_dx;
                    const double rho = (s ? k.rho2 : k.rho1) * ((double)pkc(fr, s) * (double)pkc(pi, s) - (double)pkc(fi, s) * (double)pkc(pr, s));
                    const float g_ = (float)(div - rho), r_ = (float)rho, d_ = (float)div;
                    if (s) { gl.y = g_; rl.y = r_; dl.y = d_; } else { gl.x = g_; rl.x = r_; dl.x = d_; }
                    gmax[s] = fmaxf(gmax[s], fabsf(g_));
                }
                gf[0] = fma2(gl, gl, gf[0]);
                gf[1] = fma2(rl, rl, gf[1]);
                gf[2] = fma2(dl, dl, gf[2]);
                // densities (fp32 per-site terms, packed fp32x2)
                const f2 kin2 = fma2(pr, pr, mul2(pi, pi)), m2 = fma2(fr, fr, mul2(fi, fi));
                const f2 th[3] = {lo(Bc), hi(Bc), Cc};
                const f2 nr[3] = {lo(Axp), lo(Ayp), lo(Azp)}, ni[3] = {hi(Axp), hi(Ayp), hi(Azp)};
                f2 g2 = bc(0.f), e2 = bc(0.f);
#pragma unroll
                for (int i = 0; i < 3; i++) {
                    f2 sn_, cs_;
                    __sincosf(th[i].x, &sn_.x, &cs_.x);             // U = exp(-i theta): SFU phasor (abs. error ~5e-7)
                    __sincosf(th[i].y, &sn_.y, &cs_.y);
                    const f2 dr = fma2(cs_, nr[i], fma2(sn_, ni[i], neg(fr))), di = fma2(cs_, ni[i], fma2(neg(sn_), nr[i], neg(fi)));
                    g2 = fma2(dr, dr, fma2(di, di, g2));
                    e2 = fma2(E[i], E[i], e2);
                    maxth = fmaxf(maxth, fmaxf(fabsf(th[i].x), fabsf(th[i].y)));
                }
                // plaquettes (i, j) = (x,y), (x,z), (y,z)
                const f2 P0 = sub2(sub2(add2(th[0], hi(Bxp)), lo(Byp)), th[1]);
                const f2 P1 = sub2(sub2(add2(th[0], Cxp), lo(Bzp)), th[2]);
                const f2 P2 = sub2(sub2(add2(th[1], Cyp), hi(Bzp)), th[2]);
                const f2 gw = mul2(g2, bc(k.inv_dx2)), ew = mul2(e2, make_float2(k.el1, k.el2));
                const f2 mw = mul2(fma2(P0, P0, fma2(P1, P1, mul2(P2, P2))), make_float2(k.mg1, k.mg2));
                const float kin = kin2.x + kin2.y, grad = gw.x + gw.y, elec = ew.x + ew.y, mag = mw.x + mw.y;
                ez_prev = MC;
                const float a2 = m2.x - k.sig1sq, b2 = m2.y - k.sig2sq;
                const float vint = k.kappa * a2 * b2;
                const float pot = k.lam1q * a2 * a2 + k.lam2q * b2 * b2 - vint;
                const float lag = kin - grad + (elec - mag) * k.inv_c - k.c * pot;
                df[0] += lag;
                df[1] = fmaf(kin, lag, df[1]);
                df[2] = fmaf(grad, lag, df[2]);
                df[3] = fmaf(kin, vint, df[3]);
                df[4] = fmaf(grad, vint, df[4]);
                df[5] += vint;
                df[6] += kin;
                df[7] += grad;
                df[8] += elec;
                df[9] += mag;
                df[10] += pot;
            }
            __syncthreads();                  // alpha of plane iz+1 complete; everybody is past iteration iz-1
            if (!tma || tid == 0) {
                if (iz >= 1 && iz + 2 <= nz) stage_pos(iz + 2, s_n == 2u ? 0u : s_n + 1u);      // the slot of plane iz-1
                if (iz + 2 < nz) stage_mom(iz + 2);                                             // the slot of plane iz, consumed in phase A
            }
            if (!tma) cp_async_commit();

            // ---- phase B: wrap counts of the x, y links of plane iz+1 and of the z links of plane iz ----
            if (own_ext) do_links(e_own, sc, sn, cur);
            if (has_extra) do_links(e_ext, sc, sn, cur);
            __syncthreads();

            // ---- phase C: windings, cells, counters of this thread's site ----
            if (active) {
                const uint2 Ln = XY[nxt * NELEM + e_own], Lnx = XY[nxt * NELEM + e_own + 1], Lny = XY[nxt * NELEM + e_own + COLS];
                // W_xy of plane iz+1: S = n_x(x) + n_y(x+x) - n_x(x+y) - n_y(x);  W = -S
                const unsigned Pn = Ln.x + Lnx.y, Qn = Lny.x + Ln.y;
                const uint2 Lc = XY[cur * NELEM + e_own], Lcx = XY[cur * NELEM + e_own + 1], Lcy = XY[cur * NELEM + e_own + COLS];
                const unsigned Z0 = ZW[e_own], Zx = ZW[e_own + 1], Zy = ZW[e_own + COLS], Zxy = ZW[e_own + COLS + 1];
                // W_yz(x): n_y(x) + n_z(x+y) - n_y(x+z) - n_z(x);   W_zx(x): n_z(x) + n_x(x+z) - n_z(x+x) - n_x(x)
                unsigned P[6], Q[6];
                P[0] = Pxy;            Q[0] = Qxy;                 // xy, plane iz (own)
                P[1] = Lc.y + Zy;      Q[1] = Ln.y + Z0;           // yz (own)
                P[2] = Z0 + Ln.x;      Q[2] = Zx + Lc.x;           // zx (own)
                P[3] = Lcx.y + Zxy;    Q[3] = Lnx.y + Zx;          // yz at x + x
                P[4] = Zy + Lny.x;     Q[4] = Zxy + Lcy.x;         // zx at x + y
                P[5] = Pn;             Q[5] = Qn;                  // xy, plane iz+1
                unsigned Eabs[6], flagged = 0;
#pragma unroll
                for (int q = 0; q < 6; q++) {
                    Eabs[q] = __vabsdiffu4(P[q], Q[q]);             // lanes 1 / 3 (flags) hold rubbish: masked after summing
                    flagged |= P[q] | Q[q];
                }
                int wsg[2][3];                                      // signed windings of the own plaquettes (EXPORT)
                unsigned nearbits = 0;                              // bit 3 s + o
                if (EXPORT) {
#pragma unroll
                    for (int o = 0; o < 3; o++) {
                        wsg[0][o] = (int)(Q[o] & 0xffu) - (int)(P[o] & 0xffu);
                        wsg[1][o] = (int)((Q[o] >> 16) & 0xffu) - (int)((P[o] >> 16) & 0xffu);
                    }
                }
                if (flagged & FLAG_LANES) {
                    // slow path: a plaquette with a flagged link is re-evaluated link by link from the staged fields
                    // (same arithmetic as phases A and B, so the classification is consistent): near-cut flag of the
                    // own plaquettes; with a degenerate link (chi = 0 there, reading R-15) the printed formula
                    auto ph = [&](const char *s, int e, int sec) {
                        const float4 a = *reinterpret_cast<const float4 *>(s + e * 16);
                        return site_phase(pk0(a, sec), pk1(a, sec));
                    };
                    auto th_xy = [&](const char *s, int e, int sec, int dir) {
                        const float4 b = *reinterpret_cast<const float4 *>(s + OFF_B + e * 16);
                        return dir == 0 ? pk0(b, sec) : pk1(b, sec);
                    };
                    auto th_z = [&](const char *s, int e, int sec) {
                        const int r = e / COLS;
                        const float2 cz = *reinterpret_cast<const float2 *>(s + OFF_C + (e + 2 * r + 1) * 8);
                        return sec ? cz.y : cz.x;
                    };
                    for (int q = 0; q < 6; q++) {
                        for (int sec = 0; sec < 2; sec++) {
                            unsigned fl = 0;                    // (registers only: no dynamic indexing of P, Q)
#pragma unroll
                            for (int qq = 0; qq < 6; qq++)
                                if (qq == q) fl = P[qq] | Q[qq];
                            if (!((fl >> (8 + 16 * sec)) & 0xffu)) continue;
                            const int eb = e_own + (q == 3 ? 1 : q == 4 ? COLS : 0);
                            const char *s0 = q == 5 ? sn : sc;
                            float a00, a10, a01, a11, t[4];    // corners x, x+i, x+j, x+i+j; links i(x), j(x+i), i(x+j), j(x)
                            if (q == 0 || q == 5) {             // (i, j) = (x, y)
                                a00 = ph(s0, eb, sec); a10 = ph(s0, eb + 1, sec); a01 = ph(s0, eb + COLS, sec); a11 = ph(s0, eb + COLS + 1, sec);
                                t[0] = th_xy(s0, eb, sec, 0); t[1] = th_xy(s0, eb + 1, sec, 1); t[2] = th_xy(s0, eb + COLS, sec, 0); t[3] = th_xy(s0, eb, sec, 1);
                            } else if (q == 1 || q == 3) {      // (y, z)
                                a00 = ph(sc, eb, sec); a10 = ph(sc, eb + COLS, sec); a01 = ph(sn, eb, sec); a11 = ph(sn, eb + COLS, sec);
                                t[0] = th_xy(sc, eb, sec, 1); t[1] = th_z(sc, eb + COLS, sec); t[2] = th_xy(sn, eb, sec, 1); t[3] = th_z(sc, eb, sec);
                            } else {                            // (z, x)
                                a00 = ph(sc, eb, sec); a10 = ph(sn, eb, sec); a01 = ph(sc, eb + 1, sec); a11 = ph(sn, eb + 1, sec);
                                t[0] = th_z(sc, eb, sec); t[1] = th_xy(sn, eb, sec, 0); t[2] = th_z(sc, eb + 1, sec); t[3] = th_xy(sc, eb, sec, 0);
                            }
                            const float da[4] = {a10 - a00, a11 - a10, a11 - a01, a01 - a00};
                            float chi[4];
                            bool near = false, deg = false;
#pragma unroll
                            for (int l = 0; l < 4; l++) {
                                const float tl_ = (da[l] - t[l]) * INV_2PI, d = tl_ - rintf(tl_);
                                deg |= d != d;
                                near |= fabsf(d) > NEAR_T;
                                chi[l] = d != d ? 0.f : d * 6.2831853071795865f;
                            }
                            if (deg) {
                                const float sum = chi[0] + chi[1] - chi[2] - chi[3] + (t[0] + t[1] - t[2] - t[3]);
                                const unsigned aW = (unsigned)abs(__float2int_rn(sum * INV_2PI));
                                const int W = __float2int_rn(sum * INV_2PI);
#pragma unroll
                                for (int qq = 0; qq < 6; qq++)
                                    if (qq == q) Eabs[qq] = (Eabs[qq] & VAL_LANES & ~(0xffu << (16 * sec))) | (aW << (16 * sec));
                                if (EXPORT) {
#pragma unroll
                                    for (int o = 0; o < 3; o++)
                                        if (o == q) { if (sec) wsg[1][o] = W; else wsg[0][o] = W; }
                                }
                            }
                            if (near && q < 3) nearbits |= 1u << (3 * sec + q);
                        }
                    }
                    nnear += __popc(nearbits & 7u) + (__popc(nearbits & 56u) << 16);
                }
                // own plaquettes: length sums, largest winding (|W| >= 2 is rare: exact maximum only then)
                const unsigned own = (Eabs[0] + Eabs[1] + Eabs[2]) & VAL_LANES;
                wsum += own;
                wany |= own;
                if (own & 0x00fe00feu) {                            // a lane sum >= 2: maybe a |W| >= 2
#pragma unroll
                    for (int q = 0; q < 3; q++) maxw = max(maxw, (int)max(Eabs[q] & 0xffu, (Eabs[q] >> 16) & 0xffu));
                }
                // pierced cells: the six faces of the cell at x
                const unsigned cell = (own + Eabs[3] + Eabs[4] + Eabs[5]) & VAL_LANES;
                cells[lin] = (uint8_t)cell;
                cells[V + lin] = (uint8_t)(cell >> 16);
                const unsigned nzl = ((cell + 0x00ff00ffu) >> 8) & 0x00010001u;      // 1 per lane whose cell is pierced
                csum += nzl;
                npq += (int)(nzl & (nzl >> 16));
                if (EXPORT) {
#pragma unroll
                    for (int sec = 0; sec < 2; sec++)
#pragma unroll
                        for (int o = 0; o < 3; o++)
                            codes[(size_t)(3 * sec + o) * V + lin] =
                                (uint8_t)(((wsg[sec][o] + 8) & 15) | (((nearbits >> (3 * sec + o)) & 1u) << 4));
                }
                Pxy = Pn;
                Qxy = Qn;
            }
            s_c = s_n;
            lin += NN;
        }
        if (!tma) cp_async_wait<0>();
        if (tma) { gpos += (unsigned)(nz + 1); gmom += (unsigned)nz; }

        // ---- fold this item's partials into the per-warp fp64 accumulators (fixed order: deterministic) ----
        auto add = [&](int slot, double v) { if (lane == 0) red[slot * (NTHREADS / 32) + warp] += v; };
        auto amax = [&](int slot, double v) { if (lane == 0) red[slot * (NTHREADS / 32) + warp] = fmax(red[slot * (NTHREADS / 32) + warp], v); };
#pragma unroll
        for (int i = 0; i < 6; i++) add(FR_GAUSS + i, warp_sum((double)pkc(gf[i % 3], i / 3)));
#pragma unroll
        for (int i = 0; i < 11; i++) add(FR_DENS + i, warp_sum((double)df[i]));
        add(FR_SUMW, (double)__reduce_add_sync(0xffffffffu, wsum & 0xffffu));
        add(FR_SUMW + 1, (double)__reduce_add_sync(0xffffffffu, wsum >> 16));
        add(FR_NEAR, (double)__reduce_add_sync(0xffffffffu, (unsigned)nnear & 0xffffu));
        add(FR_NEAR + 1, (double)__reduce_add_sync(0xffffffffu, (unsigned)nnear >> 16));
        add(FR_CELLS, (double)__reduce_add_sync(0xffffffffu, csum & 0xffffu));
        add(FR_CELLS + 1, (double)__reduce_add_sync(0xffffffffu, csum >> 16));
        add(FR_CELLS + 2, (double)__reduce_add_sync(0xffffffffu, (unsigned)npq));
        amax(FR_GMAX, (double)__uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(gmax[0]))));
        amax(FR_GMAX + 1, (double)__uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(gmax[1]))));
        amax(FR_MAXW, (double)__reduce_max_sync(0xffffffffu, (unsigned)max(maxw, wany ? 1 : 0)));
        amax(FR_MAXTH, (double)__uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(maxth))));
        };
        if (!(k.flags & 2) && tile_is_interior(x0, y0, N)) run_item(std::true_type{});
        else run_item(std::false_type{});
    }

    // ---- per-CTA partials: the 8 warps' accumulators in fixed order ----
    __syncthreads();
    if (tid < FUSED_NRES) {
        double r = red[tid * (NTHREADS / 32)];
        for (int w = 1; w < NTHREADS / 32; w++)
            r = tid < FUSED_NSUM ? r + red[tid * (NTHREADS / 32) + w] : fmax(r, red[tid * (NTHREADS / 32) + w]);
        partials[(size_t)blockIdx.x * RED_SLOTS + tid] = r;
    }
}

}  // namespace

// z planes per work item.  Longer chunks amortise the prologue (phases and in-plane links of the chunk's first plane)
// and the extra boundary plane: measured at 1024^3, 16 planes 30.2 ms, 32: 28.8, 64: 28.3.  The per-item fp32 partial
// sums hold at most this many terms.
int fused_zchunk(int N) { return N >= 64 ? 64 : N; }

cudaError_t launch_diag_fused(const float *pos, const float *mom, size_t V, int N, FusedCoef k, uint8_t *cells, uint8_t *codes,
                              double *partials, int *nblocks, const DiagMaps *maps, int sms, cudaStream_t st)
{
    DiagMaps m;
    if (maps) m = *maps;
    else {
        memset(&m, 0, sizeof m);
        k.flags |= 2;
    }
    const int nzo = k.nz_own ? k.nz_own : N;              // planes to sweep: the lattice, or the own planes of a z slab
    int zc = (k.flags & 64) ? 16 : (k.flags & 128) ? 32 : fused_zchunk(N);   // tuning flags
    if (zc > nzo) zc = nzo;
    const int ntx = (N + TX - 1) / TX, nty = (N + TY - 1) / TY, nzc = (nzo + zc - 1) / zc;
    const long items = (long)ntx * nty * nzc;
    long grid = (long)sms * FUSED_CTAS;
    if (grid > RED_MAX_BLOCKS) grid = RED_MAX_BLOCKS;
    if (grid > items) grid = items;
    int band = (int)((grid + ntx - 1) / ntx);
    if (band > nty) band = nty;
    if (band < 1) band = 1;
    cudaError_t e;
    if (codes) {
        e = cudaFuncSetAttribute(diag_fused_kernel<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
        diag_fused_kernel<true><<<(unsigned)grid, NTHREADS, SMEM_BYTES, st>>>(pos, mom, V, N, k, zc, band, cells, codes, partials, m);
    } else {
        e = cudaFuncSetAttribute(diag_fused_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
        if (e != cudaSuccess) return e;
        diag_fused_kernel<false><<<(unsigned)grid, NTHREADS, SMEM_BYTES, st>>>(pos, mom, V, N, k, zc, band, cells, codes, partials, m);
    }
    *nblocks = (int)grid;
    return cudaGetLastError();
}

}  // namespace u1u1
