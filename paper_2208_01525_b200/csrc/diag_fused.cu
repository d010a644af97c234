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

#include "common.cuh"
#include "kernels.h"
#include "stage.cuh"

namespace u1u1 {

namespace {

constexpr int NSLOT = 4;                                   // position ring: planes z, z+1 in use, z+2, z+3 in flight
constexpr int NMSLOT = 2;                                  // momentum ring: plane z in use, z+1 in flight
constexpr int OFF_MRING = NSLOT * SLOT_BYTES;
constexpr int OFF_ALPHA = OFF_MRING + NMSLOT * SLOT_BYTES; // float [2 planes][2 sectors][NELEM]
constexpr int OFF_XY = OFF_ALPHA + 2 * 2 * NELEM * 4;      // uint2 [2 planes][NELEM]: wrap counts of the x and y links
constexpr int OFF_Z = OFF_XY + 2 * NELEM * 8;              // uint  [NELEM]: wrap counts of the z links of plane z
constexpr int OFF_RED = OFF_Z + NELEM * 4;                 // double [FUSED_NRES][NTHREADS / 32]
constexpr int OFF_BARS = OFF_RED + FUSED_NRES * (NTHREADS / 32) * 8;
constexpr int SMEM_BYTES = OFF_BARS + 64;
static_assert(OFF_ALPHA % 16 == 0 && OFF_XY % 16 == 0 && OFF_RED % 8 == 0 && OFF_BARS % 8 == 0, "alignment");

constexpr float INV_2PI = 0.15915494309189535f;
constexpr float NEAR_T = 0.5f - 1.5915494e-6f;             // pi - |chi| < 1e-5  <=>  |t - rint t| > 1/2 - 1e-5 / 2 pi
constexpr unsigned BIAS = 32u;                             // wrap counts are stored as n + 32 in a byte lane
constexpr unsigned FLAG_LANES = 0xff00ff00u, VAL_LANES = 0x00ff00ffu;   // lanes 0 / 2: p / q values, lanes 1 / 3: their flags

// atan2 in ~20 instructions: octant reduction to t = min/max in [0, 1] and the degree-8 (in t^2) polynomial of
// Abramowitz & Stegun 4.4.49 (|error| <= 2e-8 in exact arithmetic; ~4e-7 in fp32 with the fast division).
// Never called with x = y = 0.
__device__ inline float atan2_poly(float y, float x)
{
    const float ax = fabsf(x), ay = fabsf(y);
    const float t = __fdividef(fminf(ax, ay), fmaxf(ax, ay)), s = t * t;
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
    return copysignf(r, y);
}
// phase of a site, NaN if the field is exactly zero there (the links that touch it are "degenerate")
__device__ inline float site_phase(float re, float im)
{
    return (re == 0.f && im == 0.f) ? __int_as_float(0x7fc00000) : atan2_poly(im, re);
}

// One link: wrap count n = rint(t) as a biased byte (valid for |n| <= 31, i.e. |theta| < 190; the host checks the
// largest |theta| of the sweep), flags in the next byte: bit 0 = within 1e-5 of the cut, bit 2 = degenerate.
__device__ inline unsigned link_lane(float alpha_a, float alpha_b, float theta)
{
    const float t = ((alpha_b - alpha_a) - theta) * INV_2PI;          // NaN if an end point is exactly zero
    const float nf = rintf(t);
    const unsigned near = fabsf(t - nf) > NEAR_T ? 1u : 0u;           // NaN compares false
    const unsigned deg = t != t ? 4u : 0u;
    const int n = __float2int_rn(t);                                  // NaN -> 0
    return ((unsigned)(n + (int)BIAS) & 0x3fu) | ((near | deg) << 8);
}

// link angle of the printed formula, for the slow path only
__device__ inline float chi_slow(float alpha_a, float alpha_b, float theta)
{
    const float t = ((alpha_b - alpha_a) - theta) * INV_2PI;
    const float r = (t - rintf(t)) * 6.2831853071795865f;
    return r != r ? 0.f : r;                                          // atan2(0, 0) = 0 (reading R-15)
}

struct Acc {
    double g[6];          // sum g^2, rho^2, div^2 per sector
    double d[11];         // sum L, kin L, grad L, kin V, grad V, V, kin, grad, elec, mag, pot
    double gmax[2];
    unsigned wsum;        // sum |W| of this item, lanes p (bits 0..15) and q (16..31)
    int sumw[2], nnear[2], ncell[3], maxw;
    float maxth;
};

template <bool EXPORT>
__global__ void __launch_bounds__(NTHREADS, 2)
diag_fused_kernel(const float *__restrict__ posp, const float *__restrict__ momp, size_t V, int N, FusedCoef k, int zchunk,
                  int band, uint8_t *__restrict__ cells, uint8_t *__restrict__ codes, double *__restrict__ partials,
                  const __grid_constant__ DiagMaps maps)
{
    extern __shared__ __align__(128) char smem[];
    const unsigned sbase = smem_u32(smem), bars = sbase + OFF_BARS;
    float *alpha = reinterpret_cast<float *>(smem + OFF_ALPHA);
    uint2 *XY = reinterpret_cast<uint2 *>(smem + OFF_XY);
    unsigned *ZW = reinterpret_cast<unsigned *>(smem + OFF_Z);
    const size_t NN = (size_t)N * N;
    const int tid = threadIdx.x, tx = tid & (TX - 1), ty = tid / TX, warp = tid >> 5;
    const char *pos = reinterpret_cast<const char *>(posp);
    const unsigned long long pol_stream = policy_evict_first(), pol_keep = policy_evict_last();
    const int ntx = (N + TX - 1) / TX, nty = (N + TY - 1) / TY, nzc = (N + zchunk - 1) / zchunk;
    const int items = ntx * nty * nzc;

    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < NSLOT + NMSLOT; b++) mbar_init(bars + 8 * b, 1);
        mbar_fence_init();
    }
    __syncthreads();

    Acc acc;
#pragma unroll
    for (int i = 0; i < 6; i++) acc.g[i] = 0.0;
#pragma unroll
    for (int i = 0; i < 11; i++) acc.d[i] = 0.0;
    acc.gmax[0] = acc.gmax[1] = 0.0;
    acc.sumw[0] = acc.sumw[1] = acc.nnear[0] = acc.nnear[1] = acc.ncell[0] = acc.ncell[1] = acc.ncell[2] = acc.maxw = 0;
    acc.maxth = 0.f;
    unsigned gpos = 0, gmom = 0;          // planes staged by TMA so far (ring slot and mbarrier phase bookkeeping)

    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        // item -> (tile, chunk) in band order (see step_tiled.cu)
        const int full = ntx * band * nzc, bnd = item / full, rem = item - bnd * full;
        const int rows = min(band, nty - bnd * band), bzc = rem / (ntx * rows), tl = rem - bzc * (ntx * rows);
        const int x0 = (tl % ntx) * TX, y0 = (bnd * band + tl / ntx) * TY, z0 = bzc * zchunk;
        const int wx = min(TX, N - x0), wy = min(TY, N - y0), nz = min(zchunk, N - z0);
        const bool active = tx < wx && ty < wy;
        const bool tma = !(k.flags & 2) && tile_is_interior(x0, y0, N);
        acc.wsum = 0;

        // ---- staging: relative position plane j = 0 .. nz, momentum plane m = 0 .. nz-1 ----
        CpPlan plan;
        if (!tma) make_cp_plan(plan, tid, x0, y0, wx, wy, N);
        auto pslot = [&](int j) { return tma ? (gpos + (unsigned)j) & 3u : (unsigned)j & 3u; };
        auto stage_pos = [&](int j) {         // TMA: one thread; cp.async: every thread (caller commits)
            const int z = wrapi(z0 + j, N);
            if (tma) stage_plane_tma(maps.pos, x0, y0, z, sbase + pslot(j) * SLOT_BYTES, bars + 8 * pslot(j), pol_keep);
            else stage_plane_cp(plan, tid, pos, V, (size_t)z * NN, sbase + pslot(j) * SLOT_BYTES);
        };
        auto mslot = [&](int m) { return (gmom + (unsigned)m) & 1u; };
        auto stage_mom = [&](int m) {         // TMA tiles only, one thread
            stage_plane_tma(maps.mom, x0, y0, z0 + m, sbase + OFF_MRING + mslot(m) * SLOT_BYTES, bars + 8 * (NSLOT + mslot(m)),
                            pol_stream);
        };
        auto wait_pos = [&](int j) {          // TMA only
            const unsigned g = gpos + (unsigned)j;
            mbar_wait(bars + 8 * (g & 3u), (g >> 2) & 1u);
        };
        auto wait_mom = [&](int m) {
            const unsigned g = gmom + (unsigned)m;
            mbar_wait(bars + 8 * (NSLOT + (g & 1u)), (g >> 1) & 1u);
        };

        __syncthreads();                      // the previous item's readers are done with every buffer
        if (tma) {                            // planes 0, 1 now; plane iz+3 during iteration iz = -1, 0, ...
            if (tid == 0) {
                stage_pos(0);
                stage_pos(1);
                stage_mom(0);
                if (nz > 1) stage_mom(1);
            }
        } else {
            for (int j = 0; j <= 1; j++) {
                stage_pos(j);
                cp_async_commit();
            }
        }

        // element indices of this thread's own site inside a staged plane
        const int e_own = (ty + 1) * COLS + tx + 1, e_ownC = (ty + 1) * CCOLS + tx + 2;
        const size_t gsite = (size_t)(y0 + ty) * N + (size_t)(x0 + tx);
        // E_z, H_z of plane z0 - 1 (for div E of the first plane)
        float2 ez_prev = make_float2(0.f, 0.f);
        if (active) ez_prev = __ldg(reinterpret_cast<const float2 *>(momp + 8 * V) + (size_t)wrapi(z0 - 1, N) * NN + gsite);
        unsigned Pxy = 0, Qxy = 0, Fxy = 0;   // W_xy of the current plane (and its links' flags), carried from the previous iteration

        // extended sites: the tile plus its +x column and +y row (needed by the cells of the last column / row).
        // Pass 1 = own element of every thread; pass 2 = the extra row (one warp) and the extra column (9 lanes of the
        // next warp), rotated over the warps from plane to plane to spread the load.
        auto extra_elem = [&](int iz, int &c, int &r) -> bool {
            const int w0 = (iz + 1) & 7, lane = tid & 31;
            if (warp == w0 && wy == TY) { c = lane; r = TY; return c <= wx && (c < TX); }
            if (warp == ((w0 + 1) & 7) && wx == TX) { c = TX; r = lane; return r <= wy && (r <= TY); }
            return false;
        };

        for (int iz = -1; iz < nz; iz++) {
            // ---- plane iz+1 must have landed (and the momenta of plane iz) ----
            if (tma) {
                wait_pos(iz + 1);
                if (iz >= 0) wait_mom(iz);
            } else {
                cp_async_wait<1>();
                __syncthreads();
                if (iz + 3 <= nz) stage_pos(iz + 3);      // slot of plane iz-1: every thread is past its last read
                cp_async_commit();
            }
            const int cur = iz & 1, nxt = cur ^ 1;
            const char *sc = smem + pslot(iz < 0 ? 0 : iz) * SLOT_BYTES;      // plane iz (unused for iz = -1)
            const char *sn = smem + pslot(iz + 1) * SLOT_BYTES;               // plane iz+1

            // ---- phase A: phases alpha of plane iz+1 on the extended tile ----
            auto do_alpha = [&](int c, int r) {
                const int e = (r + 1) * COLS + c + 1;
                const float4 a = *reinterpret_cast<const float4 *>(sn + e * 16);
                alpha[(nxt * 2 + 0) * NELEM + e] = site_phase(a.x, a.y);
                alpha[(nxt * 2 + 1) * NELEM + e] = site_phase(a.z, a.w);
            };
            if (tx <= wx && ty <= wy) do_alpha(tx, ty);
            {
                int c, r;
                if (extra_elem(iz, c, r)) do_alpha(c, r);
            }

            // ---- Gauss residual and densities of this thread's site in plane iz (independent of the windings) ----
            if (iz >= 0 && active) {
                const size_t lin = (size_t)(z0 + iz) * NN + gsite;
                auto A = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + (e_own + d) * 16); };
                auto B = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + OFF_B + (e_own + d) * 16); };
                auto C = [&](const char *s, int d) { return *reinterpret_cast<const float2 *>(s + OFF_C + (e_ownC + d) * 8); };
                float4 MA, MB, MBxm, MBym;
                float2 MC;
                if (tma) {
                    const char *ms = smem + OFF_MRING + mslot(iz) * SLOT_BYTES;
                    MA = A(ms, 0); MB = B(ms, 0); MBxm = B(ms, -1); MBym = B(ms, -COLS); MC = C(ms, 0);
                } else {
                    const float4 *gA = reinterpret_cast<const float4 *>(momp), *gB = reinterpret_cast<const float4 *>(momp + 4 * V);
                    const size_t zp = (size_t)(z0 + iz) * NN;
                    const int x = x0 + tx, y = y0 + ty;
                    MA = __ldcs(gA + lin);
                    MB = __ldcs(gB + lin);
                    MBxm = __ldg(gB + zp + (size_t)y * N + wrapi(x - 1, N));
                    MBym = __ldg(gB + zp + (size_t)wrapi(y - 1, N) * N + x);
                    MC = __ldcs(reinterpret_cast<const float2 *>(momp + 8 * V) + lin);
                }
                const float4 Ac = A(sc, 0), Axp = A(sc, 1), Ayp = A(sc, COLS), Azp = A(sn, 0);
                const float4 Bc = B(sc, 0), Bxp = B(sc, 1), Byp = B(sc, COLS), Bzp = B(sn, 0);
                const float2 Cc = C(sc, 0), Cxp = C(sc, 1), Cyp = C(sc, CCOLS);
                float kin = 0.f, grad = 0.f, elec = 0.f, mag = 0.f, m2[2];
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const float fr = s ? Ac.z : Ac.x, fi = s ? Ac.w : Ac.y;
                    const float pr = s ? MA.z : MA.x, pi = s ? MA.w : MA.y;
                    // Gauss (Eq. 9-10): differences and the charge density in fp64 (g is a 1e-6 cancellation)
                    const float E[3] = {s ? MB.z : MB.x, s ? MB.w : MB.y, s ? MC.y : MC.x};
                    const float Em[3] = {s ? MBxm.z : MBxm.x, s ? MBym.w : MBym.y, s ? ez_prev.y : ez_prev.x};
                    double div = 0.0;
#pragma unroll
                    for (int i = 0; i < 3; i++) div += ((double)E[i] - (double)Em[i]) * k.inv_dx;
                    const double rho = (s ? k.rho2 : k.rho1) * ((double)fr * (double)pi - (double)fi * (double)pr);
                    const double g = div - rho;
                    acc.g[3 * s + 0] += g * g;
                    acc.g[3 * s + 1] += rho * rho;
                    acc.g[3 * s + 2] += div * div;
                    acc.gmax[s] = fmax(acc.gmax[s], fabs(g));
                    // densities (fp32 per-site terms)
                    kin += pr * pr + pi * pi;
                    m2[s] = fr * fr + fi * fi;
                    const float th[3] = {s ? Bc.z : Bc.x, s ? Bc.w : Bc.y, s ? Cc.y : Cc.x};
                    const float nr[3] = {s ? Axp.z : Axp.x, s ? Ayp.z : Ayp.x, s ? Azp.z : Azp.x};
                    const float ni[3] = {s ? Axp.w : Axp.y, s ? Ayp.w : Ayp.y, s ? Azp.w : Azp.y};
                    float g2 = 0.f, e2 = 0.f;
#pragma unroll
                    for (int i = 0; i < 3; i++) {
                        float sn_, cs_;
                        __sincosf(th[i], &sn_, &cs_);               // U = exp(-i theta): SFU phasor (abs. error ~5e-7)
                        const float dr = (cs_ * nr[i] + sn_ * ni[i]) - fr, di = (cs_ * ni[i] - sn_ * nr[i]) - fi;
                        g2 += dr * dr + di * di;
                        e2 += E[i] * E[i];
                        acc.maxth = fmaxf(acc.maxth, fabsf(th[i]));
                    }
                    // plaquettes (i, j) = (x,y), (x,z), (y,z)
                    const float ty_x = s ? Bxp.w : Bxp.y, tx_y = s ? Byp.z : Byp.x;
                    const float tz_x = s ? Cxp.y : Cxp.x, tx_z = s ? Bzp.z : Bzp.x;
                    const float tz_y = s ? Cyp.y : Cyp.x, ty_z = s ? Bzp.w : Bzp.y;
                    const float P0 = th[0] + ty_x - tx_y - th[1], P1 = th[0] + tz_x - tx_z - th[2], P2 = th[1] + tz_y - ty_z - th[2];
                    grad += g2 * k.inv_dx2;
                    elec += e2 * (s ? k.el2 : k.el1);
                    mag += (P0 * P0 + P1 * P1 + P2 * P2) * (s ? k.mg2 : k.mg1);
                }
                ez_prev = MC;
                const float a2 = m2[0] - k.sig1sq, b2 = m2[1] - k.sig2sq;
                const float vint = k.kappa * a2 * b2;
                const float pot = k.lam1q * a2 * a2 + k.lam2q * b2 * b2 - vint;
                const float lag = kin - grad + (elec - mag) * k.inv_c - k.c * pot;
                acc.d[0] += (double)lag;
                acc.d[1] += (double)(kin * lag);
                acc.d[2] += (double)(grad * lag);
                acc.d[3] += (double)(kin * vint);
                acc.d[4] += (double)(grad * vint);
                acc.d[5] += (double)vint;
                acc.d[6] += (double)kin;
                acc.d[7] += (double)grad;
                acc.d[8] += (double)elec;
                acc.d[9] += (double)mag;
                acc.d[10] += (double)pot;
            }
            __syncthreads();                  // alpha of plane iz+1 complete; momenta of plane iz consumed
            if (tma && tid == 0) {
                if (iz + 3 <= nz) stage_pos(iz + 3);          // slot of plane iz-1: every thread is past iteration iz-1
                if (iz >= 0 && iz + 2 < nz) stage_mom(iz + 2);        // slot of plane iz, consumed in phase A
            }

            // ---- phase B: wrap counts of the x, y links of plane iz+1 and of the z links of plane iz ----
            auto do_links = [&](int c, int r) {
                const int e = (r + 1) * COLS + c + 1;
                const float4 Bn = *reinterpret_cast<const float4 *>(sn + OFF_B + e * 16);
                unsigned X = 0, Y = 0, Z = 0;
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const float *an = alpha + (nxt * 2 + s) * NELEM;
                    const float a0 = an[e];
                    X |= (c < wx ? link_lane(a0, an[e + 1], s ? Bn.z : Bn.x) : BIAS) << (16 * s);
                    Y |= (r < wy ? link_lane(a0, an[e + COLS], s ? Bn.w : Bn.y) : BIAS) << (16 * s);
                    if (iz >= 0) {
                        const float2 Cz = *reinterpret_cast<const float2 *>(sc + OFF_C + ((r + 1) * CCOLS + c + 2) * 8);
                        Z |= link_lane(alpha[(cur * 2 + s) * NELEM + e], a0, s ? Cz.y : Cz.x) << (16 * s);
                    }
                }
                XY[nxt * NELEM + e] = make_uint2(X, Y);
                if (iz >= 0) ZW[e] = Z;
            };
            if (tx <= wx && ty <= wy) do_links(tx, ty);
            {
                int c, r;
                if (extra_elem(iz, c, r)) do_links(c, r);
            }
            __syncthreads();

            // ---- phase C: windings, cells, counters of this thread's site ----
            if (active) {
                const uint2 Ln = XY[nxt * NELEM + e_own], Lnx = XY[nxt * NELEM + e_own + 1], Lny = XY[nxt * NELEM + e_own + COLS];
                // W_xy of plane iz+1: S = n_x(x) + n_y(x+x) - n_x(x+y) - n_y(x);  W = -S
                const unsigned Pn = Ln.x + Lnx.y, Qn = Lny.x + Ln.y, Fn = (Ln.x | Lnx.y | Lny.x | Ln.y) & FLAG_LANES;
                if (iz >= 0) {
                    const size_t lin = (size_t)(z0 + iz) * NN + gsite;
                    const uint2 Lc = XY[cur * NELEM + e_own], Lcx = XY[cur * NELEM + e_own + 1], Lcy = XY[cur * NELEM + e_own + COLS];
                    const unsigned Z0 = ZW[e_own], Zx = ZW[e_own + 1], Zy = ZW[e_own + COLS], Zxy = ZW[e_own + COLS + 1];
                    // W_yz(x): n_y(x) + n_z(x+y) - n_y(x+z) - n_z(x);   W_zx(x): n_z(x) + n_x(x+z) - n_z(x+x) - n_x(x)
                    unsigned P[5], Q[5];
                    P[0] = Pxy;            Q[0] = Qxy;                 // xy, plane iz (own)
                    P[1] = Lc.y + Zy;      Q[1] = Ln.y + Z0;           // yz (own)
                    P[2] = Z0 + Ln.x;      Q[2] = Zx + Lc.x;           // zx (own)
                    P[3] = Lcx.y + Zxy;    Q[3] = Lnx.y + Zx;          // yz at x + x
                    P[4] = Zy + Lny.x;     Q[4] = Zxy + Lcy.x;         // zx at x + y
                    unsigned Eabs[6], flagged = (Pn | Qn) & FLAG_LANES;
#pragma unroll
                    for (int q = 0; q < 5; q++) {
                        Eabs[q] = __vabsdiffu4(P[q], Q[q]) & VAL_LANES;
                        flagged |= (P[q] | Q[q]) & FLAG_LANES;
                    }
                    Eabs[5] = __vabsdiffu4(Pn, Qn) & VAL_LANES;        // xy, plane iz+1
                    int wsg[2][3];                                      // signed windings of the own plaquettes (EXPORT)
                    unsigned nearbits = 0;                              // bit 3 s + o
                    if (EXPORT) {
#pragma unroll
                        for (int o = 0; o < 3; o++) {
                            wsg[0][o] = (int)(Q[o] & 0xffu) - (int)(P[o] & 0xffu);
                            wsg[1][o] = (int)((Q[o] >> 16) & 0xffu) - (int)((P[o] >> 16) & 0xffu);
                        }
                    }
                    if (flagged) {
                        // slow path: near-cut flags of the own plaquettes; plaquettes with a degenerate link by the
                        // printed formula with chi = 0 on those links
                        auto Af = [&](const char *s, int e) { return *reinterpret_cast<const float4 *>(s + e * 16); };
                        auto th_xy = [&](const char *s, int e, int sec, int dir) {
                            const float4 b = *reinterpret_cast<const float4 *>(s + OFF_B + e * 16);
                            return dir == 0 ? (sec ? b.z : b.x) : (sec ? b.w : b.y);
                        };
                        auto th_z = [&](const char *s, int e, int sec) {
                            const int r = e / COLS, c = e - r * COLS;
                            const float2 cz = *reinterpret_cast<const float2 *>(s + OFF_C + (r * CCOLS + c + 1) * 8);
                            return sec ? cz.y : cz.x;
                        };
                        auto ph = [&](const char *s, int e, int sec) {
                            const float4 a = Af(s, e);
                            return sec ? site_phase(a.z, a.w) : site_phase(a.x, a.y);
                        };
                        // plaquette q (0 xy cur, 1 yz, 2 zx, 3 yz at x+x, 4 zx at x+y, 5 xy nxt) of sector sec by the formula
                        auto formula = [&](int q, int sec) {
                            const int eb = e_own + (q == 3 ? 1 : q == 4 ? COLS : 0);
                            const char *s0 = q == 5 ? sn : sc;
                            float a00, a10, a01, a11, t1, t2, t3, t4;    // corners x, x+i, x+j, x+i+j; links i(x), j(x+i), i(x+j), j(x)
                            if (q == 0 || q == 5) {                       // (i, j) = (x, y)
                                a00 = ph(s0, eb, sec); a10 = ph(s0, eb + 1, sec); a01 = ph(s0, eb + COLS, sec); a11 = ph(s0, eb + COLS + 1, sec);
                                t1 = th_xy(s0, eb, sec, 0); t2 = th_xy(s0, eb + 1, sec, 1); t3 = th_xy(s0, eb + COLS, sec, 0); t4 = th_xy(s0, eb, sec, 1);
                            } else if (q == 1 || q == 3) {                // (y, z)
                                a00 = ph(sc, eb, sec); a10 = ph(sc, eb + COLS, sec); a01 = ph(sn, eb, sec); a11 = ph(sn, eb + COLS, sec);
                                t1 = th_xy(sc, eb, sec, 1); t2 = th_z(sc, eb + COLS, sec); t3 = th_xy(sn, eb, sec, 1); t4 = th_z(sc, eb, sec);
                            } else {                                      // (z, x)
                                a00 = ph(sc, eb, sec); a10 = ph(sn, eb, sec); a01 = ph(sc, eb + 1, sec); a11 = ph(sn, eb + 1, sec);
                                t1 = th_z(sc, eb, sec); t2 = th_xy(sn, eb, sec, 0); t3 = th_z(sc, eb + 1, sec); t4 = th_xy(sc, eb, sec, 0);
                            }
                            const float sum = chi_slow(a00, a10, t1) + chi_slow(a10, a11, t2) - chi_slow(a01, a11, t3) - chi_slow(a00, a01, t4) +
                                              (t1 + t2 - t3 - t4);
                            return __float2int_rn(sum * INV_2PI);
                        };
#pragma unroll
                        for (int q = 0; q < 6; q++) {
                            // OR of the flags of the plaquette's four links (lane 1: p, lane 3: q)
                            unsigned orf;
                            if (q == 0) orf = Fxy;
                            else if (q == 1) orf = Lc.y | Zy | Ln.y | Z0;
                            else if (q == 2) orf = Z0 | Ln.x | Zx | Lc.x;
                            else if (q == 3) orf = Lcx.y | Zxy | Lnx.y | Zx;
                            else if (q == 4) orf = Zy | Lny.x | Zxy | Lcy.x;
                            else orf = Fn;
                            orf &= FLAG_LANES;
                            if (!orf) continue;
#pragma unroll
                            for (int sec = 0; sec < 2; sec++) {
                                const unsigned fs = (orf >> (8 + 16 * sec)) & 5u;     // bit 0 near, bit 2 degenerate
                                if (fs & 4u) {
                                    const int W = formula(q, sec);
                                    Eabs[q] = (Eabs[q] & ~(0xffu << (16 * sec))) | ((unsigned)abs(W) << (16 * sec));
                                    if (EXPORT && q < 3) wsg[sec][q] = W;
                                }
                                if ((fs & 1u) && q < 3) nearbits |= 1u << (3 * sec + q);
                            }
                        }
                    }
                    // own plaquettes: length sums, near-cut counts, largest winding
                    const unsigned own = Eabs[0] + Eabs[1] + Eabs[2];
                    acc.wsum += own;
                    acc.nnear[0] += __popc(nearbits & 7u);
                    acc.nnear[1] += __popc(nearbits & 56u);
                    if ((Eabs[0] | Eabs[1] | Eabs[2]) & 0x00fe00feu) {
#pragma unroll
                        for (int q = 0; q < 3; q++) acc.maxw = max(acc.maxw, (int)max(Eabs[q] & 0xffu, Eabs[q] >> 16));
                    } else if (own) {
                        acc.maxw = max(acc.maxw, 1);
                    }
                    // pierced cells: the six faces of the cell at x
                    const unsigned cell = own + Eabs[3] + Eabs[4] + Eabs[5];
                    const unsigned cp = cell & 0xffu, cq = cell >> 16;
                    cells[lin] = (uint8_t)cp;
                    cells[V + lin] = (uint8_t)cq;
                    acc.ncell[0] += cp > 0;
                    acc.ncell[1] += cq > 0;
                    acc.ncell[2] += (cp > 0) && (cq > 0);
                    if (EXPORT) {
#pragma unroll
                        for (int sec = 0; sec < 2; sec++)
#pragma unroll
                            for (int o = 0; o < 3; o++)
                                codes[(size_t)(3 * sec + o) * V + lin] =
                                    (uint8_t)(((wsg[sec][o] + 8) & 15) | (((nearbits >> (3 * sec + o)) & 1u) << 4));
                    }
                }
                Pxy = Pn;
                Qxy = Qn;
                Fxy = Fn;
            }
        }
        if (!tma) cp_async_wait<0>();
        if (tma) { gpos += (unsigned)(nz + 1); gmom += (unsigned)nz; }
        acc.sumw[0] += (int)(acc.wsum & 0xffffu);
        acc.sumw[1] += (int)(acc.wsum >> 16);
    }

    // ---- per-CTA partials (deterministic two-stage reduction, common.cuh) ----
    double v[FUSED_NRES];
#pragma unroll
    for (int i = 0; i < 6; i++) v[FR_GAUSS + i] = acc.g[i];
    v[FR_SUMW] = acc.sumw[0]; v[FR_SUMW + 1] = acc.sumw[1];
    v[FR_NEAR] = acc.nnear[0]; v[FR_NEAR + 1] = acc.nnear[1];
    v[FR_CELLS] = acc.ncell[0]; v[FR_CELLS + 1] = acc.ncell[1]; v[FR_CELLS + 2] = acc.ncell[2];
#pragma unroll
    for (int i = 0; i < 11; i++) v[FR_DENS + i] = acc.d[i];
    v[FR_GMAX] = acc.gmax[0]; v[FR_GMAX + 1] = acc.gmax[1];
    v[FR_MAXW] = acc.maxw;
    v[FR_MAXTH] = acc.maxth;
    double *red = reinterpret_cast<double *>(smem + OFF_RED);
    const int lane = tid & 31;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < FUSED_NRES; i++) {
        const double r = i < FUSED_NSUM ? warp_sum(v[i]) : warp_max(v[i]);
        if (lane == 0) red[i * (NTHREADS / 32) + warp] = r;
    }
    __syncthreads();
    if (tid < FUSED_NRES) {
        double r = red[tid * (NTHREADS / 32)];
        for (int w = 1; w < NTHREADS / 32; w++) r = tid < FUSED_NSUM ? r + red[tid * (NTHREADS / 32) + w] : fmax(r, red[tid * (NTHREADS / 32) + w]);
        partials[(size_t)blockIdx.x * RED_SLOTS + tid] = r;
    }
}

}  // namespace

int fused_zchunk(int N) { return N >= 32 ? 32 : N; }

cudaError_t launch_diag_fused(const float *pos, const float *mom, size_t V, int N, FusedCoef k, uint8_t *cells, uint8_t *codes,
                              double *partials, int *nblocks, const DiagMaps *maps, int sms, cudaStream_t st)
{
    DiagMaps m;
    if (maps) m = *maps;
    else {
        memset(&m, 0, sizeof m);
        k.flags |= 2;
    }
    const int zc = fused_zchunk(N);
    const int ntx = (N + TX - 1) / TX, nty = (N + TY - 1) / TY, nzc = (N + zc - 1) / zc;
    const long items = (long)ntx * nty * nzc;
    long grid = (long)sms * 2;
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
