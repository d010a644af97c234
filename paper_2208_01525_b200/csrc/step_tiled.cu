// step_tiled.cu -- the production fused kick+drift kernel (Eq. 17-26).
//
// One CTA owns an xy tile of TX x TY sites and marches through a chunk of z planes.  The three position
// packs of each plane (A = phi,psi; B = in-plane links of both sectors; C = z links; tile + one-site halo)
// are staged into a 4-slot shared-memory ring TWO planes ahead of the arithmetic:
//   * tiles that do not touch the lattice boundary: three TMA box loads per plane (cp.async.bulk.tensor,
//     issued by one thread, completion on an mbarrier), plus three TMA boxes for the tile's momenta;
//   * boundary / ragged tiles (periodic wrap cannot be expressed as a TMA box): per-thread cp.async
//     (LDGSTS) with the wrap resolved in a per-thread load plan.
// Only planes z and z+1 live in shared memory: everything a site needs from plane z-1 -- the backward z hop
// conj(U_z(x-z)) f(x-z) and the plaquettes P_yz(x-z), P_zx(x-z) -- was computed by the SAME thread one
// iteration earlier and is carried in registers (the plaquettes bit-identically, see plaq()).
// Every stencil operand is a vector read from shared memory, and each site's 20 words make one HBM round
// trip: positions in through the ring (+ halo, served by L2), momenta in, 3 + 3 vector stores out (new
// positions to the other ping-pong buffer, momenta in place).
#include <cstring>

#include "common.cuh"
#include "kernels.h"
#include "stage.cuh"
#include "step_site.cuh"

namespace u1u1 {

namespace {

constexpr int NSLOT = 4;            // ring: z, z+1 in use, z+2 and z+3 in flight
// momentum ring (TMA tiles only): 2 slots of MA float4[NTHREADS] | MB float4[NTHREADS] | MC float2[NTHREADS]
constexpr int MOFF_B = NTHREADS * 16, MOFF_C = NTHREADS * 32, MSLOT_BYTES = NTHREADS * 40;
constexpr int OFF_MRING = NSLOT * SLOT_BYTES;
constexpr int OFF_BARS = OFF_MRING + 2 * MSLOT_BYTES;           // fullP[4], fullM[2]
constexpr int SMEM_BYTES = OFF_BARS + 64;                       // 76 352 B -> 3 CTAs per SM

// exp(-i theta): libm sincosf (1-2 ulp) or, with FAST, the SFU approximations.  MUFU.SIN/COS take the angle
// in turns and reduce it themselves (one FMUL by 1/(2 pi) + 2 MUFU); error max(5e-7, 6e-8 |theta|) -- 5e-7 at any
// |theta| in the RR instances, which reduce the angle explicitly first (tuning flag 2048, f32x2.cuh).  The
// discrete Gauss law holds for ANY complex U used consistently for a link, so this error never enters it
// (DESIGN.md section 8).
template <bool FAST>
__device__ inline void phasor(float th, float &sn, float &cs)
{
    if (FAST) __sincosf(th, &sn, &cs);
    else sincosf(th, &sn, &cs);
}

// Difference-form phasor: sn = sin(theta) and c1 = 1 - cos(theta) = 2 sin^2(theta/2) from the half angle, so
// that U f' - f = (f' - f) - c1 f' -/+ i sn f' is formed from SMALL terms (no cancellation against f itself).
template <bool FAST>
__device__ inline void phasor_diff(float th, float &sn, float &c1)
{
    float sh, ch;
    phasor<FAST>(0.5f * th, sh, ch);
    const float sh2 = sh + sh;          // exact, so sn and c1 are bit-identical to 2 sh ch and 2 sh sh
    sn = sh2 * ch;
    c1 = sh2 * sh;
}

// P = ((a + b) - c) - d, always in this order: a plaquette evaluated at two different sites from the same
// four links gives the same bits, so the rounding errors of the curl are themselves a lattice curl and
// drop out of the Gauss law ("consistent plaquettes").
__device__ inline float plaq(float a, float b, float c, float d)
{
    return __fsub_rn(__fsub_rn(__fadd_rn(a, b), c), d);
}

__device__ inline float ln4(const float4 &v, int i) { return i == 0 ? v.x : i == 1 ? v.y : i == 2 ? v.z : v.w; }
__device__ inline float ln2(const float2 &v, int i) { return i == 0 ? v.x : v.y; }
__device__ inline void set4(float4 &v, int i, float a) { if (i == 0) v.x = a; else if (i == 1) v.y = a; else if (i == 2) v.z = a; else v.w = a; }
__device__ inline void set2(float2 &v, int i, float a) { if (i == 0) v.x = a; else v.y = a; }

// R = arithmetic type of the kick chain (hops, Laplacian, currents, potential, momentum update):
// double keeps the discrete Gauss identity Im(phi* D-D+ phi) = d-_i Im(phi* D+_i phi) at fp32-STORAGE
// roundoff instead of fp32-ARITHMETIC roundoff (measured ~30x smaller residual).
// DIFF (fp32 chain only): the hops enter as differences d_i = U_i f(x+i) - f(x), d'_i = conj(U_i(x-i)) f(x-i) - f(x),
// evaluated without cancellation; the Laplacian is their plain sum and the current is Im(f* d_i).  Rounding
// errors then scale with |D f| dx instead of |f|, which brings the fp32 chain's Gauss residual close to the
// storage floor wherever the fields are smooth.
// SLAB: the buffers hold a z slab with one halo plane on either side (common.cuh); no periodic wrap in z, and the
// slab's top / bottom output planes are also stored into the neighbouring slabs' halo planes.
// PK (only with FAST, float, DIFF): both sectors at once in packed fp32x2 instructions; bit-identical to the scalar
// difference-form chain (same IEEE operations in the same order), which stays available under tuning flag 1.
template <bool FAST, typename R, bool DIFF, bool SLAB, bool PK, bool RR>
__global__ void __launch_bounds__(NTHREADS, sizeof(R) == 8 ? 2 : 3)
step_tiled_kernel(Lattice L, StepCoef k, int zchunk, int band, const __grid_constant__ StepMaps maps)
{
    extern __shared__ __align__(128) char smem[];
    const unsigned sbase = smem_u32(smem), bars = sbase + OFF_BARS;
    const int N = L.N;
    const size_t V = L.V, NN = (size_t)N * N;
    const int tid = threadIdx.x, tx = tid & (TX - 1), ty = tid / TX;
    // 1-d grid, launch order = (tile x fastest, tile row within a band of `band` rows, z chunk, band): the CTAs that
    // are resident together cover one band of tile rows of one z chunk, and the next wave continues with the NEXT
    // chunk of the same band, whose two boundary planes the previous wave has just read
    const int NZO = SLAB ? L.nz_own : N, ZB = SLAB ? 1 : 0;     // own planes and the buffer index of the first of them
    const int ntx = (N + TX - 1) / TX, nty = (N + TY - 1) / TY, nzc = (NZO + zchunk - 1) / zchunk;
    const int full = ntx * band * nzc, bnd = blockIdx.x / full, rem = blockIdx.x - bnd * full;
    const int rows = min(band, nty - bnd * band), bzc = rem / (ntx * rows), tl = rem - bzc * (ntx * rows);
    const int x0 = (tl % ntx) * TX, y0 = (bnd * band + tl / ntx) * TY, z0 = ZB + bzc * zchunk;
    const int wx = min(TX, N - x0), wy = min(TY, N - y0), nz = min(zchunk, ZB + NZO - z0);
    const bool active = tx < wx && ty < wy;
    // TMA boxes cannot wrap: only tiles whose halo lies inside the lattice take the TMA path (CTA-uniform)
    const bool tma = !(k.flags & 2) && tile_is_interior(x0, y0, N);
    const bool tmom = tma && !(k.flags & 4);        // momenta by TMA boxes (default on TMA tiles), else ld.global.cs
    const char *pos = reinterpret_cast<const char *>(L.pos_in);
    const unsigned long long pol_stream = policy_evict_first();
    const unsigned long long pol_keep = policy_evict_last();

    // ---- staging of relative plane j (z = z0 + j, j = -1 .. nz) into ring slot (j + 1) & 3 ----
    CpPlan plan;                  // cp.async path: this thread's copies of one halo plane
    if (!tma) make_cp_plan(plan, tid, x0, y0, wx, wy, N);
    auto stage_cp = [&](int j) {          // every thread; caller commits the group
        stage_plane_cp(plan, tid, pos, V, (size_t)(SLAB ? z0 + j : wrapi(z0 + j, N)) * NN, sbase + ((j + 1) & 3) * SLOT_BYTES);
    };
    auto stage_tma = [&](int j) {         // one thread
        // evict-last: the neighbouring tiles re-read these lines as halo within a few planes (measured: -1 % DRAM reads)
        stage_plane_tma(maps.pos, x0, y0, SLAB ? z0 + j : wrapi(z0 + j, N), sbase + ((j + 1) & 3) * SLOT_BYTES,
                        bars + 8 * ((j + 1) & 3), pol_keep);
    };
    auto stage_mom_tma = [&](int m) {     // one thread; momenta of relative plane m into ring slot m & 1
        const unsigned slot = sbase + OFF_MRING + (m & 1) * MSLOT_BYTES, bar = bars + 8 * (4 + (m & 1));
        mbar_expect_tx(bar, MSLOT_BYTES);
        tma_load_3d_hint(slot, &maps.mom.A, 4 * x0, y0, z0 + m, bar, pol_stream);
        tma_load_3d_hint(slot + MOFF_B, &maps.mom.B, 4 * x0, y0, z0 + m, bar, pol_stream);
        tma_load_3d_hint(slot + MOFF_C, &maps.mom.C, 2 * x0, y0, z0 + m, bar, pol_stream);
    };

    // ---- prologue: planes -1 .. 2 in flight, wait for -1 and 0 ----
    if (tma) {
        if (tid == 0) {
#pragma unroll
            for (int b = 0; b < 6; b++) mbar_init(bars + 8 * b, 1);
            mbar_fence_init();
        }
        __syncthreads();
        if (tid == 0) {
            for (int j = -1; j <= 2; j++)
                if (j <= nz) stage_tma(j);
            if (tmom) stage_mom_tma(0);
        }
        mbar_wait(bars + 0, 0);
        mbar_wait(bars + 8, 0);
    } else {
        for (int j = -1; j <= 2; j++) {
            if (j <= nz) stage_cp(j);
            cp_async_commit();
        }
        cp_async_wait<2>();
        __syncthreads();
    }

    const int e_own = (ty + 1) * COLS + tx + 1;     // this thread's site inside a staged plane
    const size_t gsite = (size_t)(y0 + ty) * N + (size_t)(x0 + tx);
    const R aS = k.aS, bS = k.bS, aG = k.aG, bG = k.bG, inv_dx2 = k.inv_dx2, inv_dx3 = k.inv_dx3;
    constexpr int XP = 1, XM = -1, YP = COLS, YM = -COLS;
    auto A = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + (e_own + d) * 16); };
    auto B = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + OFF_B + (e_own + d) * 16); };
    const int e_ownC = (ty + 1) * CCOLS + tx + 2;
    auto C = [&](const char *s, int d) { return *reinterpret_cast<const float2 *>(s + OFF_C + (e_ownC + d) * 8); };
    constexpr int CYP = CCOLS, CYM = -CCOLS;

    // ---- carried from plane z-1: backward z hop and the two plaquettes that contain theta_z(x - z) ----
    R bzr[2] = {0, 0}, bzi[2] = {0, 0};
    float Pyz_c[2] = {0.f, 0.f}, Pzx_c[2] = {0.f, 0.f};
    PkCarry cy = {bc(0.f), bc(0.f), bc(0.f), bc(0.f), make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)};                              // the same, packed (PK)
    if (PK && active) {
        const char *sc = smem, *sp = smem + SLOT_BYTES;          // planes -1 and 0
        auto pA = [&](int p, int dx, int dy) { return A(p ? sp : sc, dy * COLS + dx); };
        auto pB = [&](int p, int dx, int dy) { return B(p ? sp : sc, dy * COLS + dx); };
        auto pC = [&](int p, int dx, int dy) { return C(p ? sp : sc, dy * CCOLS + dx); };
        pk_carry_init<RR>(cy, pA, pB, pC);
    }
    if (!PK && active) {
        const char *sc = smem, *sp = smem + SLOT_BYTES;          // planes -1 and 0
        const float4 Ac = A(sc, 0), Bc = B(sc, 0), Bzp = B(sp, 0);
        const float2 Cc = C(sc, 0), Cxp = C(sc, XP), Cyp = C(sc, CYP);
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int a0 = s, a1 = s + 2;
            const float thz = ln2(Cc, s);
            if (DIFF) {
                const float4 Azp = A(sp, 0);
                const float fr = ln4(Ac, a0), fi = ln4(Ac, a1);
                float sn, c1;
                phasor_diff<FAST>(thz, sn, c1);
                bzr[s] = fmaf(-sn, fi, fmaf(-c1, fr, fr - ln4(Azp, a0)));
                bzi[s] = fmaf(sn, fr, fmaf(-c1, fi, fi - ln4(Azp, a1)));
            } else {
                float snf, csf;
                phasor<FAST>(thz, snf, csf);
                const R sn = snf, cs = csf, fr = ln4(Ac, a0), fi = ln4(Ac, a1);
                bzr[s] = cs * fr - sn * fi;
                bzi[s] = cs * fi + sn * fr;
            }
            Pyz_c[s] = plaq(ln4(Bc, a1), ln2(Cyp, s), ln4(Bzp, a1), thz);
            Pzx_c[s] = plaq(thz, ln4(Bzp, a0), ln2(Cxp, s), ln4(Bc, a0));
        }
    }

    for (int iz = 0; iz < nz; iz++) {
        // plane iz+1 must have landed; the slot of plane iz-1 (read by every thread in the previous
        // iteration) is recycled for plane iz+3, so its refill is issued after the barrier
        if (tma) {
            __syncthreads();
            if (tid == 0) {
                if (iz + 3 <= nz) stage_tma(iz + 3);
                if (tmom && iz + 1 < nz) stage_mom_tma(iz + 1);
            }
            mbar_wait(bars + 8 * ((iz + 2) & 3), ((iz + 2) >> 2) & 1);
            if (tmom) mbar_wait(bars + 8 * (4 + (iz & 1)), (iz >> 1) & 1);
        } else {
            cp_async_wait<1>();
            __syncthreads();
            if (iz + 3 <= nz) stage_cp(iz + 3);
            cp_async_commit();
        }
        if (!active) continue;

        const char *sc = smem + ((iz + 1) & 3) * SLOT_BYTES;   // plane z
        const char *sp = smem + ((iz + 2) & 3) * SLOT_BYTES;   // plane z+1
        const size_t lin = (size_t)(z0 + iz) * NN + gsite;

        float4 MA, MB;
        float2 MC;
        if (tmom) {
            const char *ms = smem + OFF_MRING + (iz & 1) * MSLOT_BYTES;
            MA = *reinterpret_cast<const float4 *>(ms + tid * 16);
            MB = *reinterpret_cast<const float4 *>(ms + MOFF_B + tid * 16);
            MC = *reinterpret_cast<const float2 *>(ms + MOFF_C + tid * 8);
        } else {
            MA = __ldcs(reinterpret_cast<const float4 *>(L.mom) + lin);
            MB = __ldcs(reinterpret_cast<const float4 *>(L.mom + 4 * V) + lin);
            MC = __ldcs(reinterpret_cast<const float2 *>(L.mom + 8 * V) + lin);
        }

        const float4 Ac = A(sc, 0), Axp = A(sc, XP), Axm = A(sc, XM), Ayp = A(sc, YP), Aym = A(sc, YM);
        const float4 Azp = A(sp, 0);
        const float4 Bc = B(sc, 0), Bxp = B(sc, XP), Bxm = B(sc, XM), Byp = B(sc, YP), Bym = B(sc, YM);
        const float4 Bxmyp = B(sc, XM + YP), Bxpym = B(sc, XP + YM);
        const float4 Bzp = B(sp, 0), Bxmzp = B(sp, XM), Bymzp = B(sp, YM);
        const float2 Cc = C(sc, 0), Cxp = C(sc, XP), Cxm = C(sc, XM), Cyp = C(sc, CYP), Cym = C(sc, CYM);

        float4 OA, OB;
        float2 OC;

        if constexpr (PK) {
            // both sectors at once in packed fp32x2 instructions (step_site.cuh)
            auto pA = [&](int p, int dx, int dy) { return A(p ? sp : sc, dy * COLS + dx); };
            auto pB = [&](int p, int dx, int dy) { return B(p ? sp : sc, dy * COLS + dx); };
            auto pC = [&](int p, int dx, int dy) { return C(p ? sp : sc, dy * CCOLS + dx); };
            pk_site_update<RR>(cy, pA, pB, pC, k, MA, MB, MC, OA, OB, OC);
        }

        const R m2p = (R)Ac.x * (R)Ac.x + (R)Ac.z * (R)Ac.z;
        const R m2q = (R)Ac.y * (R)Ac.y + (R)Ac.w * (R)Ac.w;
#pragma unroll
        for (int s = 0; s < (PK ? 0 : 2); s++) {
            const int a0 = s, a1 = s + 2;                       // lanes of this sector in packs A and B
            const R fr = ln4(Ac, a0), fi = ln4(Ac, a1);
            // ---- covariant Laplacian and currents (Eq. 17-18; current of Eq. 20-21) ----
            const float thc[3] = {ln4(Bc, a0), ln4(Bc, a1), ln2(Cc, s)};
            const float thm[2] = {ln4(Bxm, a0), ln4(Bym, a1)};                      // theta_i(x - i), i = x, y
            const float fpr[3] = {ln4(Axp, a0), ln4(Ayp, a0), ln4(Azp, a0)};       // f(x + i)
            const float fpi[3] = {ln4(Axp, a1), ln4(Ayp, a1), ln4(Azp, a1)};
            const float fmr[2] = {ln4(Axm, a0), ln4(Aym, a0)};                      // f(x - i), i = x, y
            const float fmi[2] = {ln4(Axm, a1), ln4(Aym, a1)};
            R lap_re = bzr[s], lap_im = bzi[s], J[3];
            if (!DIFF) {
                lap_re += (R)-6 * fr;
                lap_im += (R)-6 * fi;
            }
#pragma unroll
            for (int i = 0; i < 3; i++) {
                if (DIFF) {
                    const float f_r = ln4(Ac, a0), f_i = ln4(Ac, a1);
                    float sn, c1;
                    phasor_diff<FAST>(thc[i], sn, c1);
                    const float dr = fmaf(sn, fpi[i], fmaf(-c1, fpr[i], fpr[i] - f_r));
                    const float di = fmaf(-sn, fpr[i], fmaf(-c1, fpi[i], fpi[i] - f_i));
                    lap_re += dr;
                    lap_im += di;
                    J[i] = f_r * di - f_i * dr;
                    if (i == 2) {              // backward z difference of the NEXT plane: conj(U_z(x)) f(x) - f(x+z)
                        bzr[s] = fmaf(-sn, f_i, fmaf(-c1, f_r, f_r - fpr[2]));
                        bzi[s] = fmaf(sn, f_r, fmaf(-c1, f_i, f_i - fpi[2]));
                    } else {
                        phasor_diff<FAST>(thm[i], sn, c1);
                        lap_re += fmaf(-sn, fmi[i], fmaf(-c1, fmr[i], fmr[i] - f_r));
                        lap_im += fmaf(sn, fmr[i], fmaf(-c1, fmi[i], fmi[i] - f_i));
                    }
                    continue;
                }
                float snf, csf;
                phasor<FAST>(thc[i], snf, csf);
                R sn = snf, cs = csf;
                const R hr = cs * (R)fpr[i] + sn * (R)fpi[i], hi = cs * (R)fpi[i] - sn * (R)fpr[i];
                lap_re += hr;
                lap_im += hi;
                J[i] = fr * hi - fi * hr;
                if (i == 2) {                  // backward z hop of the NEXT plane: conj(U_z(x)) f(x)
                    bzr[s] = cs * fr - sn * fi;
                    bzi[s] = cs * fi + sn * fr;
                } else {
                    phasor<FAST>(thm[i], snf, csf);
                    sn = snf; cs = csf;
                    lap_re += cs * (R)fmr[i] - sn * (R)fmi[i];
                    lap_im += cs * (R)fmi[i] + sn * (R)fmr[i];
                }
            }
            const R sig = s ? k.sig2sq : k.sig1sq, sigo = s ? k.sig1sq : k.sig2sq;
            const R m2 = s ? m2q : m2p, m2o = s ? m2p : m2q;
            const R bracket = (R)(s ? k.lamh2 : k.lamh1) * (m2 - sig) - (R)k.kap * (m2o - sigo);
            float pr, pi;
            if (DIFF) {                 // small increment first, then ONE rounding at the size of the momentum
                const float m0 = ln4(MA, a0), m1 = ln4(MA, a1);
                pr = m0 + fmaf(k.aSm1, m0, k.bS * (float)(lap_re * inv_dx2 - fr * bracket));
                pi = m1 + fmaf(k.aSm1, m1, k.bS * (float)(lap_im * inv_dx2 - fi * bracket));
            } else {
                pr = (float)(aS * (R)ln4(MA, a0) + bS * (lap_re * inv_dx2 - fr * bracket));
                pi = (float)(aS * (R)ln4(MA, a1) + bS * (lap_im * inv_dx2 - fi * bracket));
            }
            set4(MA, a0, pr);
            set4(MA, a1, pi);
            set4(OA, a0, fmaf(k.dtau, pr, ln4(Ac, a0)));
            set4(OA, a1, fmaf(k.dtau, pi, ln4(Ac, a1)));

            // ---- lattice curl of the plaquettes, sum_{j != i} [P_ij(x) - P_ij(x-j)] (Eq. 20-21) ----
            const float Pxy = plaq(thc[0], ln4(Bxp, a1), ln4(Byp, a0), thc[1]);
            const float Pxy_my = plaq(ln4(Bym, a0), ln4(Bxpym, a1), thc[0], thm[1]);
            const float Pxy_mx = plaq(thm[0], thc[1], ln4(Bxmyp, a0), ln4(Bxm, a1));
            const float Pyz = plaq(thc[1], ln2(Cyp, s), ln4(Bzp, a1), thc[2]);
            const float Pyz_mz = Pyz_c[s];
            const float Pyz_my = plaq(thm[1], thc[2], ln4(Bymzp, a1), ln2(Cym, s));
            const float Pzx = plaq(thc[2], ln4(Bzp, a0), ln2(Cxp, s), thc[0]);
            const float Pzx_mx = plaq(ln2(Cxm, s), ln4(Bxmzp, a0), thc[2], thm[0]);
            const float Pzx_mz = Pzx_c[s];
            Pyz_c[s] = Pyz;
            Pzx_c[s] = Pzx;
            const float cc[3] = {(Pxy - Pxy_my) - (Pzx - Pzx_mz), (Pyz - Pyz_mz) - (Pxy - Pxy_mx),
                                 (Pzx - Pzx_mx) - (Pyz - Pyz_my)};
            const R cur = s ? k.cur2 : k.cur1;
            float e0, e1, e2;
            if (DIFF) {
                const float g0 = ln4(MB, a0), g1 = ln4(MB, a1), g2 = ln2(MC, s);
                e0 = g0 + fmaf(k.aGm1, g0, k.bG * (float)(cur * J[0] - (R)cc[0] * inv_dx3));
                e1 = g1 + fmaf(k.aGm1, g1, k.bG * (float)(cur * J[1] - (R)cc[1] * inv_dx3));
                e2 = g2 + fmaf(k.aGm1, g2, k.bG * (float)(cur * J[2] - (R)cc[2] * inv_dx3));
            } else {
                e0 = (float)(aG * (R)ln4(MB, a0) + bG * (cur * J[0] - (R)cc[0] * inv_dx3));
                e1 = (float)(aG * (R)ln4(MB, a1) + bG * (cur * J[1] - (R)cc[1] * inv_dx3));
                e2 = (float)(aG * (R)ln2(MC, s) + bG * (cur * J[2] - (R)cc[2] * inv_dx3));
            }
            set4(MB, a0, e0);
            set4(MB, a1, e1);
            set2(MC, s, e2);
            set4(OB, a0, fmaf(k.dtau_dx, e0, thc[0]));
            set4(OB, a1, fmaf(k.dtau_dx, e1, thc[1]));
            set2(OC, s, fmaf(k.dtau_dx, e2, thc[2]));
        }
        __stcs(reinterpret_cast<float4 *>(L.mom) + lin, MA);
        __stcs(reinterpret_cast<float4 *>(L.mom + 4 * V) + lin, MB);
        __stcs(reinterpret_cast<float2 *>(L.mom + 8 * V) + lin, MC);
        __stcs(reinterpret_cast<float4 *>(L.pos_out) + lin, OA);
        __stcs(reinterpret_cast<float4 *>(L.pos_out + 4 * V) + lin, OB);
        __stcs(reinterpret_cast<float2 *>(L.pos_out + 8 * V) + lin, OC);
        if (SLAB) {                     // the exchange: boundary planes go straight into the neighbours' halo planes
            if (z0 + iz == L.nz_own) {
                const size_t pl = gsite, PV = L.peer_up_V;          // plane 0 of the slab above
                reinterpret_cast<float4 *>(L.peer_up_out)[pl] = OA;
                reinterpret_cast<float4 *>(L.peer_up_out + 4 * PV)[pl] = OB;
                reinterpret_cast<float2 *>(L.peer_up_out + 8 * PV)[pl] = OC;
            }
            if (z0 + iz == 1) {
                const size_t pl = L.peer_dn_plane * NN + gsite, PV = L.peer_dn_V;
                reinterpret_cast<float4 *>(L.peer_dn_out)[pl] = OA;
                reinterpret_cast<float4 *>(L.peer_dn_out + 4 * PV)[pl] = OB;
                reinterpret_cast<float2 *>(L.peer_dn_out + 8 * PV)[pl] = OC;
            }
        }
    }
    if (!tma) cp_async_wait<0>();
}

int pick_zchunk(int N, int sms)
{
    // enough CTAs to fill the SMs x 3 several times over, chunks long enough to amortise the 2-plane prologue --
    // but no longer: neighbouring CTAs drift apart while they march, and a halo line that the neighbour fetched too
    // long ago has left L2.  With the band launch order below the two boundary planes of a chunk are re-read by the
    // very next wave, so short chunks cost little (measured at 1024^3, band order: 8 planes 29.65 ms, 12: 29.2,
    // 16: 29.05, 24: 29.25, 32: 29.45; plain 3-d grid order: 32: 29.8, 64: 30.6, 128: 32.3, 512: 34.6)
    const int tiles = ((N + TX - 1) / TX) * ((N + TY - 1) / TY);
    int zc = 16;
    while (zc > 8 && (long)tiles * ((N + zc - 1) / zc) < (long)sms * 3 * 4) zc >>= 1;
    return zc < N ? zc : N;
}

template <bool FAST, typename R, bool DIFF, bool SLAB = false, bool PK = false, bool RR = false>
cudaError_t launch_one(const Lattice &L, StepCoef k, cudaStream_t st, const StepMaps *m, int sms)
{
    // per device and cheap: set on every launch rather than caching a per-process flag
    cudaError_t ea = cudaFuncSetAttribute(step_tiled_kernel<FAST, R, DIFF, SLAB, PK, RR>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (ea != cudaSuccess) return ea;
    StepMaps maps;
    if (!m) {
        memset(&maps, 0, sizeof maps);
        k.flags |= 2;                       // no tile can lie strictly inside such a lattice: cp.async path only
    } else {
        maps = *m;
    }
    const int zc = pick_zchunk(L.N, sms);
    const int nzo = SLAB ? L.nz_own : L.N;
    const int ntx = (L.N + TX - 1) / TX, nty = (L.N + TY - 1) / TY, nzc = (nzo + zc - 1) / zc;
    // band height = the tile rows one wave of resident CTAs covers (SMs x CTAs per SM / tiles per row)
    const int per_sm = sizeof(R) == 8 ? 2 : 3;
    int band = (k.flags & 8) ? nty : (sms * per_sm + ntx - 1) / ntx;     // tuning flag 8: the order of a plain 3-d grid
    if (band > nty) band = nty;
    const unsigned grid = (unsigned)ntx * nty * nzc;
    step_tiled_kernel<FAST, R, DIFF, SLAB, PK, RR><<<grid, NTHREADS, SMEM_BYTES, st>>>(L, k, zc, band, maps);
    return cudaGetLastError();
}

}  // namespace

bool step_tiled_supports(int N) { return N >= 8 && (N % 4) == 0; }

// mode bit 0: SFU sin/cos; bit 1: fp32 kick chain (default is the fp64 chain); 4 / 5: fp32 chain in difference form
// maps: tensor maps of (L.pos_in, L.mom), or NULL for lattices too small for any interior tile; sms = SM count
cudaError_t launch_step_tiled(const Lattice &L, const StepCoef &k, cudaStream_t st, int mode, const StepMaps *maps, int sms)
{
    if (L.nz_own) return mode == 5 ? launch_one<true, float, true, true, true>(L, k, st, maps, sms) : cudaErrorNotSupported;
    switch (mode) {
        case 0: return launch_one<false, double, false>(L, k, st, maps, sms);
        case 1: return launch_one<true, double, false>(L, k, st, maps, sms);
        case 2: return launch_one<false, float, false>(L, k, st, maps, sms);
        case 3: return launch_one<true, float, false>(L, k, st, maps, sms);
        case 4: return launch_one<false, float, true>(L, k, st, maps, sms);
        default:            // the production instance: packed fp32x2 chain (tuning flag 1: the same chain in scalar instructions)
            // (tuning flag 2048: the packed chain with explicit range reduction of the link phases)
            return (k.flags & 1) ? launch_one<true, float, true>(L, k, st, maps, sms)
                 : (k.flags & 2048) ? launch_one<true, float, true, false, true, true>(L, k, st, maps, sms)
                                    : launch_one<true, float, true, false, true>(L, k, st, maps, sms);
    }
}

bool step_tiled_uses_tma(int N) { return N >= COLS + 2; }

}  // namespace u1u1
