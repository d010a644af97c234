// step_tb.cu -- TWO fused kick+drift steps per pass over the lattice (temporal blocking; Eq. 17-26).
//
// The one-step kernel (step_tiled.cu) moves every site's 20 words through HBM once per step: 160 B per site-update,
// which is where it saturates.  Here a CTA advances its 32 x 16 tile (TX x TBY, stage.cuh) by two
// steps before anything goes back to HBM -- 80 B per site-update:
//   step 1 is evaluated on the tile AND its one-site halo (34 x 18 sites, from positions staged with a TWO-site halo);
//   its new positions go to a shared-memory ring, never to HBM;
//   step 2 is the one-step kernel's body, reading that ring instead of staged HBM planes.
// Both steps march through the z planes of a chunk together, step 1 one plane ahead of step 2; everything a site needs
// from the plane below is carried in registers as in the one-step kernel.  A CTA has 16 "inner" warps (one tile site per
// thread: step 1 and step 2) and 4 "halo" warps (the 100 sites around the tile: step 1 only), so every thread owns
// exactly one step-1 site.  The arithmetic per site is pk_site_update() of step_site.cuh for both steps: the result is
// bit-identical to two launches of the one-step kernel.
// Momenta of halo sites belong to neighbouring tiles, which update them in this same launch: the kernel reads momenta
// from one buffer and writes them to ANOTHER (the caller's aux buffer, u1u1_set_aux).  Redundant work: step 1 runs on
// 612 / 512 of the sites and on two extra planes per chunk of 128.
// Shared memory (201 152 B, one CTA of 640 threads per SM, 96 registers): 3 position slots (the two planes step 1 reads
// + one in flight), 2 momentum slots (tile only; the halo threads prefetch their site's momenta into registers), 3 slots
// of step-1 positions (the two planes step 2 reads + the one step 1 writes, so one __syncthreads per plane suffices).
// (TB_TY = 8 builds the first version of the round: 32 x 8 tiles, 352 threads, 2 CTAs per SM at 80 registers; 5 % slower.)
#include <cstring>
#include <type_traits>

#include "common.cuh"
#include "kernels.h"
#include "stage.cuh"
#include "step_site.cuh"

namespace u1u1 {

namespace {

// step 1 carries the site's own packs A and B from plane to plane in registers (step_site.cuh, OWN): at 96 registers that
// fits without spills and saves two 128-bit shared-memory reads per step-1 site; in step 2 as well it would spill
constexpr bool OWN1 = TBY == 16, OWN2 = false;
constexpr int NIN = TX * TBY;                   // inner threads (512)
constexpr int NHALO = 2 * COLS + 2 * TBY;       // halo sites (100)
constexpr int TB_THREADS = NIN + 32 * ((NHALO + 31) / 32);        // + halo warps (4): 640
constexpr int TB_CTAS = TBY == 8 ? 2 : 1;       // CTAs per SM
// a slot of step-1 positions: A float4[TBY + 2][COLS], then the x, y and z links as three float2[TBY + 2][COLS] arrays of
// (p, q) pairs.  Splitting pack B makes the stencil reads that need only the x or only the y links (6 of step 2's 21)
// contiguous 64-bit reads: two shared-memory wavefronts per warp instead of the four a 64-bit read at a 16-byte pitch
// takes (two-way bank conflict per half-warp) -- the layout of THIS ring is free, the staged HBM planes' is not.
constexpr int I_OFF_X = (TBY + 2) * COLS * 16, I_OFF_Y = I_OFF_X + (TBY + 2) * COLS * 8, I_OFF_C = I_OFF_Y + (TBY + 2) * COLS * 8;
constexpr int I_SLOT = ((I_OFF_C + (TBY + 2) * COLS * 8 + 127) / 128) * 128;
constexpr int NP = 3;                           // position ring
constexpr int MOFF_B = NIN * 16, MOFF_C = NIN * 32, MSLOT_BYTES = NIN * 40;      // momentum slot: MA | MB | MC of the tile
constexpr int OFF_M = NP * P2_SLOT_BYTES;
constexpr int OFF_I = OFF_M + 2 * MSLOT_BYTES;  // ring of step-1 positions (one-site halo, slot layout of stage.cuh): 3 slots
constexpr int OFF_BARS = OFF_I + 3 * I_SLOT;
constexpr int SMEM_BYTES = OFF_BARS + 64;       // 201 152 B (TBY = 16), one CTA per SM
constexpr int NCP_P = (3 * P2_ELEM + TB_THREADS - 1) / TB_THREADS;      // cp.async copies per thread and position plane (4)
static_assert(OFF_M % 128 == 0 && OFF_I % 128 == 0 && OFF_BARS % 8 == 0, "alignment");
static_assert(TB_CTAS * (SMEM_BYTES + 1024) <= 233472, "CTAs per SM");

// TMA: the tile's two-site halo lies inside the lattice, positions and momenta arrive by TMA boxes; otherwise
// (boundary / ragged tiles) by per-thread cp.async with the periodic wrap resolved in a per-thread plan.
template <bool TMA, bool RR>
__device__ __forceinline__ void tb_tile(const TbLattice &L, const StepCoef &k1, const StepCoef &k2, const TbMaps &maps, char *smem,
                                        int x0, int y0, int z0, int wx, int wy, int nz)
{
    const unsigned sbase = smem_u32(smem), bars = sbase + OFF_BARS;
    const int N = L.N;
    const size_t V = L.V, NN = (size_t)N * N;
    const int tid = threadIdx.x;

    // ---- this thread's step-1 site (c1, r1) relative to the tile origin; inner threads also own it in step 2 ----
    const bool inner = tid < NIN;
    int c1, r1;
    bool act;
    if (inner) {
        c1 = tid & (TX - 1);
        r1 = tid / TX;
        act = TMA || (c1 < wx && r1 < wy);
    } else {
        const int h = tid - NIN;
        if (h < COLS) { c1 = h - 1; r1 = -1; act = c1 <= wx; }
        else if (h < 2 * COLS) { c1 = h - COLS - 1; r1 = wy; act = c1 <= wx; }
        else if (h < 2 * COLS + TBY) { c1 = -1; r1 = h - 2 * COLS; act = r1 < wy; }
        else { c1 = wx; r1 = h - 2 * COLS - TBY; act = h < NHALO && r1 < wy; }
    }
    const int eP = (r1 + 2) * P2_COLS + c1 + 2;                        // element index in a position slot (two-site halo)
    const int eI = (r1 + 1) * COLS + c1 + 1;                           // in a slot of step-1 positions (one-site halo)
    // in-plane site index: the own site of an inner thread (output), the periodic image of a halo thread's site (momenta)
    const size_t gsite = (size_t)wrapi(y0 + r1, N) * N + (size_t)wrapi(x0 + c1, N);

    // ---- staging ----
    // running plane counters: position plane pp = 0 .. nz+3 is relative plane pp - 2, momentum plane mm = 0 .. nz+1 is
    // relative plane mm - 1; ring slot = pp % 3 resp. mm & 1
    const char *posb = reinterpret_cast<const char *>(L.pos_in), *momb = reinterpret_cast<const char *>(L.mom_in);
    // evict-last on both the position and the momentum boxes: the neighbouring tiles re-read the position halo and the
    // halo threads re-read the momentum lines; evict-first on the momenta was measured and made no difference
    const unsigned long long pol_keep = policy_evict_last();
    int planP[NCP_P];                         // cp.async path: in-plane site of each of this thread's copies (-1: none)
    if (!TMA) {
#pragma unroll
        for (int q = 0; q < NCP_P; q++) {
            const int item = tid + q * TB_THREADS, pack = item / P2_ELEM, e = item - pack * P2_ELEM, r = e / P2_COLS, c = e - r * P2_COLS;
            planP[q] = (pack < 3 && r <= wy + 3 && c <= wx + 3) ? wrapi(y0 - 2 + r, N) * N + wrapi(x0 - 2 + c, N) : -1;
        }
    }
    auto stage_P = [&](int pp, unsigned slot) {       // TMA: one thread; cp.async: every thread (caller commits)
        const int z = wrapi(z0 + pp - 2, N);
        const unsigned dst = sbase + slot * P2_SLOT_BYTES;
        if (TMA) {
            const unsigned bar = bars + 8 * slot;
            mbar_expect_tx(bar, P2_SLOT_BYTES);
            tma_load_3d_hint(dst, &maps.pos.A, 4 * (x0 - 2), y0 - 2, z, bar, pol_keep);
            tma_load_3d_hint(dst + P2_OFF_B, &maps.pos.B, 4 * (x0 - 2), y0 - 2, z, bar, pol_keep);
            tma_load_3d_hint(dst + P2_OFF_C, &maps.pos.C, 2 * (x0 - 2), y0 - 2, z, bar, pol_keep);
        } else {
#pragma unroll
            for (int q = 0; q < NCP_P; q++) {
                if (planP[q] < 0) continue;
                const int item = tid + q * TB_THREADS, pack = item / P2_ELEM, e = item - pack * P2_ELEM;
                const size_t site = (size_t)z * NN + (size_t)planP[q];
                if (pack == 0) cp_async16(dst + e * 16, posb + site * 16);
                else if (pack == 1) cp_async16(dst + P2_OFF_B + e * 16, posb + 16 * V + site * 16);
                else cp_async8(dst + P2_OFF_C + e * 8, posb + 32 * V + site * 8);
            }
        }
    };
    auto stage_M = [&](int mm) {                      // the tile's momenta of relative plane mm - 1
        const int z = wrapi(z0 + mm - 1, N);
        const unsigned dst = sbase + OFF_M + (mm & 1) * MSLOT_BYTES;
        if (TMA) {
            const unsigned bar = bars + 8 * (NP + (mm & 1));
            mbar_expect_tx(bar, MSLOT_BYTES);
            tma_load_3d_hint(dst, &maps.mom.A, 4 * x0, y0, z, bar, pol_keep);
            tma_load_3d_hint(dst + MOFF_B, &maps.mom.B, 4 * x0, y0, z, bar, pol_keep);
            tma_load_3d_hint(dst + MOFF_C, &maps.mom.C, 2 * x0, y0, z, bar, pol_keep);
        } else if (inner && act) {
            const size_t site = (size_t)z * NN + gsite;
            cp_async16(dst + tid * 16, momb + site * 16);
            cp_async16(dst + MOFF_B + tid * 16, momb + 16 * V + site * 16);
            cp_async8(dst + MOFF_C + tid * 8, momb + 32 * V + site * 8);
        }
    };
    const bool issuer = !TMA || tid == 0;
    // halo threads: the momenta of their site in relative plane mm - 1, straight into registers one plane ahead
    float4 MAo = make_float4(0.f, 0.f, 0.f, 0.f), MBo = MAo;        // inner threads: step-1 momenta of the plane step 2 works on next
    float2 MCo = make_float2(0.f, 0.f);
    auto prefetch_M = [&](int mm) {
        const size_t lin = (size_t)wrapi(z0 + mm - 1, N) * NN + gsite;
        MAo = __ldg(reinterpret_cast<const float4 *>(L.mom_in) + lin);
        MBo = __ldg(reinterpret_cast<const float4 *>(L.mom_in + 4 * V) + lin);
        MCo = __ldg(reinterpret_cast<const float2 *>(L.mom_in + 8 * V) + lin);
    };

    // accessors of pk_site_update (A / B / C of the site displaced by (dx, dy) in plane p = 0 or 1): step 1 reads two
    // position slots (two-site halo, pitch P2_COLS), step 2 two slots of step-1 positions (one-site halo, stage.cuh layout)
#define TB_ACC1(P0, P1)                                                                                                      \
    auto fA = [&](int p, int dx, int dy) { return *reinterpret_cast<const float4 *>((p ? (P1) : (P0)) + (eP + dy * P2_COLS + dx) * 16); };            \
    auto fB = [&](int p, int dx, int dy) { return *reinterpret_cast<const float4 *>((p ? (P1) : (P0)) + P2_OFF_B + (eP + dy * P2_COLS + dx) * 16); }; \
    auto fC = [&](int p, int dx, int dy) { return *reinterpret_cast<const float2 *>((p ? (P1) : (P0)) + P2_OFF_C + (eP + dy * P2_COLS + dx) * 8); }
#define TB_ACC2(P0, P1)                                                                                                      \
    auto fA = [&](int p, int dx, int dy) { return *reinterpret_cast<const float4 *>((p ? (P1) : (P0)) + (eI + dy * COLS + dx) * 16); };         \
    auto fB = [&](int p, int dx, int dy) {                                                                                      \
        const float2 bx = *reinterpret_cast<const float2 *>((p ? (P1) : (P0)) + I_OFF_X + (eI + dy * COLS + dx) * 8);          \
        const float2 by = *reinterpret_cast<const float2 *>((p ? (P1) : (P0)) + I_OFF_Y + (eI + dy * COLS + dx) * 8);          \
        return make_float4(bx.x, bx.y, by.x, by.y);         /* the half a caller does not use is never loaded */            \
    };                                                                                                                          \
    auto fC = [&](int p, int dx, int dy) { return *reinterpret_cast<const float2 *>((p ? (P1) : (P0)) + I_OFF_C + (eI + dy * COLS + dx) * 8); }

    // ---- prologue: position planes 0, 1, 2 and momentum planes 0, 1 in flight; step-1 carry from planes 0, 1 ----
    if (TMA) {
        if (tid == 0) {
#pragma unroll
            for (int b = 0; b < NP + 2; b++) mbar_init(bars + 8 * b, 1);
            mbar_fence_init();
        }
        __syncthreads();
    }
    if (issuer) {
        stage_P(0, 0);
        stage_P(1, 1);
        stage_P(2, 2);
        stage_M(0);
        stage_M(1);
    }
    if (!inner && act) prefetch_M(0);
    if (TMA) {
        mbar_wait(bars + 0, 0);
        mbar_wait(bars + 8, 0);
    } else {
        cp_async_commit();
        cp_async_wait<0>();
        __syncthreads();
    }
    PkCarry cy1 = {bc(0.f), bc(0.f), bc(0.f), bc(0.f), make_float4(0.f, 0.f, 0.f, 0.f), make_float4(0.f, 0.f, 0.f, 0.f)}, cy2 = cy1;
    if (act) {
        const char *p0 = smem, *p1 = smem + P2_SLOT_BYTES;
        TB_ACC1(p0, p1);
        pk_carry_init<RR, OWN1>(cy1, fA, fB, fC);
    }
    __syncthreads();                          // everybody is done with position plane 0: its slot takes plane 3
    if (issuer) stage_P(3, 0);
    if (!TMA) cp_async_commit();

    unsigned sP = 1;                          // ring slot of position plane t + 1
    // slots of the step-1 planes t, t-1, t-2 as explicit pointers rotated at the end of every iteration (computing them from
    // the parity of t was miscompiled in the peeled iteration t = 1: DESIGN.md section 12)
    char *iCur = smem + OFF_I, *iPrev = smem + OFF_I + I_SLOT, *iFree = smem + OFF_I + 2 * I_SLOT;
    // iteration t: step 1 on relative plane t - 1 (position planes t+1, t+2; momentum plane t), then step 2 on relative
    // plane t - 2 (step-1 planes t-1, t)
    for (int t = 0; t <= nz + 1; t++) {
        const unsigned sP1 = sP == 2u ? 0u : sP + 1u;                // slot of position plane t + 2
        if (TMA) {
            mbar_wait(bars + 8 * sP1, ((unsigned)(t + 2) / 3u) & 1u);
            if (inner) mbar_wait(bars + 8 * (NP + (t & 1)), (unsigned)(t >> 1) & 1u);
        }
        // ---- (a) step 1 of this thread's site in relative plane t - 1 ----
        float4 MA = make_float4(0.f, 0.f, 0.f, 0.f), MB = MA;
        float2 MC = make_float2(0.f, 0.f);
        if (act) {
            if (inner) {
                const char *ms = smem + OFF_M + (t & 1) * MSLOT_BYTES;
                MA = *reinterpret_cast<const float4 *>(ms + tid * 16);
                MB = *reinterpret_cast<const float4 *>(ms + MOFF_B + tid * 16);
                MC = *reinterpret_cast<const float2 *>(ms + MOFF_C + tid * 8);
            } else {
                MA = MAo;
                MB = MBo;
                MC = MCo;
                if (t + 1 <= nz + 1) prefetch_M(t + 1);
            }
            const char *p0 = smem + sP * P2_SLOT_BYTES, *p1 = smem + sP1 * P2_SLOT_BYTES;
            TB_ACC1(p0, p1);
            float4 OA, OB;
            float2 OC;
            pk_site_update<RR, OWN1>(cy1, fA, fB, fC, k1, MA, MB, MC, OA, OB, OC);
            *reinterpret_cast<float4 *>(iCur + eI * 16) = OA;
            *reinterpret_cast<float2 *>(iCur + I_OFF_X + eI * 8) = make_float2(OB.x, OB.y);
            *reinterpret_cast<float2 *>(iCur + I_OFF_Y + eI * 8) = make_float2(OB.z, OB.w);
            *reinterpret_cast<float2 *>(iCur + I_OFF_C + eI * 8) = OC;
        }
        if (!TMA) cp_async_wait<0>();         // the copies issued one iteration ago have landed
        // the one barrier of the iteration: step-1 plane t is complete; position plane t+1 and momentum plane t are consumed;
        // everybody is past step 2 of the previous iteration, whose older step-1 plane the NEXT iteration overwrites
        __syncthreads();
        if (issuer) {
            if (t + 4 <= nz + 3) stage_P(t + 4, sP);
            if (t + 2 <= nz + 1) stage_M(t + 2);
        }
        if (!TMA) cp_async_commit();

        // ---- (b) step 2 of the inner sites in relative plane t - 2 ----
        if (inner && act && t >= 1) {
            TB_ACC2(iPrev, iCur);
            if (t == 1) {
                pk_carry_init<RR, OWN2>(cy2, fA, fB, fC);
            } else {
                float4 OA, OB;
                float2 OC;
                pk_site_update<RR, OWN2>(cy2, fA, fB, fC, k2, MAo, MBo, MCo, OA, OB, OC);
                const size_t lin = (size_t)(z0 + t - 2) * NN + gsite;
                __stcs(reinterpret_cast<float4 *>(L.mom_out) + lin, MAo);
                __stcs(reinterpret_cast<float4 *>(L.mom_out + 4 * V) + lin, MBo);
                __stcs(reinterpret_cast<float2 *>(L.mom_out + 8 * V) + lin, MCo);
                __stcs(reinterpret_cast<float4 *>(L.pos_out) + lin, OA);
                __stcs(reinterpret_cast<float4 *>(L.pos_out + 4 * V) + lin, OB);
                __stcs(reinterpret_cast<float2 *>(L.pos_out + 8 * V) + lin, OC);
            }
        }
        if (inner) {
            MAo = MA;
            MBo = MB;
            MCo = MC;
        }
        sP = sP1;
        char *sw = iFree;                     // rotate the step-1 ring: the slot of plane t-2 is written next
        iFree = iPrev;
        iPrev = iCur;
        iCur = sw;
    }
    if (!TMA) cp_async_wait<0>();
#undef TB_ACC1
#undef TB_ACC2
}

// RR: explicit range reduction of the link phases in front of the SFU (step_site.cuh; tuning flag 2048)
template <bool RR>
__global__ void __launch_bounds__(TB_THREADS, TB_CTAS)
step_tb_kernel(TbLattice L, StepCoef k1, StepCoef k2, int zchunk, int band, const __grid_constant__ TbMaps maps)
{
    extern __shared__ __align__(128) char smem[];
    const int N = L.N;
    // (tile, z chunk) of this CTA in band order (step_tiled.cu)
    const int ntx = (N + TX - 1) / TX, nty = (N + TBY - 1) / TBY, nzc = (N + zchunk - 1) / zchunk;
    const int full = ntx * band * nzc, bnd = blockIdx.x / full, rem = blockIdx.x - bnd * full;
    const int rows = min(band, nty - bnd * band), bzc = rem / (ntx * rows), tl = rem - bzc * (ntx * rows);
    const int x0 = (tl % ntx) * TX, y0 = (bnd * band + tl / ntx) * TBY, z0 = bzc * zchunk;
    const int nz = min(zchunk, N - z0);
    // CTA-uniform choice of the staging path
    if (!(k1.flags & 2) && x0 >= 2 && x0 + TX + 2 <= N && y0 >= 2 && y0 + TBY + 2 <= N)
        tb_tile<true, RR>(L, k1, k2, maps, smem, x0, y0, z0, TX, TBY, nz);
    else
        tb_tile<false, RR>(L, k1, k2, maps, smem, x0, y0, z0, min(TX, N - x0), min(TBY, N - y0), nz);
}

}  // namespace

bool step_tb_supports(int N) { return N >= 8 && (N % 4) == 0; }

cudaError_t launch_step_tb(const TbLattice &L, StepCoef k1, StepCoef k2, cudaStream_t st, const TbMaps *m, int sms)
{
    const bool rr = (k1.flags & 2048) != 0;
    cudaError_t ea = cudaFuncSetAttribute(rr ? step_tb_kernel<true> : step_tb_kernel<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM_BYTES);
    if (ea != cudaSuccess) return ea;
    TbMaps maps;
    if (!m) {
        memset(&maps, 0, sizeof maps);
        k1.flags |= 2;                      // no tile can lie strictly inside such a lattice: cp.async path only
    } else {
        maps = *m;
    }
    // z chunk: the two extra step-1 planes and the prologue per chunk want long chunks, L2 reuse of the halos and enough CTAs
    // want short ones (measured at 1024^3 with the 32 x 16 tile: 16 planes 23.1 ms, 32: 22.3, 64: 21.9, 128: 21.6, 256: 21.7)
    int zc = (k1.flags & 512) ? 16 : (k1.flags & 1024) ? 64 : 128;
    const int N = L.N;
    const int ntx = (N + TX - 1) / TX, nty = (N + TBY - 1) / TBY;
    while (zc > 8 && (long)ntx * nty * ((N + zc - 1) / zc) < (long)sms * TB_CTAS * 4) zc >>= 1;
    if (zc > N) zc = N;
    const int nzc = (N + zc - 1) / zc;
    int band = (k1.flags & 8) ? nty : (sms * TB_CTAS + ntx - 1) / ntx;
    if (band > nty) band = nty;
    if (rr) step_tb_kernel<true><<<(unsigned)(ntx * nty * nzc), TB_THREADS, SMEM_BYTES, st>>>(L, k1, k2, zc, band, maps);
    else step_tb_kernel<false><<<(unsigned)(ntx * nty * nzc), TB_THREADS, SMEM_BYTES, st>>>(L, k1, k2, zc, band, maps);
    return cudaGetLastError();
}

}  // namespace u1u1
