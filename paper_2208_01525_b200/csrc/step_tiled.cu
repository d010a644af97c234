// step_tiled.cu -- the production fused kick+drift kernel (Eq. 17-26).
//
// One CTA owns an xy tile of TX x TY sites and marches through a chunk of z planes.  The three position
// packs of each plane (A = phi,psi; B = in-plane links of both sectors; C = z links; tile + one-site halo,
// periodic wrap resolved at load time) are staged into a 4-slot shared-memory ring with cp.async
// (LDGSTS 16 B / 8 B), one plane ahead of the arithmetic.  Every stencil operand -- the covariant
// 7-point Laplacian of phi, psi through the link phases and the plaquette curl of theta^A, theta^B -- is
// a vector read from shared memory (7 + 11 LDS.128 and 8 LDS.64 per site for BOTH sectors), and each
// site's 20 words make one HBM round trip: 3 vector loads of positions (+ halo, served by L2), 3 of
// momenta, 3 + 3 vector stores (new positions to the other ping-pong buffer, momenta in place).
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

constexpr int TX = 32;              // tile width  (one warp along x)
constexpr int TY = 8;               // tile height (one warp per row)
constexpr int NTHREADS = TX * TY;
constexpr int ROWS = TY + 2;        // + halo rows y0-1, y0+wy
constexpr int COLS = TX + 2;        // + halo columns x0-1, x0+wx
constexpr int NELEM = ROWS * COLS;  // staged sites per plane (340)
// one ring slot: A float4[NELEM] | B float4[NELEM] | C float2[NELEM]  = 13 600 B
constexpr int SLOT_BYTES = NELEM * (16 + 16 + 8);
constexpr int OFF_B = NELEM * 16, OFF_C = NELEM * 32;
constexpr int NSLOT = 4;            // ring: z-1, z, z+1 in use, z+2 in flight
constexpr int NITEM = (3 * NELEM + NTHREADS - 1) / NTHREADS;   // copies per thread per plane (4)
// momentum ring: every thread prefetches ITS OWN site's three momentum packs one plane ahead (private data:
// no barrier needed, only cp.async.wait_group), 2 slots of MA float4[NTHREADS] | MB float4[NTHREADS] | MC float2[NTHREADS]
constexpr int MSLOT_BYTES = NTHREADS * (16 + 16 + 8);
constexpr int MOFF_B = NTHREADS * 16, MOFF_C = NTHREADS * 32;
constexpr int SMEM_BYTES = NSLOT * SLOT_BYTES + 2 * MSLOT_BYTES;

__device__ inline void cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ inline void cp_async8(void *smem_dst, const void *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ inline void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N_>
__device__ inline void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N_) : "memory"); }

__device__ inline int wrapi(int v, int N) { return v < 0 ? v + N : (v >= N ? v - N : v); }

// What one thread copies for every plane (fixed across planes; only the z offset changes).
struct LoadPlan {
    size_t goff[NITEM];   // global BYTE offset inside the position buffer, without z
    int soff[NITEM];      // shared byte offset inside a slot; -1 = nothing
    int width[NITEM];     // bytes per site of this pack (16 or 8): z stride = width * N^2
};

__device__ inline LoadPlan make_plan(int N, size_t V, int x0, int y0, int wx, int wy)
{
    LoadPlan p;
#pragma unroll
    for (int k = 0; k < NITEM; k++) {
        const int item = threadIdx.x + k * NTHREADS;      // pack-major, then row, then column
        const int pack = item / NELEM, e = item - pack * NELEM, r = e / COLS, c = e - r * COLS;
        const bool ok = pack < 3 && r <= wy + 1 && c <= wx + 1;
        const int y = wrapi(r == wy + 1 ? y0 + wy : y0 - 1 + r, N);
        const int x = wrapi(c == wx + 1 ? x0 + wx : x0 - 1 + c, N);
        const size_t lin = (size_t)y * N + (size_t)x;
        const int w = pack == 2 ? 8 : 16;
        p.width[k] = w;
        p.goff[k] = (pack == 0 ? 0 : pack == 1 ? 16 * V : 32 * V) + lin * w;
        p.soff[k] = ok ? (pack == 0 ? 0 : pack == 1 ? OFF_B : OFF_C) + e * w : -1;
    }
    return p;
}

__device__ inline void load_plane(const LoadPlan &p, const char *pos, char *slot, size_t zplane /* z N^2 */)
{
#pragma unroll
    for (int k = 0; k < NITEM; k++) {
        if (p.soff[k] < 0) continue;
        if (p.width[k] == 16) cp_async16(slot + p.soff[k], pos + p.goff[k] + zplane * 16);
        else cp_async8(slot + p.soff[k], pos + p.goff[k] + zplane * 8);
    }
    cp_async_commit();
}

// exp(-i theta): accurate sincosf (1-2 ulp) or, with FAST, two-constant range reduction to [-pi, pi]
// followed by the SFU approximations (abs. error ~ 5e-7).
template <bool FAST>
__device__ inline void phasor(float th, float &sn, float &cs)
{
    if (FAST) {
        // MUFU.SIN/COS take the angle in turns and reduce it themselves: one FMUL by 1/(2 pi) + 2 MUFU.
        // Error max(5e-7, 6e-8 |theta|): the explicit two-constant reduction only pays for |theta| >> 8.
        __sincosf(th, &sn, &cs);
    } else {
        sincosf(th, &sn, &cs);
    }
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
// roundoff instead of fp32-ARITHMETIC roundoff (measured 10-40x smaller residual).
template <bool FAST, typename R>
__global__ void __launch_bounds__(NTHREADS, sizeof(R) == 8 ? 2 : 3) step_tiled_kernel(Lattice L, StepCoef k, int zchunk)
{
    extern __shared__ __align__(16) char ring[];    // NSLOT * SLOT_BYTES | 2 * MSLOT_BYTES
    char *const mring = ring + NSLOT * SLOT_BYTES;
    const int N = L.N;
    const size_t V = L.V, NN = (size_t)N * N;
    const int tx = threadIdx.x & (TX - 1), ty = threadIdx.x / TX;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * zchunk;
    const int wx = min(TX, N - x0), wy = min(TY, N - y0), nz = min(zchunk, N - z0);
    const bool active = tx < wx && ty < wy;
    const LoadPlan plan = make_plan(N, V, x0, y0, wx, wy);
    const char *pos = reinterpret_cast<const char *>(L.pos_in);

    // prologue: planes z0-1, z0, z0+1 into slots 0, 1, 2
#pragma unroll
    for (int j = 0; j < 3; j++) load_plane(plan, pos, ring + j * SLOT_BYTES, (size_t)wrapi(z0 - 1 + j, N) * NN);

    const int e_own = (ty + 1) * COLS + tx + 1;     // this thread's site inside a staged plane
    const size_t gsite = (size_t)(y0 + ty) * N + (size_t)(x0 + tx);
    const char *momb = reinterpret_cast<const char *>(L.mom);
    auto load_mom = [&](int slot, size_t lin) {
        char *m = mring + slot * MSLOT_BYTES;
        cp_async16(m + threadIdx.x * 16, momb + lin * 16);
        cp_async16(m + MOFF_B + threadIdx.x * 16, momb + 16 * V + lin * 16);
        cp_async8(m + MOFF_C + threadIdx.x * 8, momb + 32 * V + lin * 8);
    };
    if (active) load_mom(0, (size_t)z0 * NN + gsite);
    cp_async_commit();
    const R aS = k.aS, bS = k.bS, aG = k.aG, bG = k.bG, inv_dx2 = k.inv_dx2, inv_dx3 = k.inv_dx3;
    const R dtau = k.dtau, dtau_dx = k.dtau_dx;
    constexpr int XP = 1, XM = -1, YP = COLS, YM = -COLS;

    for (int iz = 0; iz < nz; iz++) {
        // plane z+1 (issued one iteration ago) has landed for this thread; the barrier publishes every
        // thread's copies and guarantees slot (iz+3)%4 (plane z-2) is no longer being read
        cp_async_wait<0>();
        __syncthreads();
        if (iz + 1 < nz) {
            if (active) load_mom((iz + 1) & 1, (size_t)(z0 + iz + 1) * NN + gsite);
            load_plane(plan, pos, ring + ((iz + 3) & 3) * SLOT_BYTES, (size_t)wrapi(z0 + iz + 2, N) * NN);
        }
        if (!active) continue;

        const char *sm = ring + ((iz + 0) & 3) * SLOT_BYTES;   // plane z-1
        const char *sc = ring + ((iz + 1) & 3) * SLOT_BYTES;   // plane z
        const char *sp = ring + ((iz + 2) & 3) * SLOT_BYTES;   // plane z+1
        auto A = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + (e_own + d) * 16); };
        auto B = [&](const char *s, int d) { return *reinterpret_cast<const float4 *>(s + OFF_B + (e_own + d) * 16); };
        auto C = [&](const char *s, int d) { return *reinterpret_cast<const float2 *>(s + OFF_C + (e_own + d) * 8); };
        const size_t lin = (size_t)(z0 + iz) * NN + gsite;

        // momenta of this site: prefetched one plane ahead into this thread's private ring entry
        const char *mslot = mring + (iz & 1) * MSLOT_BYTES;
        float4 MA = *reinterpret_cast<const float4 *>(mslot + threadIdx.x * 16);
        float4 MB = *reinterpret_cast<const float4 *>(mslot + MOFF_B + threadIdx.x * 16);
        float2 MC = *reinterpret_cast<const float2 *>(mslot + MOFF_C + threadIdx.x * 8);

        const float4 Ac = A(sc, 0), Axp = A(sc, XP), Axm = A(sc, XM), Ayp = A(sc, YP), Aym = A(sc, YM);
        const float4 Azp = A(sp, 0), Azm = A(sm, 0);
        const float4 Bc = B(sc, 0), Bxp = B(sc, XP), Bxm = B(sc, XM), Byp = B(sc, YP), Bym = B(sc, YM);
        const float4 Bxmyp = B(sc, XM + YP), Bxpym = B(sc, XP + YM);
        const float4 Bzp = B(sp, 0), Bxmzp = B(sp, XM), Bymzp = B(sp, YM), Bzm = B(sm, 0);
        const float2 Cc = C(sc, 0), Cxp = C(sc, XP), Cxm = C(sc, XM), Cyp = C(sc, YP), Cym = C(sc, YM);
        const float2 Czm = C(sm, 0), Cxpzm = C(sm, XP), Cypzm = C(sm, YP);

        const R m2p = (R)Ac.x * (R)Ac.x + (R)Ac.y * (R)Ac.y;
        const R m2q = (R)Ac.z * (R)Ac.z + (R)Ac.w * (R)Ac.w;
        float4 OA, OB;
        float2 OC;

#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int a0 = 2 * s, a1 = 2 * s + 1;               // lanes of this sector in packs A and B
            const R fr = ln4(Ac, a0), fi = ln4(Ac, a1);
            // ---- covariant Laplacian and currents (Eq. 17-18; current of Eq. 20-21) ----
            const float thc[3] = {ln4(Bc, a0), ln4(Bc, a1), ln2(Cc, s)};
            const float thm[3] = {ln4(Bxm, a0), ln4(Bym, a1), ln2(Czm, s)};        // theta_i(x - i)
            const float fpr[3] = {ln4(Axp, a0), ln4(Ayp, a0), ln4(Azp, a0)};       // f(x + i)
            const float fpi[3] = {ln4(Axp, a1), ln4(Ayp, a1), ln4(Azp, a1)};
            const float fmr[3] = {ln4(Axm, a0), ln4(Aym, a0), ln4(Azm, a0)};       // f(x - i)
            const float fmi[3] = {ln4(Axm, a1), ln4(Aym, a1), ln4(Azm, a1)};
            R lap_re = (R)-6 * fr, lap_im = (R)-6 * fi, J[3];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                float snf, csf;
                phasor<FAST>(thc[i], snf, csf);
                R sn = snf, cs = csf;
                const R hr = cs * (R)fpr[i] + sn * (R)fpi[i], hi = cs * (R)fpi[i] - sn * (R)fpr[i];
                phasor<FAST>(thm[i], snf, csf);
                sn = snf; cs = csf;
                const R br = cs * (R)fmr[i] - sn * (R)fmi[i], bi = cs * (R)fmi[i] + sn * (R)fmr[i];
                lap_re += hr + br;
                lap_im += hi + bi;
                J[i] = fr * hi - fi * hr;
            }
            const R sig = s ? k.sig2sq : k.sig1sq, sigo = s ? k.sig1sq : k.sig2sq;
            const R m2 = s ? m2q : m2p, m2o = s ? m2p : m2q;
            const R bracket = (R)(s ? k.lamh2 : k.lamh1) * (m2 - sig) - (R)k.kap * (m2o - sigo);
            const float pr = (float)(aS * (R)ln4(MA, a0) + bS * (lap_re * inv_dx2 - fr * bracket));
            const float pi = (float)(aS * (R)ln4(MA, a1) + bS * (lap_im * inv_dx2 - fi * bracket));
            set4(MA, a0, pr);
            set4(MA, a1, pi);
            set4(OA, a0, fmaf(k.dtau, pr, ln4(Ac, a0)));
            set4(OA, a1, fmaf(k.dtau, pi, ln4(Ac, a1)));

            // ---- lattice curl of the plaquettes, sum_{j != i} [P_ij(x) - P_ij(x-j)] (Eq. 20-21) ----
            const float Pxy = plaq(thc[0], ln4(Bxp, a1), ln4(Byp, a0), thc[1]);
            const float Pxy_my = plaq(ln4(Bym, a0), ln4(Bxpym, a1), thc[0], thm[1]);
            const float Pxy_mx = plaq(thm[0], thc[1], ln4(Bxmyp, a0), ln4(Bxm, a1));
            const float Pyz = plaq(thc[1], ln2(Cyp, s), ln4(Bzp, a1), thc[2]);
            const float Pyz_mz = plaq(ln4(Bzm, a1), ln2(Cypzm, s), thc[1], thm[2]);
            const float Pyz_my = plaq(thm[1], thc[2], ln4(Bymzp, a1), ln2(Cym, s));
            const float Pzx = plaq(thc[2], ln4(Bzp, a0), ln2(Cxp, s), thc[0]);
            const float Pzx_mx = plaq(ln2(Cxm, s), ln4(Bxmzp, a0), thc[2], thm[0]);
            const float Pzx_mz = plaq(thm[2], thc[0], ln2(Cxpzm, s), ln4(Bzm, a0));
            const float cc[3] = {(Pxy - Pxy_my) - (Pzx - Pzx_mz), (Pyz - Pyz_mz) - (Pxy - Pxy_mx),
                                 (Pzx - Pzx_mx) - (Pyz - Pyz_my)};
            const R cur = s ? k.cur2 : k.cur1;
            const float e0 = (float)(aG * (R)ln4(MB, a0) + bG * (cur * J[0] - (R)cc[0] * inv_dx3));
            const float e1 = (float)(aG * (R)ln4(MB, a1) + bG * (cur * J[1] - (R)cc[1] * inv_dx3));
            const float e2 = (float)(aG * (R)ln2(MC, s) + bG * (cur * J[2] - (R)cc[2] * inv_dx3));
            set4(MB, a0, e0);
            set4(MB, a1, e1);
            set2(MC, s, e2);
            set4(OB, a0, fmaf(k.dtau_dx, e0, thc[0]));
            set4(OB, a1, fmaf(k.dtau_dx, e1, thc[1]));
            set2(OC, s, fmaf(k.dtau_dx, e2, thc[2]));
        }
        (void)dtau; (void)dtau_dx;
        __stcs(reinterpret_cast<float4 *>(L.mom) + lin, MA);
        __stcs(reinterpret_cast<float4 *>(L.mom + 4 * V) + lin, MB);
        __stcs(reinterpret_cast<float2 *>(L.mom + 8 * V) + lin, MC);
        __stcs(reinterpret_cast<float4 *>(L.pos_out) + lin, OA);
        __stcs(reinterpret_cast<float4 *>(L.pos_out + 4 * V) + lin, OB);
        __stcs(reinterpret_cast<float2 *>(L.pos_out + 8 * V) + lin, OC);
    }
    cp_async_wait<0>();
}

int pick_zchunk(int N)
{
    // enough CTAs to fill 148 SMs x 3 several times over, chunks long enough to amortise the 2-plane prologue
    const int tiles = ((N + TX - 1) / TX) * ((N + TY - 1) / TY);
    int zc = 64;
    while (zc > 8 && (long)tiles * ((N + zc - 1) / zc) < 148L * 3 * 4) zc >>= 1;
    return zc < N ? zc : N;
}

template <bool FAST, typename R>
cudaError_t launch_one(const Lattice &L, const StepCoef &k, cudaStream_t st)
{
    constexpr int SMEM = SMEM_BYTES;
    static bool configured = false;
    if (!configured) {
        cudaError_t e = cudaFuncSetAttribute(step_tiled_kernel<FAST, R>, cudaFuncAttributeMaxDynamicSharedMemorySize, SMEM);
        if (e != cudaSuccess) return e;
        configured = true;
    }
    const int zc = pick_zchunk(L.N);
    dim3 grid((L.N + TX - 1) / TX, (L.N + TY - 1) / TY, (L.N + zc - 1) / zc);
    step_tiled_kernel<FAST, R><<<grid, NTHREADS, SMEM, st>>>(L, k, zc);
    return cudaGetLastError();
}

}  // namespace

bool step_tiled_supports(int N) { return N >= 8 && (N % 4) == 0; }

// mode bit 0: SFU sin/cos; bit 1: fp32 kick chain (default is the fp64 chain)
cudaError_t launch_step_tiled(const Lattice &L, const StepCoef &k, cudaStream_t st, int mode)
{
    switch (mode & 3) {
        case 0: return launch_one<false, double>(L, k, st);
        case 1: return launch_one<true, double>(L, k, st);
        case 2: return launch_one<false, float>(L, k, st);
        default: return launch_one<true, float>(L, k, st);
    }
}

}  // namespace u1u1
