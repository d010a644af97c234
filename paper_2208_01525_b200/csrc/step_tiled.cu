// step_tiled.cu -- the production fused kick+drift kernel (Eq. 17-26).
//
// One CTA owns an xy tile of TX x TY sites and marches through a chunk of z planes.  The 10 position
// words of each plane (tile + one-site halo, periodic wrap resolved at load time) are staged into a
// 4-slot shared-memory ring with cp.async (LDGSTS, 16-byte interior / 4-byte halo columns), one plane
// ahead of the arithmetic, so every stencil operand -- the covariant 7-point Laplacian of phi, psi
// through the link phases, and the curl-curl of theta^A, theta^B -- is read from shared memory and each
// site's 20 words make one HBM round trip: read 10 positions (+ halo, from L2) and 10 momenta, write 10
// new positions (to the other ping-pong buffer) and 10 momenta (in place).
//
// curl-curl: sum_{j != i} [P_ij(x) - P_ij(x-j)] = -Lap theta_i(x) + D(x+i) - D(x), with
// D(x) = sum_j [theta_j(x) - theta_j(x-j)] the backward lattice divergence -- the exact lattice form
// of curl curl = -Laplacian + grad div; algebraically identical to PAPER.md:139 Eq. 20's plaquette
// differences, fewer shared-memory reads.
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

constexpr int TX = 32;              // tile width  (one warp along x: conflict-free shared rows)
constexpr int TY = 8;               // tile height (one warp per row)
constexpr int NTHREADS = TX * TY;
constexpr int ROWS = TY + 2;        // + halo rows y0-1, y0+wy
constexpr int PITCH = TX + 8;       // interior at columns 4..4+wx-1 (16-byte aligned), halos at 3 and 4+wx
constexpr int PLANE = NPOS * ROWS * PITCH;   // floats per staged plane (4000 -> 16 000 B)
constexpr int NSLOT = 4;            // ring: z-1, z, z+1 in use, z+2 in flight
constexpr int NROWITEM = 4;         // 16-byte row items per thread: ceil(10*10*8 / 256)

__device__ inline void cp_async16(float *smem_dst, const float *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ inline void cp_async4(float *smem_dst, const float *gsrc)
{
    const unsigned s = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;\n" ::"r"(s), "l"(gsrc) : "memory");
}
__device__ inline void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N_>
__device__ inline void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N_) : "memory"); }

__device__ inline int wrapi(int v, int N) { return v < 0 ? v + N : (v >= N ? v - N : v); }

// What one thread copies for every plane (fixed across planes; only the z offset changes).
struct LoadPlan {
    size_t goff[NROWITEM];   // global float offset (component plane + row + column), without z
    int soff[NROWITEM];      // shared float offset inside a slot; -1 = nothing
    size_t hgoff;            // halo-column element
    int hsoff;
};

__device__ inline LoadPlan make_plan(int N, size_t V, int x0, int y0, int wx, int wy)
{
    LoadPlan p;
    const int t = threadIdx.x;
#pragma unroll
    for (int k = 0; k < NROWITEM; k++) {
        const int item = t + k * NTHREADS;          // (comp, row, col4) = (item/80, (item/8)%10, item%8)
        const int q = item & 7, r = (item >> 3) % ROWS, c = item / (8 * ROWS);
        const bool ok = c < NPOS && r <= wy + 1 && 4 * q < wx;
        const int y = wrapi(r == wy + 1 ? y0 + wy : y0 - 1 + r, N);
        p.goff[k] = (size_t)c * V + (size_t)y * N + (size_t)(x0 + 4 * q);
        p.soff[k] = ok ? (c * ROWS + r) * PITCH + 4 + 4 * q : -1;
    }
    {
        const int side = t & 1, r = (t >> 1) % ROWS, c = t / (2 * ROWS);
        const bool ok = c < NPOS && r <= wy + 1;
        const int y = wrapi(r == wy + 1 ? y0 + wy : y0 - 1 + r, N);
        const int x = side ? wrapi(x0 + wx, N) : wrapi(x0 - 1, N);
        p.hgoff = (size_t)c * V + (size_t)y * N + (size_t)x;
        p.hsoff = ok ? (c * ROWS + r) * PITCH + (side ? 4 + wx : 3) : -1;
    }
    return p;
}

__device__ inline void load_plane(const LoadPlan &p, const float *pos, float *slot, size_t zoff)
{
#pragma unroll
    for (int k = 0; k < NROWITEM; k++)
        if (p.soff[k] >= 0) cp_async16(slot + p.soff[k], pos + p.goff[k] + zoff);
    if (p.hsoff >= 0) cp_async4(slot + p.hsoff, pos + p.hgoff + zoff);
    cp_async_commit();
}

// exp(-i theta): accurate sincosf (Cody-Waite + minimax polynomials; 1-2 ulp) or, with FAST, two-constant
// range reduction to [-pi, pi] followed by the SFU approximations (abs. error ~ 5e-7).
template <bool FAST>
__device__ inline void phasor(float th, float &sn, float &cs)
{
    if (FAST) {
        const float n = rintf(th * 0.15915494309189535f);
        float r = fmaf(n, -6.2831854820251465f, th);     // 2 pi = 6.2831854820251465 - 1.7484556e-7
        r = fmaf(n, 1.7484556000744883e-7f, r);
        sn = __sinf(r);
        cs = __cosf(r);
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

// R = arithmetic type of the kick chain (hops, Laplacian, currents, potential, momentum update):
// double keeps the discrete Gauss identity Im(phi* D-D+ phi) = d-_i Im(phi* D+_i phi) at fp32-STORAGE
// roundoff instead of fp32-ARITHMETIC roundoff (40x smaller residual, measured).
template <bool FAST, typename R>
__global__ void __launch_bounds__(NTHREADS, sizeof(R) == 8 ? 2 : 3) step_tiled_kernel(Lattice L, StepCoef k, int zchunk)
{
    extern __shared__ __align__(16) float ring[];   // NSLOT * PLANE floats
    const int N = L.N;
    const size_t V = L.V, NN = (size_t)N * N;
    const int tx = threadIdx.x & (TX - 1), ty = threadIdx.x / TX;
    const int x0 = blockIdx.x * TX, y0 = blockIdx.y * TY, z0 = blockIdx.z * zchunk;
    const int wx = min(TX, N - x0), wy = min(TY, N - y0), nz = min(zchunk, N - z0);
    const bool active = tx < wx && ty < wy;
    const LoadPlan plan = make_plan(N, V, x0, y0, wx, wy);
    const float *pos = L.pos_in;

    // prologue: planes z0-1, z0, z0+1 into slots 0, 1, 2
#pragma unroll
    for (int j = 0; j < 3; j++) load_plane(plan, pos, ring + j * PLANE, (size_t)wrapi(z0 - 1 + j, N) * NN);

    const int own = (ty + 1) * PITCH + tx + 4;      // this thread's site inside a component plane
    const size_t gsite = (size_t)(y0 + ty) * N + (size_t)(x0 + tx);
    const R aS = k.aS, bS = k.bS, aG = k.aG, bG = k.bG, inv_dx2 = k.inv_dx2, inv_dx3 = k.inv_dx3;
    const R dtau = k.dtau, dtau_dx = k.dtau_dx;

    for (int iz = 0; iz < nz; iz++) {
        // plane z+1 (issued one iteration ago) has landed for this thread; the barrier publishes every
        // thread's copies and guarantees slot (iz+3)%4 (plane z-2) is no longer being read
        cp_async_wait<0>();
        __syncthreads();
        if (iz + 1 < nz)
            load_plane(plan, pos, ring + ((iz + 3) & 3) * PLANE, (size_t)wrapi(z0 + iz + 2, N) * NN);
        if (!active) continue;

        const float *pm = ring + ((iz + 0) & 3) * PLANE + own;   // plane z-1
        const float *pc = ring + ((iz + 1) & 3) * PLANE + own;   // plane z
        const float *pp = ring + ((iz + 2) & 3) * PLANE + own;   // plane z+1
        const size_t g = (size_t)(z0 + iz) * NN + gsite;

        // momenta of this site: issued first so their latency overlaps the arithmetic
        float M[NMOM];
#pragma unroll
        for (int c = 0; c < NMOM; c++) M[c] = __ldcs(L.mom + (size_t)c * V + g);

        constexpr int CP = ROWS * PITCH;                       // component stride inside a slot
        const R m2p = (R)pc[0] * (R)pc[0] + (R)pc[CP] * (R)pc[CP];
        const R m2q = (R)pc[2 * CP] * (R)pc[2 * CP] + (R)pc[3 * CP] * (R)pc[3 * CP];

#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int F = 2 * s * CP, T = (4 + 3 * s) * CP;    // scalar and link component offsets
            const R fr = pc[F], fi = pc[F + CP];
            // ---- covariant Laplacian and currents (Eq. 17-18; current of Eq. 20-21) ----
            const float thc[3] = {pc[T], pc[T + CP], pc[T + 2 * CP]};
            const float thm[3] = {pc[T - 1], pc[T + CP - PITCH], pm[T + 2 * CP]};   // theta_i(x - i)
            const float fpr[3] = {pc[F + 1], pc[F + PITCH], pp[F]};                 // f(x + i)
            const float fpi[3] = {pc[F + CP + 1], pc[F + CP + PITCH], pp[F + CP]};
            const float fmr[3] = {pc[F - 1], pc[F - PITCH], pm[F]};                 // f(x - i)
            const float fmi[3] = {pc[F + CP - 1], pc[F + CP - PITCH], pm[F + CP]};
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
            const float pr = (float)(aS * (R)M[2 * s] + bS * (lap_re * inv_dx2 - fr * bracket));
            const float pi = (float)(aS * (R)M[2 * s + 1] + bS * (lap_im * inv_dx2 - fi * bracket));
            __stcs(L.mom + (size_t)(2 * s) * V + g, pr);
            __stcs(L.mom + (size_t)(2 * s + 1) * V + g, pi);
            __stcs(L.pos_out + (size_t)(2 * s) * V + g, (float)(fr + dtau * (R)pr));
            __stcs(L.pos_out + (size_t)(2 * s + 1) * V + g, (float)(fi + dtau * (R)pi));

            // ---- lattice curl of the plaquettes, sum_{j != i} [P_ij(x) - P_ij(x-j)] (Eq. 20-21) ----
            const float *tx_ = pc + T, *ty_ = pc + T + CP, *tz_ = pc + T + 2 * CP;   // plane z
            const float *txp = pp + T, *typ = pp + T + CP;                            // plane z+1
            const float *txm = pm + T, *tym = pm + T + CP, *tzm = pm + T + 2 * CP;   // plane z-1
            const float Pxy = plaq(thc[0], ty_[1], tx_[PITCH], thc[1]);
            const float Pxy_my = plaq(tx_[-PITCH], ty_[1 - PITCH], thc[0], thm[1]);
            const float Pxy_mx = plaq(thm[0], thc[1], tx_[PITCH - 1], ty_[-1]);
            const float Pyz = plaq(thc[1], tz_[PITCH], typ[0], thc[2]);
            const float Pyz_mz = plaq(tym[0], tzm[PITCH], thc[1], thm[2]);
            const float Pyz_my = plaq(thm[1], thc[2], typ[-PITCH], tz_[-PITCH]);
            const float Pzx = plaq(thc[2], txp[0], tz_[1], thc[0]);
            const float Pzx_mx = plaq(tz_[-1], txp[-1], thc[2], thm[0]);
            const float Pzx_mz = plaq(thm[2], thc[0], tzm[1], txm[0]);
            const float cc[3] = {(Pxy - Pxy_my) - (Pzx - Pzx_mz), (Pyz - Pyz_mz) - (Pxy - Pxy_mx),
                                 (Pzx - Pzx_mx) - (Pyz - Pyz_my)};
            const R cur = s ? k.cur2 : k.cur1;
#pragma unroll
            for (int i = 0; i < 3; i++) {
                const int c = 4 + 3 * s + i;
                const float e = (float)(aG * (R)M[c] + bG * (cur * J[i] - (R)cc[i] * inv_dx3));
                __stcs(L.mom + (size_t)c * V + g, e);
                __stcs(L.pos_out + (size_t)c * V + g, (float)((R)thc[i] + dtau_dx * (R)e));
            }
        }
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

}  // namespace

bool step_tiled_supports(int N) { return N >= 8 && (N % 4) == 0; }

template <bool FAST, typename R>
static cudaError_t launch_one(const Lattice &L, const StepCoef &k, cudaStream_t st)
{
    constexpr int SMEM = NSLOT * PLANE * (int)sizeof(float);
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
