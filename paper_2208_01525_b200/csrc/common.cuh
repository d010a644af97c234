// common.cuh -- internal layout, per-step coefficients and reduction helpers shared by the CUDA
// kernels of libu1u1.so.  Nothing here is shared with oracle/ (separate code base by design).
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace u1u1 {

// ------------------------------------------------------------------------------------------------
// Internal HBM layout: packed vectors per site, site index lin = x + N (y + N z).
// A position buffer (10 V floats) and the momentum buffer (10 V floats) have the same shape:
//   pack A: float4[V]  (phi_re, psi_re, phi_im, psi_im)        | momenta: (Pi_re, Psi_re, Pi_im, Psi_im)
//   pack B: float4[V]  (thetaA_x, thetaB_x, thetaA_y, thetaB_y) | (E_x, H_x, E_y, H_y)
//   pack C: float2[V]  (thetaA_z, thetaB_z)                     | (E_z, H_z)
// so one site moves as 3 vector loads + 6 vector stores, and a stencil neighbour's scalars (both
// sectors) or in-plane links (both sectors) arrive in one 128-bit shared-memory read.
// The SAME quantity of the two sectors always sits in an aligned pair of adjacent words: the two sectors obey the
// same equations, so the step kernel runs them through the packed fp32x2 instructions of sm_100 (FFMA2 / FADD2 /
// FMUL2: one issue slot for both sectors) straight from the 64-bit halves of its vector loads.
// state buffer = [pos0 | pos1 | mom], 30 V floats.
// "Logical" component order used by the scalar accessors: 0 phi_re 1 phi_im 2 psi_re 3 psi_im
// 4..6 thetaA_xyz 7..9 thetaB_xyz (momenta: Pi, Psi, E_xyz, H_xyz).
// ------------------------------------------------------------------------------------------------
constexpr int NPOS = 10;
constexpr int NMOM = 10;

struct Lattice {
    const float *pos_in;  // positions at tau (read)
    float *pos_out;       // positions at tau + dtau (written)
    float *mom;           // momenta, updated in place
    size_t V;             // sites in one buffer: N^3, or N * N * (nz_own + 2) for a z slab
    int N;
    // z slab of a lattice that is split over several GPUs (zero for the ordinary cubic lattice):
    // the buffers hold planes 0 .. nz_own + 1, plane 0 and plane nz_own + 1 being copies of the neighbouring slabs'
    // boundary planes.  The step kernel updates planes 1 .. nz_own and ALSO stores its top / bottom plane of pos_out
    // into the halo plane of the neighbour above / below (plain stores through peer memory: NVLink when the neighbour
    // lives on another GPU), so the exchange rides on the kernel's own output pass.
    int nz_own;           // 0: cubic lattice, periodic in z inside the buffer
    float *peer_up_out;   // pos_out buffer of the slab above (its plane 0 receives this slab's top plane)
    float *peer_dn_out;   // pos_out buffer of the slab below (its plane nz_own_dn + 1 receives this slab's bottom plane)
    size_t peer_dn_plane; // nz_own_dn + 1
    size_t peer_up_V, peer_dn_V;   // sites in the neighbours' buffers (their pack offsets)
};

// float offset of logical component c (0..9) of site lin inside a 10 V-float buffer
__host__ __device__ inline size_t comp_off(int c, size_t lin, size_t V)
{
    if (c < 4) return 4 * lin + (size_t)(2 * (c & 1) + (c >> 1));
    const int s = (c - 4) / 3, i = (c - 4) % 3;
    return i < 2 ? 4 * V + 4 * lin + (size_t)(2 * i + s) : 8 * V + 2 * lin + (size_t)s;
}

// first (re / x link) and second (im / y link) word of sector s in a float4 of pack A or B; word of sector s in pack C
__host__ __device__ inline float pk0(const float4 &v, int s) { return s ? v.y : v.x; }
__host__ __device__ inline float pk1(const float4 &v, int s) { return s ? v.w : v.z; }
__host__ __device__ inline float pkc(const float2 &v, int s) { return s ? v.y : v.x; }

// canonical component -> (is_momentum, logical component)
__host__ __device__ inline void canonical_to_internal(int c, int &is_mom, int &plane)
{
    // canonical: 0 phi_re 1 phi_im 2 Pi_re 3 Pi_im 4 psi_re 5 psi_im 6 Psi_re 7 Psi_im
    //            8..10 thetaA 11..13 E 14..16 thetaB 17..19 H
    if (c < 8) {
        is_mom = (c >> 1) & 1;
        plane = (c >> 2) * 2 + (c & 1);
    } else if (c < 14) {
        is_mom = c >= 11;
        plane = 4 + (c - (is_mom ? 11 : 8));
    } else {
        is_mom = c >= 17;
        plane = 7 + (c - (is_mom ? 17 : 14));
    }
}

// Per-step coefficients, computed on the host in fp64 (PAPER.md:133 Eq. 19, :147 Eq. 22, :89 Eq. 12)
// and rounded once to fp32.  Friction (BASELINE.json prephase) is folded into the four kick factors.
struct StepCoef {
    float aS, bS;          // Pi+  = aS Pi-  + bS [lap - c phi (...)],  aS = f(1-delta)/(1+delta), bS = f dtau/(1+delta)
    float aG, bG;          // E+   = aG E-   + bG [-curl + current],    aG = f(1-omega)/(1+omega), bG = f dtau/(1+omega)
    float lamh1, lamh2;    // c lambda_p0/2, c lambda_q0/2
    float kap;             // c kappa_0
    float sig1sq, sig2sq;  // sigma_p^2, sigma_q^2
    float cur1, cur2;      // 2 e_p0^2 c / dx, 2 e_q0^2 c / dx
    float inv_dx2;         // 1/dx^2
    float inv_dx3;         // 1/dx^3
    float dtau;            // drift of the scalars
    float dtau_dx;         // drift of the link phases: theta += dtau dx E
    float aSm1, aGm1;      // aS - 1, aG - 1 (rounded from fp64): Pi+ = Pi- + [(aS-1) Pi- + bS (...)] keeps ONE rounding at |Pi|
    int flags;             // tuning switches of the tiled kernel (kernel_variant >> 4), 0 in production:
                           // 2 = no TMA (cp.async staging everywhere), 4 = momenta by ld.global.cs, 8 = plain grid order
};

// Coefficients of the diagnostic sweeps.
struct DiagCoef {
    double c;              // a^{2s}
    double cG;             // Gauss-law coefficient c (1+delta)/(1+omega) of the last step
    double inv_dx;
    double inv_dx2;
    double e1, e2, lam1, lam2, kappa, sig1sq, sig2sq;
};

// ------------------------------------------------------------------------------------------------
// Deterministic two-stage reductions: every block writes NRED doubles of partial sums (and maxima),
// a one-block kernel folds the partials.  No atomics, so results are bit-reproducible run to run.
// ------------------------------------------------------------------------------------------------
constexpr int RED_BLOCK = 256;
constexpr int RED_MAX_BLOCKS = 1184;     // cap on reduction / grid-stride blocks: sizes the partials buffer, device independent
constexpr int RED_SLOTS = 32;

__device__ inline double warp_sum(double v)
{
    for (int o = 16; o > 0; o >>= 1) v += __shfl_down_sync(0xffffffffu, v, o);
    return v;
}
__device__ inline double warp_max(double v)
{
    for (int o = 16; o > 0; o >>= 1) v = fmax(v, __shfl_down_sync(0xffffffffu, v, o));
    return v;
}

// Reduce `n` per-thread values (first n_sum are summed, the rest are maxima) over the block and
// store them at out[blockIdx.x * RED_SLOTS + k].
template <int NVAL>
__device__ inline void block_reduce_store(const double (&v)[NVAL], int n_sum, double *out)
{
    __shared__ double sm[NVAL][RED_BLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < NVAL; k++) {
        double r = (k < n_sum) ? warp_sum(v[k]) : warp_max(v[k]);
        if (lane == 0) sm[k][warp] = r;
    }
    __syncthreads();
    if (threadIdx.x < NVAL) {
        const int k = threadIdx.x;
        double r = sm[k][0];
        for (int w = 1; w < RED_BLOCK / 32; w++) r = (k < n_sum) ? r + sm[k][w] : fmax(r, sm[k][w]);
        out[(size_t)blockIdx.x * RED_SLOTS + k] = r;
    }
}

}  // namespace u1u1
