// init.cu -- seeded initial-condition generator ("both complex scalar fields having
// magnitudes set by the vacuum expectation value and with random phases") and the canonical <->
// internal layout copies.  The generator is Philox4x32-10 (Salmon et al., SC'11), implemented here
// from its published definition: counter = (site index lo, hi, 0, 0), key = (seed lo, hi).
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

__device__ inline void philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3, uint32_t k0,
                                     uint32_t k1, uint32_t out[4])
{
#pragma unroll
    for (int r = 0; r < 10; r++) {
        const uint32_t hi0 = __umulhi(0xD2511F53u, c0), lo0 = 0xD2511F53u * c0;
        const uint32_t hi1 = __umulhi(0xCD9E8D57u, c2), lo1 = 0xCD9E8D57u * c2;
        const uint32_t n0 = hi1 ^ c1 ^ k0, n2 = hi0 ^ c3 ^ k1;
        c0 = n0; c1 = lo1; c2 = n2; c3 = lo0;
        k0 += 0x9E3779B9u;
        k1 += 0xBB67AE85u;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

// init_kind 0: unit-modulus scalars with iid uniform phases 2 pi r / 2^32 (r[0] -> phi, r[1] -> psi).
// Phases are evaluated in fp64 and rounded once, so the result is the fp32 rounding of the exact value.
// `pos` holds `n_own` sites starting at buffer site `lin_off` (0 / all of them for the cubic lattice; one plane in / the
// own planes for a z slab), whose GLOBAL site indices -- the Philox counters -- start at `gidx_off`.
__global__ void init_random_phase_kernel(float *pos, size_t n_own, size_t lin_off, size_t gidx_off, uint64_t seed, double eta1,
                                         double eta2)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n_own; i += (size_t)gridDim.x * blockDim.x) {
        const size_t lin = i + gidx_off;
        uint32_t r[4];
        philox4x32_10((uint32_t)lin, (uint32_t)(lin >> 32), 0u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), r);
        double sn, cs;
        sincospi(2.0 * ((double)r[0] * (1.0 / 4294967296.0)), &sn, &cs);
        float4 a;
        a.x = (float)(eta1 * cs);
        a.z = (float)(eta1 * sn);
        sincospi(2.0 * ((double)r[1] * (1.0 / 4294967296.0)), &sn, &cs);
        a.y = (float)(eta2 * cs);
        a.w = (float)(eta2 * sn);
        reinterpret_cast<float4 *>(pos)[i + lin_off] = a;           // pack A
    }
}

// init_kind 1, stage 1: complex white noise, N(0,1) per real component, Box-Muller on the site's four
// Philox words: u1 = (r+1)/2^32 in (0,1], u2 = r/2^32.  Written to 4 planes of `dst`.
// The whole smoothed generator works in fp64 (noise, taps, the three separable passes, the normalisation) in the
// 80 B/site of the second position buffer and the momentum buffer, which are free at init time: the smoothed field
// can be as small as ~1e-4 of its rms at some site, so fp32 intermediates would cost 1e-4 of phase accuracy there.
__global__ void init_noise_kernel(double *dst, size_t V, uint64_t seed)
{
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        uint32_t r[4];
        philox4x32_10((uint32_t)lin, (uint32_t)(lin >> 32), 0u, 0u, (uint32_t)seed, (uint32_t)(seed >> 32), r);
#pragma unroll
        for (int k = 0; k < 2; k++) {
            const double u1 = ((double)r[2 * k] + 1.0) * (1.0 / 4294967296.0);
            const double u2 = (double)r[2 * k + 1] * (1.0 / 4294967296.0);
            const double rad = sqrt(-2.0 * log(u1));
            double sn, cs;
            sincospi(2.0 * u2, &sn, &cs);
            dst[(size_t)(2 * k) * V + lin] = rad * cs;
            dst[(size_t)(2 * k + 1) * V + lin] = rad * sn;
        }
    }
}

struct Taps {
    double w[65];  // weights for d = -trunc..trunc
    int trunc;
};

// stage 2: one separable pass of the periodic Gaussian along direction `dir` on 4 planes.
__global__ void smooth_pass_kernel(const double *src, double *dst, size_t V, int N, int dir, Taps t)
{
    const size_t stride = dir == 0 ? 1 : (dir == 1 ? (size_t)N : (size_t)N * N);
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < 4 * V;
         lin += (size_t)gridDim.x * blockDim.x) {
        const size_t plane = lin / V, sidx = lin - plane * V;
        const int coord = (int)((sidx / stride) % (size_t)N);
        const size_t base = plane * V + sidx - (size_t)coord * stride;
        double acc = 0.0;
        for (int d = -t.trunc; d <= t.trunc; d++) {
            int cc = coord + d;
            cc = ((cc % N) + N) % N;
            acc += t.w[d + t.trunc] * src[base + (size_t)cc * stride];
        }
        dst[lin] = acc;
    }
}

// stage 3: normalise to |phi| = eta1, |psi| = eta2 (zero -> phase 0).
__global__ void normalise_kernel(const double *src, float *pos, size_t V, double eta1, double eta2)
{
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const double re = src[(size_t)(2 * s) * V + lin], im = src[(size_t)(2 * s + 1) * V + lin];
            const double n = sqrt(re * re + im * im), eta = s ? eta2 : eta1;
            pos[comp_off(2 * s, lin, V)] = (float)(n > 0 ? eta * re / n : eta);
            pos[comp_off(2 * s + 1, lin, V)] = (float)(n > 0 ? eta * im / n : 0.0);
        }
    }
}

// canonical [20][V] (component planes) <-> internal packed vectors.  ncomp canonical components
// starting at c0 are moved; `canon` points at component c0's plane.
__global__ void relayout_kernel(float *pos, float *mom, float *canon, size_t V, size_t n_own, size_t lin_off, int c0, int ncomp,
                                int to_canonical)
{
    // n_own canonical sites per component, stored from buffer site lin_off on; V = sites in the buffer (pack offsets)
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < (size_t)ncomp * n_own;
         i += (size_t)gridDim.x * blockDim.x) {
        const int c = c0 + (int)(i / n_own);
        const size_t lin = i % n_own + lin_off;
        int is_mom, comp;
        canonical_to_internal(c, is_mom, comp);
        float *internal = (is_mom ? mom : pos) + comp_off(comp, lin, V);
        if (to_canonical) canon[i] = *internal;
        else *internal = canon[i];
    }
}

// internal <- periodic tiling of a smaller canonical state [20][n][n][n] (N a multiple of n)
__global__ void import_tiled_kernel(float *pos, float *mom, const float *canon, size_t V, int N, int n)
{
    const size_t v = (size_t)n * n * n;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < 20 * V; i += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / V);
        const size_t lin = i % V;
        const int x = (int)(lin % (size_t)N), y = (int)((lin / (size_t)N) % (size_t)N), z = (int)(lin / ((size_t)N * N));
        int is_mom, comp;
        canonical_to_internal(c, is_mom, comp);
        (is_mom ? mom : pos)[comp_off(comp, lin, V)] = canon[(size_t)c * v + ((size_t)(z % n) * n + (size_t)(y % n)) * n + (size_t)(x % n)];
    }
}

// canonical sub-block [20][bz][by][bx] starting at (x0,y0,z0), periodic wrap (for sampled parity checks)
__global__ void export_block_kernel(const float *pos, const float *mom, size_t V, int N, int x0, int y0,
                                    int z0, int bx, int by, int bz, float *dst)
{
    const size_t nb = (size_t)bx * by * bz;
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < 20 * nb;
         i += (size_t)gridDim.x * blockDim.x) {
        const int c = (int)(i / nb);
        size_t r = i - (size_t)c * nb;
        const int ix = (int)(r % bx); r /= bx;
        const int iy = (int)(r % by);
        const int iz = (int)(r / by);
        const int x = ((x0 + ix) % N + N) % N, y = ((y0 + iy) % N + N) % N, z = ((z0 + iz) % N + N) % N;
        int is_mom, plane;
        canonical_to_internal(c, is_mom, plane);
        dst[i] = (is_mom ? mom : pos)[comp_off(plane, (size_t)x + (size_t)N * ((size_t)y + (size_t)N * z), V)];
    }
}

constexpr int GRID = RED_MAX_BLOCKS;      // grid-stride kernels: a few blocks per SM on any device

}  // namespace

cudaError_t launch_init_random_phase(float *pos, size_t n_own, size_t lin_off, size_t gidx_off, uint64_t seed, double eta1,
                                     double eta2, cudaStream_t st)
{
    init_random_phase_kernel<<<GRID, 256, 0, st>>>(pos, n_own, lin_off, gidx_off, seed, eta1, eta2);
    return cudaGetLastError();
}

cudaError_t launch_init_smoothed(float *pos, double *tmp_a, double *tmp_b, size_t V, int N, uint64_t seed,
                                 double width, int trunc, double eta1, double eta2, cudaStream_t st)
{
    Taps t;
    t.trunc = trunc;
    for (int d = -trunc; d <= trunc; d++) t.w[d + trunc] = exp(-(double)(d * d) / (2.0 * width * width));
    init_noise_kernel<<<GRID, 256, 0, st>>>(tmp_a, V, seed);
    double *a = tmp_a, *b = tmp_b;
    for (int dir = 0; dir < 3; dir++) {
        smooth_pass_kernel<<<GRID, 256, 0, st>>>(a, b, V, N, dir, t);
        double *s = a; a = b; b = s;
    }
    normalise_kernel<<<GRID, 256, 0, st>>>(a, pos, V, eta1, eta2);
    return cudaGetLastError();
}

cudaError_t launch_export_block(const float *pos, const float *mom, size_t V, int N, int x0, int y0, int z0,
                                int bx, int by, int bz, float *dst, cudaStream_t st)
{
    export_block_kernel<<<64, 256, 0, st>>>(pos, mom, V, N, x0, y0, z0, bx, by, bz, dst);
    return cudaGetLastError();
}

cudaError_t launch_import_tiled(float *pos, float *mom, const float *canon, size_t V, int N, int n, cudaStream_t st)
{
    import_tiled_kernel<<<GRID, 256, 0, st>>>(pos, mom, canon, V, N, n);
    return cudaGetLastError();
}

cudaError_t launch_relayout(float *pos, float *mom, float *canon, size_t V, size_t n_own, size_t lin_off, int c0, int ncomp,
                            int to_canonical, cudaStream_t st)
{
    relayout_kernel<<<GRID, 256, 0, st>>>(pos, mom, canon, V, n_own, lin_off, c0, ncomp, to_canonical);
    return cudaGetLastError();
}

}  // namespace u1u1
