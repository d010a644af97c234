// diag.cu -- the small diagnostic kernels around the fused sweep of diag_fused.cu: the stand-alone Gauss-law monitor
// (Eq. 9-10; u1u1_gauss_violation reads only the 56 B/site it needs), the fast method's overlap count
// with one cell of tolerance (:234), the decoder of the winding codes, and the folding kernel of the deterministic
// two-stage reductions (warp shuffles -> shared -> per-block partials -> one folding block).
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

struct Wrap {
    int N;
    __device__ int p(int v) const { return v + 1 == N ? 0 : v + 1; }
    __device__ int m(int v) const { return v == 0 ? N - 1 : v - 1; }
    __device__ size_t at(int x, int y, int z) const
    {
        return (size_t)x + (size_t)N * ((size_t)y + (size_t)N * (size_t)z);
    }
};

__device__ inline void site_xyz(size_t lin, int N, int &x, int &y, int &z)
{
    x = (int)(lin % (size_t)N);
    const size_t r = lin / (size_t)N;
    y = (int)(r % (size_t)N);
    z = (int)(r / (size_t)N);
}

// ---------------------------------------------------------------------------------------------
// Gauss monitor.  Partials per block: [sum g_p^2, sum rho_p^2, sum div_p^2, sum g_q^2, sum rho_q^2,
// sum div_q^2 | max|g_p|, max|g_q|].
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(RED_BLOCK) gauss_kernel(const float *pos, const float *mom, size_t V,
                                                          int N, DiagCoef k, double *partials)
{
    const Wrap w{N};
    const float4 *PA = reinterpret_cast<const float4 *>(pos);
    const float4 *MA = reinterpret_cast<const float4 *>(mom), *MB = reinterpret_cast<const float4 *>(mom + 4 * V);
    const float2 *MC = reinterpret_cast<const float2 *>(mom + 8 * V);
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const float4 a = PA[lin], ma = MA[lin], eb = MB[lin], ebx = MB[w.at(w.m(x), y, z)], eby = MB[w.at(x, w.m(y), z)];
        const float2 ec = MC[lin], ecz = MC[w.at(x, y, w.m(z))];
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const float E[3] = {pk0(eb, s), pk1(eb, s), pkc(ec, s)};
            const float Em[3] = {pk0(ebx, s), pk1(eby, s), pkc(ecz, s)};
            double div = 0.0;
#pragma unroll
            for (int i = 0; i < 3; i++) div += ((double)E[i] - (double)Em[i]) * k.inv_dx;
            const double fr = pk0(a, s), fi = pk1(a, s);
            const double pr = pk0(ma, s), pi = pk1(ma, s);
            const double e0 = s ? k.e2 : k.e1;
            const double rho = 2.0 * e0 * e0 * k.cG * (fr * pi - fi * pr);
            const double g = div - rho;
            acc[3 * s + 0] += g * g;
            acc[3 * s + 1] += rho * rho;
            acc[3 * s + 2] += div * div;
            acc[6 + s] = fmax(acc[6 + s], fabs(g));
        }
    }
    block_reduce_store<8>(acc, 6, partials);
}


// Winding code byte: bits 0..3 = W + 8 (W in [-8, 7]), bit 4 = near-branch-cut flag (written by diag_fused.cu).
__device__ inline int decode_w(uint8_t code) { return (int)(code & 15) - 8; }

// Fast method with one cell of tolerance ("non-zero at the same location, or displaced by one cell in
// any direction"; reading R-13b): a pierced p cell counts if a pierced q cell lies in its periodic 3x3x3
// neighbourhood, and vice versa.  The dilation is separable.  A thread owns four consecutive x cells (one 32-bit word
// per type; N is a multiple of 4) of one row y and marches through a chunk of z planes: per plane it ORs the words
// of rows y-1, y, y+1 (plus the bytes at x-1 and x+4) into a bit per cell, spreads that bit one cell left and right,
// and keeps the results of planes z-1, z, z+1 in registers -- 18 loads per four cells instead of 54, whatever the
// string density.  Partials: [#p cells with a q cell within one cell, #q cells with a p cell within one cell].
constexpr int TOL_ZC = 32;
__global__ void __launch_bounds__(RED_BLOCK) overlap_tol_kernel(const uint8_t *cells, size_t V, int N, double *partials)
{
    const Wrap w{N};
    const int nw = N / 4, nzc = (N + TOL_ZC - 1) / TOL_ZC;
    const size_t NN = (size_t)N * N, ncol = (size_t)nw * N * nzc;
    int acc[2] = {0, 0};
    auto nonzero_bytes = [](uint32_t v) {                     // 0x01 in every byte lane of v that is non-zero
        v |= v >> 4; v |= v >> 2; v |= v >> 1;
        return v & 0x01010101u;
    };
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < ncol; q += (size_t)gridDim.x * blockDim.x) {
        const int xw = (int)(q % (size_t)nw);
        const size_t r = q / (size_t)nw;
        const int y = (int)(r % (size_t)N), z0 = (int)(r / (size_t)N) * TOL_ZC, nz = min(TOL_ZC, N - z0);
        const int x = 4 * xw, xl = w.m(x), xr = x + 4 == N ? 0 : x + 4;
        const size_t rows[3] = {(size_t)w.m(y) * N, (size_t)y * N, (size_t)w.p(y) * N};
        // xy-dilated pierced bits (0x01 per cell) of both types in plane z
        auto plane = [&](int z, uint32_t &dp, uint32_t &dq, uint32_t &cp, uint32_t &cq) {
            const size_t zp = (size_t)z * NN;
            uint32_t mid[2] = {0, 0}, lft[2] = {0, 0}, rgt[2] = {0, 0}, own[2];
#pragma unroll
            for (int t = 0; t < 2; t++) {
#pragma unroll
                for (int b = 0; b < 3; b++) {
                    const uint8_t *src = cells + (size_t)t * V + zp + rows[b];
                    const uint32_t m = *reinterpret_cast<const uint32_t *>(src + x);
                    if (b == 1) own[t] = m;
                    mid[t] |= m;
                    lft[t] |= src[xl];
                    rgt[t] |= src[xr];
                }
                const uint32_t m = nonzero_bytes(mid[t]);
                mid[t] = m | (m << 8) | (lft[t] ? 1u : 0u) | (m >> 8) | (rgt[t] ? 0x01000000u : 0u);
            }
            dp = mid[0]; dq = mid[1]; cp = own[0]; cq = own[1];
        };
        uint32_t dpm, dqm, dpc, dqc, dpn, dqn, cpc, cqc, cpn, cqn, u0, u1;
        plane(w.m(z0), dpm, dqm, u0, u1);
        plane(z0, dpc, dqc, cpc, cqc);
        for (int iz = 0; iz < nz; iz++) {
            const int z = z0 + iz;
            plane(w.p(z), dpn, dqn, cpn, cqn);
            acc[0] += __popc(nonzero_bytes(cpc) & (dqm | dqc | dqn));
            acc[1] += __popc(nonzero_bytes(cqc) & (dpm | dpc | dpn));
            dpm = dpc; dqm = dqc; dpc = dpn; dqc = dqn; cpc = cpn; cqc = cqn;
        }
    }
    const double a[2] = {(double)acc[0], (double)acc[1]};
    block_reduce_store<2>(a, 2, partials);
}

// Fold `nblocks` partial rows into result[0..nval): first n_sum slots summed, the rest maxima.
__global__ void __launch_bounds__(RED_BLOCK) fold_kernel(const double *partials, int nblocks, int nval,
                                                         int n_sum, double *result)
{
    __shared__ double sm[RED_BLOCK];
    for (int k = 0; k < nval; k++) {
        double r = 0.0;
        for (int b = threadIdx.x; b < nblocks; b += RED_BLOCK) {
            const double v = partials[(size_t)b * RED_SLOTS + k];
            r = (k < n_sum) ? r + v : fmax(r, v);
        }
        sm[threadIdx.x] = r;
        __syncthreads();
        for (int o = RED_BLOCK / 2; o > 0; o >>= 1) {
            if (threadIdx.x < o)
                sm[threadIdx.x] = (k < n_sum) ? sm[threadIdx.x] + sm[threadIdx.x + o]
                                              : fmax(sm[threadIdx.x], sm[threadIdx.x + o]);
            __syncthreads();
        }
        if (threadIdx.x == 0) result[k] = sm[0];
        __syncthreads();
    }
}

__global__ void decode_windings_kernel(const uint8_t *codes, size_t n, int8_t *w_out, uint8_t *near_out)
{
    for (size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x; i < n;
         i += (size_t)gridDim.x * blockDim.x) {
        const uint8_t c = codes[i];
        if (w_out) w_out[i] = (int8_t)decode_w(c);
        if (near_out) near_out[i] = (c >> 4) & 1;
    }
}

int red_blocks(size_t V)
{
    const size_t need = (V + RED_BLOCK - 1) / RED_BLOCK;
    return (int)(need < (size_t)RED_MAX_BLOCKS ? need : (size_t)RED_MAX_BLOCKS);
}

}  // namespace

cudaError_t launch_fold(const double *partials, int nblocks, int nval, int n_sum, double *result, cudaStream_t st)
{
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nblocks, nval, n_sum, result);
    return cudaGetLastError();
}

cudaError_t launch_gauss(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                         double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V);
    gauss_kernel<<<nb, RED_BLOCK, 0, st>>>(pos, mom, V, N, k, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 8, 6, result);
    return cudaGetLastError();
}

cudaError_t launch_overlap_tol(const uint8_t *cells, size_t V, int N, double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V / 4);
    overlap_tol_kernel<<<nb, RED_BLOCK, 0, st>>>(cells, V, N, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 2, 2, result);
    return cudaGetLastError();
}

cudaError_t launch_decode_windings(const uint8_t *codes, size_t n, int8_t *w_out, uint8_t *near_out,
                                   cudaStream_t st)
{
    decode_windings_kernel<<<RED_MAX_BLOCKS, 256, 0, st>>>(codes, n, w_out, near_out);
    return cudaGetLastError();
}

}  // namespace u1u1
