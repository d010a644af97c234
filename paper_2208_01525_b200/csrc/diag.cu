// diag.cu -- read-only diagnostic sweeps: Gauss-law monitor (Eq. 9-10), per-plaquette
// windings and pierced cells (:183-194, :234, :252), Lagrangian / velocity / energy sums (:196-224,
// Eq. 33, 36-37).  Per-site terms in fp32, combinations and accumulation in fp64, deterministic
// two-stage block reductions (warp shuffles -> shared -> per-block partials -> one folding block).
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
    double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t nb[3] = {w.at(w.m(x), y, z), w.at(x, w.m(y), z), w.at(x, y, w.m(z))};
#pragma unroll
        for (int s = 0; s < 2; s++) {
            double div = 0.0;
#pragma unroll
            for (int i = 0; i < 3; i++)
                div += ((double)mom[comp_off(4 + 3 * s + i, lin, V)] -
                        (double)mom[comp_off(4 + 3 * s + i, nb[i], V)]) * k.inv_dx;
            const double fr = pos[comp_off(2 * s, lin, V)], fi = pos[comp_off(2 * s + 1, lin, V)];
            const double pr = mom[comp_off(2 * s, lin, V)], pi = mom[comp_off(2 * s + 1, lin, V)];
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

// ---------------------------------------------------------------------------------------------
// Link angle chi_i(x) = arg( conj(f(x)) U_i(x) f(x+i) ) in (-pi, pi], atan2(0,0) = 0.
// ---------------------------------------------------------------------------------------------
__device__ inline float link_angle(const float *pos, int f0, int tcomp, size_t V, size_t c, size_t nb)
{
    float sn, cs;
    sincosf(pos[comp_off(tcomp, c, V)], &sn, &cs);
    const float ar = pos[comp_off(f0, nb, V)], ai = pos[comp_off(f0 + 1, nb, V)];
    const float hr = cs * ar + sn * ai, hi = cs * ai - sn * ar;
    const float fr = pos[comp_off(f0, c, V)], fi = pos[comp_off(f0 + 1, c, V)];
    const float re = fr * hr + fi * hi, im = fr * hi - fi * hr;
    return (re == 0.f && im == 0.f) ? 0.f : atan2f(im, re);
}

__device__ inline int near_cut(float chi) { return (3.14159265358979323846 - fabs((double)chi)) < 1e-5; }

// Winding code byte: bits 0..3 = W + 8 (W in [-8, 7]), bit 4 = near-branch-cut flag.
__device__ inline uint8_t encode_w(int w, int nearflag) { return (uint8_t)(((w + 8) & 15) | (nearflag << 4)); }
__device__ inline int decode_w(uint8_t code) { return (int)(code & 15) - 8; }

// One thread per site, both sectors, three orientations (xy, yz, zx).  Each thread evaluates the 9
// link angles its three plaquettes need (3x redundant across neighbours; this sweep runs once per
// 20-100 steps).  Partials: [sum|W_p|, sum|W_q|, near_p, near_q | max|W|].
__global__ void __launch_bounds__(RED_BLOCK) winding_kernel(const float *pos, size_t V, int N,
                                                            uint8_t *codes, double *partials)
{
    const Wrap w{N};
    double acc[5] = {0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t nb[3] = {w.at(w.p(x), y, z), w.at(x, w.p(y), z), w.at(x, y, w.p(z))};
        // forward neighbours of the forward neighbours: nb2[i][j] = x + i + j
        const int xs[3] = {w.p(x), x, x}, ys[3] = {y, w.p(y), y}, zs[3] = {z, z, w.p(z)};
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int f0 = 2 * s, t0 = 4 + 3 * s;
            float chi0[3];
#pragma unroll
            for (int i = 0; i < 3; i++) chi0[i] = link_angle(pos, f0, t0 + i, V, lin, nb[i]);
#pragma unroll
            for (int o = 0; o < 3; o++) {
                const int i = o, j = (o + 1) % 3;              // (xy), (yz), (zx)
                // x+i+j
                const size_t nij = w.at(j == 0 ? w.p(xs[i]) : xs[i], j == 1 ? w.p(ys[i]) : ys[i],
                                        j == 2 ? w.p(zs[i]) : zs[i]);
                const float c1 = chi0[i];
                const float c2 = link_angle(pos, f0, t0 + j, V, nb[i], nij);  // chi_j(x+i)
                const float c3 = link_angle(pos, f0, t0 + i, V, nb[j], nij);  // chi_i(x+j)
                const float c4 = chi0[j];
                const float P = pos[comp_off(t0 + i, lin, V)] + pos[comp_off(t0 + j, nb[i], V)] -
                                pos[comp_off(t0 + i, nb[j], V)] - pos[comp_off(t0 + j, lin, V)];
                const float sum = c1 + c2 - c3 - c4 + P;
                const int W = __float2int_rn(sum * 0.15915494309189535f);
                const int nr = near_cut(c1) | near_cut(c2) | near_cut(c3) | near_cut(c4);
                codes[(size_t)(3 * s + o) * V + lin] = encode_w(W, nr);
                acc[s] += (double)abs(W);
                acc[2 + s] += (double)nr;
                acc[4] = fmax(acc[4], (double)abs(W));
            }
        }
    }
    block_reduce_store<5>(acc, 4, partials);
}

// Pierced-cell arrays and the fast-method overlap count.  Partials: [N_p, N_q, N_pq].
__global__ void __launch_bounds__(RED_BLOCK) cells_kernel(const uint8_t *codes, size_t V, int N,
                                                          uint8_t *cells, double *partials)
{
    const Wrap w{N};
    double acc[3] = {0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t nx = w.at(w.p(x), y, z), ny = w.at(x, w.p(y), z), nz = w.at(x, y, w.p(z));
        int C[2];
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const uint8_t *Wxy = codes + (size_t)(3 * s + 0) * V, *Wyz = codes + (size_t)(3 * s + 1) * V,
                          *Wzx = codes + (size_t)(3 * s + 2) * V;
            C[s] = abs(decode_w(Wxy[lin])) + abs(decode_w(Wxy[nz])) + abs(decode_w(Wyz[lin])) +
                   abs(decode_w(Wyz[nx])) + abs(decode_w(Wzx[lin])) + abs(decode_w(Wzx[ny]));
            cells[(size_t)s * V + lin] = (uint8_t)C[s];
        }
        acc[0] += C[0] > 0;
        acc[1] += C[1] > 0;
        acc[2] += (C[0] > 0) && (C[1] > 0);
    }
    block_reduce_store<3>(acc, 3, partials);
}

// Lagrangian, velocity-estimator and energy sums.  Partials:
// [sum L, sum kin L, sum grad L, sum kin V, sum grad V, sum V, sum kin, sum grad, sum elec, sum mag, sum pot]
__global__ void __launch_bounds__(RED_BLOCK) density_kernel(const float *pos, const float *mom, size_t V,
                                                            int N, DiagCoef k, double *partials)
{
    const Wrap w{N};
    double acc[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t nb[3] = {w.at(w.p(x), y, z), w.at(x, w.p(y), z), w.at(x, y, w.p(z))};
        double kin = 0, grad = 0, elec = 0, mag = 0, m2[2];
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const int f0 = 2 * s, t0 = 4 + 3 * s;
            const float fr = pos[comp_off(f0, lin, V)], fi = pos[comp_off(f0 + 1, lin, V)];
            const float pr = mom[comp_off(f0, lin, V)], pi = mom[comp_off(f0 + 1, lin, V)];
            const double inv2e2 = 1.0 / (2.0 * (s ? k.e2 * k.e2 : k.e1 * k.e1));
            kin += (double)pr * pr + (double)pi * pi;
            m2[s] = (double)fr * fr + (double)fi * fi;
            float thc[3];
#pragma unroll
            for (int i = 0; i < 3; i++) {
                thc[i] = pos[comp_off(t0 + i, lin, V)];
                float sn, cs;
                sincosf(thc[i], &sn, &cs);
                const float ar = pos[comp_off(f0, nb[i], V)], ai = pos[comp_off(f0 + 1, nb[i], V)];
                const float dr = (cs * ar + sn * ai) - fr, di = (cs * ai - sn * ar) - fi;
                grad += ((double)dr * dr + (double)di * di) * k.inv_dx2;
                const double e = mom[comp_off(t0 + i, lin, V)];
                elec += e * e * inv2e2;
            }
#pragma unroll
            for (int i = 0; i < 3; i++)
#pragma unroll
                for (int j = i + 1; j < 3; j++) {
                    const float P = thc[i] + pos[comp_off(t0 + j, nb[i], V)] - pos[comp_off(t0 + i, nb[j], V)] - thc[j];
                    const double F = (double)P * k.inv_dx2;
                    mag += F * F * inv2e2;
                }
        }
        const double a2 = m2[0] - k.sig1sq, b2 = m2[1] - k.sig2sq;
        const double vint = k.kappa * a2 * b2;
        const double pot = 0.25 * k.lam1 * a2 * a2 + 0.25 * k.lam2 * b2 * b2 - vint;
        const double lag = kin - grad + (elec - mag) / k.c - k.c * pot;
        acc[0] += lag;
        acc[1] += kin * lag;
        acc[2] += grad * lag;
        acc[3] += kin * vint;
        acc[4] += grad * vint;
        acc[5] += vint;
        acc[6] += kin;
        acc[7] += grad;
        acc[8] += elec;
        acc[9] += mag;
        acc[10] += pot;
    }
    block_reduce_store<11>(acc, 11, partials);
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

cudaError_t launch_gauss(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                         double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V);
    gauss_kernel<<<nb, RED_BLOCK, 0, st>>>(pos, mom, V, N, k, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 8, 6, result);
    return cudaGetLastError();
}

cudaError_t launch_windings(const float *pos, size_t V, int N, uint8_t *codes, uint8_t *cells,
                            double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V);
    winding_kernel<<<nb, RED_BLOCK, 0, st>>>(pos, V, N, codes, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 5, 4, result);
    cells_kernel<<<nb, RED_BLOCK, 0, st>>>(codes, V, N, cells, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 3, 3, result + 8);
    return cudaGetLastError();
}

cudaError_t launch_densities(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                             double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V);
    density_kernel<<<nb, RED_BLOCK, 0, st>>>(pos, mom, V, N, k, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 11, 11, result);
    return cudaGetLastError();
}

cudaError_t launch_decode_windings(const uint8_t *codes, size_t n, int8_t *w_out, uint8_t *near_out,
                                   cudaStream_t st)
{
    decode_windings_kernel<<<148 * 8, 256, 0, st>>>(codes, n, w_out, near_out);
    return cudaGetLastError();
}

}  // namespace u1u1
