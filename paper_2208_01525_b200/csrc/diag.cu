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
            const float E[3] = {s ? eb.z : eb.x, s ? eb.w : eb.y, s ? ec.y : ec.x};
            const float Em[3] = {s ? ebx.z : ebx.x, s ? eby.w : eby.y, s ? ecz.y : ecz.x};
            double div = 0.0;
#pragma unroll
            for (int i = 0; i < 3; i++) div += ((double)E[i] - (double)Em[i]) * k.inv_dx;
            const double fr = s ? a.z : a.x, fi = s ? a.w : a.y;
            const double pr = s ? ma.z : ma.x, pi = s ? ma.w : ma.y;
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


// Winding code byte: bits 0..3 = W + 8 (W in [-8, 7]), bit 4 = near-branch-cut flag.
__device__ inline uint8_t encode_w(int w, int nearflag) { return (uint8_t)(((w + 8) & 15) | (nearflag << 4)); }
__device__ inline int decode_w(uint8_t code) { return (int)(code & 15) - 8; }

// ---------------------------------------------------------------------------------------------
// Windings (reading R-12), tiled.  chi_i(x) = arg(conj(f(x)) U_i(x) f(x+i)) is the principal value of
// v = alpha(x+i) - alpha(x) - theta_i(x) with alpha = arg f, so ONE atan2 per site and sector replaces a
// sincos + atan2 per link: chi = v - 2 pi rint(v / 2 pi).  A CTA owns a 32 x 8 tile, marches in z, keeps the
// phases alpha of the tile + its (+x, +y) halo for planes z and z+1 in shared memory, and evaluates the nine
// link angles each site's three plaquettes need from them.  W = rint((sum of chi + P) / 2 pi) as before;
// a link whose end point is exactly zero has chi = 0 (atan2(0,0) = 0, R-15).
// Partials: [sum|W_p|, sum|W_q|, near_p, near_q | max|W|].
// ---------------------------------------------------------------------------------------------
constexpr int WTX = 32, WTY = 8, WEX = WTX + 1, WEY = WTY + 1, WNE = WEX * WEY, WZC = 32;

// atan2 in ~20 instructions: octant reduction to t = min/max in [0, 1] and the degree-8 (in t^2) polynomial of
// Abramowitz & Stegun 4.4.49 (|error| <= 2e-8 in exact arithmetic; ~4e-7 in fp32 with the fast division), the same
// accuracy as libm's atan2f at a fifth of the instructions.  Never called with x = y = 0.
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

__device__ inline float chi_of(float alpha_a, float alpha_b, float theta)
{
    const float v = (alpha_b - alpha_a) - theta;                       // NaN if an end point is exactly zero
    const float n = (fmaf(v, 0.15915494309189535f, 12582912.f)) - 12582912.f;      // rint(v / 2 pi), |v| < 2^22
    float r = fmaf(n, -6.2831854820251465f, v);                        // 2 pi = 6.2831854820251465 - 1.7484556e-7
    r = fmaf(n, 1.7484556000744883e-7f, r);
    return r != r ? 0.f : r;             // within rounding of (-pi, pi]; anything at the cut is flagged near-cut
}
// near-cut flag in fp32: pi - |chi| < 1e-5  <=>  |chi| > 3.14158265...
__device__ inline int near_cut32(float chi) { return fabsf(chi) > 3.14158265f; }

__global__ void __launch_bounds__(RED_BLOCK) winding_tiled_kernel(const float *pos, size_t V, int N, uint8_t *codes,
                                                                  double *partials, int ntx, int nty, int nzc)
{
    __shared__ float alpha[2][2][WNE];                // [plane buffer][sector][extended tile site]
    const Wrap w{N};
    const size_t NN = (size_t)N * N;
    const float4 *PA = reinterpret_cast<const float4 *>(pos), *PB = reinterpret_cast<const float4 *>(pos + 4 * V);
    const float2 *PC = reinterpret_cast<const float2 *>(pos + 8 * V);
    const int tid = threadIdx.x, tx = tid & (WTX - 1), ty = tid / WTX;
    int sumw[2] = {0, 0}, nnear[2] = {0, 0}, maxw = 0;
    const int items = ntx * nty * nzc;
    for (int item = blockIdx.x; item < items; item += gridDim.x) {
        const int bx = item % ntx, by = (item / ntx) % nty, bz = item / (ntx * nty);
        const int x0 = bx * WTX, y0 = by * WTY, z0 = bz * WZC;
        const int wx = min(WTX, N - x0), wy = min(WTY, N - y0), nz = min(WZC, N - z0);
        const bool active = tx < wx && ty < wy;
        // phases of plane z (periodic) for the tile and its +x / +y halo into buffer b
        auto fill = [&](int z, int b) {
            for (int e = tid; e < WNE; e += RED_BLOCK) {
                const int ey = e / WEX, ex = e - ey * WEX;
                if (ex > wx || ey > wy) continue;
                const int x = x0 + ex == N ? 0 : x0 + ex, y = y0 + ey == N ? 0 : y0 + ey;
                const float4 a = PA[(size_t)z * NN + (size_t)y * N + x];
                alpha[b][0][e] = (a.x == 0.f && a.y == 0.f) ? __int_as_float(0x7fc00000) : atan2_poly(a.y, a.x);
                alpha[b][1][e] = (a.z == 0.f && a.w == 0.f) ? __int_as_float(0x7fc00000) : atan2_poly(a.w, a.z);
            }
        };
        __syncthreads();                               // previous item's readers are done
        fill(z0, 0);
        for (int iz = 0; iz < nz; iz++) {
            const int z = z0 + iz, zp = w.p(z), cur = iz & 1, nxt = cur ^ 1;
            fill(zp, nxt);
            __syncthreads();
            if (active) {
                const int x = x0 + tx, y = y0 + ty, xp = w.p(x), yp = w.p(y);
                const size_t lin = w.at(x, y, z), lx = w.at(xp, y, z), ly = w.at(x, yp, z), lz = w.at(x, y, zp);
                const float4 Bc = PB[lin], Bx = PB[lx], By = PB[ly], Bz = PB[lz];
                const float2 Cc = PC[lin], Cx = PC[lx], Cy = PC[ly];
                const int e = ty * WEX + tx;
#pragma unroll
                for (int s = 0; s < 2; s++) {
                    const float *ac = alpha[cur][s], *an = alpha[nxt][s];
                    const float a0 = ac[e], ax = ac[e + 1], ay = ac[e + WEX], axy = ac[e + WEX + 1];
                    const float az = an[e], axz = an[e + 1], ayz = an[e + WEX];
                    const float tx0 = s ? Bc.z : Bc.x, ty0 = s ? Bc.w : Bc.y, tz0 = s ? Cc.y : Cc.x;   // theta_i(x)
                    const float ty_x = s ? Bx.w : Bx.y, tz_x = s ? Cx.y : Cx.x;                          // theta_{y,z}(x + x)
                    const float tx_y = s ? By.z : By.x, tz_y = s ? Cy.y : Cy.x;                          // theta_{x,z}(x + y)
                    const float tx_z = s ? Bz.z : Bz.x, ty_z = s ? Bz.w : Bz.y;                          // theta_{x,y}(x + z)
                    const float cx = chi_of(a0, ax, tx0), cy = chi_of(a0, ay, ty0), cz = chi_of(a0, az, tz0);
                    // orientation o = (i, j): chi_i(x) + chi_j(x+i) - chi_i(x+j) - chi_j(x) + P_ij(x)
                    const float c2[3] = {chi_of(ax, axy, ty_x), chi_of(ay, ayz, tz_y), chi_of(az, axz, tx_z)};
                    const float c3[3] = {chi_of(ay, axy, tx_y), chi_of(az, ayz, ty_z), chi_of(ax, axz, tz_x)};
                    const float c1[3] = {cx, cy, cz}, c4[3] = {cy, cz, cx};
                    const float P[3] = {tx0 + ty_x - tx_y - ty0, ty0 + tz_y - ty_z - tz0, tz0 + tx_z - tz_x - tx0};
#pragma unroll
                    for (int o = 0; o < 3; o++) {
                        const float sum = c1[o] + c2[o] - c3[o] - c4[o] + P[o];
                        const int W = __float2int_rn(sum * 0.15915494309189535f);
                        const int nr = near_cut32(c1[o]) | near_cut32(c2[o]) | near_cut32(c3[o]) | near_cut32(c4[o]);
                        codes[(size_t)(3 * s + o) * V + lin] = encode_w(W, nr);
                        sumw[s] += abs(W);
                        nnear[s] += nr;
                        maxw = max(maxw, abs(W));
                    }
                }
            }
            __syncthreads();                           // buffer `cur` is refilled next iteration
        }
    }
    const double acc[5] = {(double)sumw[0], (double)sumw[1], (double)nnear[0], (double)nnear[1], (double)maxw};
    block_reduce_store<5>(acc, 4, partials);
}

// Pierced-cell arrays and the fast-method overlap count.  Partials: [N_p, N_q, N_pq].
__global__ void __launch_bounds__(RED_BLOCK) cells_kernel(const uint8_t *codes, size_t V, int N,
                                                          uint8_t *cells, double *partials)
{
    // four consecutive x sites per thread (N is a multiple of 4): 32-bit loads of the code bytes
    const Wrap w{N};
    double acc[3] = {0, 0, 0};
    auto mag = [](uint32_t word, int k) { return abs((int)((word >> (8 * k)) & 15u) - 8); };   // |W| of byte k
    for (size_t q = (size_t)blockIdx.x * blockDim.x + threadIdx.x; q < V / 4; q += (size_t)gridDim.x * blockDim.x) {
        const size_t lin = 4 * q;
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t ny = w.at(x, w.p(y), z), nz = w.at(x, y, w.p(z)), nx4 = w.at(x + 4 == N ? 0 : x + 4, y, z);
        uint32_t C[2] = {0, 0};
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const uint8_t *Wxy = codes + (size_t)(3 * s + 0) * V, *Wyz = codes + (size_t)(3 * s + 1) * V,
                          *Wzx = codes + (size_t)(3 * s + 2) * V;
            const uint32_t xy0 = *reinterpret_cast<const uint32_t *>(Wxy + lin), xy1 = *reinterpret_cast<const uint32_t *>(Wxy + nz);
            const uint32_t yz0 = *reinterpret_cast<const uint32_t *>(Wyz + lin), zx0 = *reinterpret_cast<const uint32_t *>(Wzx + lin);
            const uint32_t zx1 = *reinterpret_cast<const uint32_t *>(Wzx + ny);
            const uint32_t yz1 = (yz0 >> 8) | ((uint32_t)Wyz[nx4] << 24);                    // W_yz at x + 1
#pragma unroll
            for (int k = 0; k < 4; k++) {
                const int c = mag(xy0, k) + mag(xy1, k) + mag(yz0, k) + mag(yz1, k) + mag(zx0, k) + mag(zx1, k);
                C[s] |= (uint32_t)c << (8 * k);
            }
            *reinterpret_cast<uint32_t *>(cells + (size_t)s * V + lin) = C[s];
        }
#pragma unroll
        for (int k = 0; k < 4; k++) {
            const int cp = (C[0] >> (8 * k)) & 255, cq = (C[1] >> (8 * k)) & 255;
            acc[0] += cp > 0;
            acc[1] += cq > 0;
            acc[2] += (cp > 0) && (cq > 0);
        }
    }
    block_reduce_store<3>(acc, 3, partials);
}

// Fast method with one cell of tolerance ("non-zero at the same location, or displaced by one cell in
// any direction"; reading R-13b): a pierced p cell counts if a pierced q cell lies in its 3x3x3 neighbourhood
// (periodic), and vice versa.  Pierced cells are sparse, so almost every thread stops after two byte loads.
// Partials: [#p cells with a q cell within one cell, #q cells with a p cell within one cell].
__global__ void __launch_bounds__(RED_BLOCK) overlap_tol_kernel(const uint8_t *cells, size_t V, int N, double *partials)
{
    const Wrap w{N};
    double acc[2] = {0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        const int cp = cells[lin], cq = cells[V + lin];
        if ((cp | cq) == 0) continue;
        if (cp > 0 && cq > 0) {                // exact overlap: both counts, no search
            acc[0] += 1.0;
            acc[1] += 1.0;
            continue;
        }
        // pierced by one type only: look for the OTHER type in the 3x3x3 neighbourhood, stop at the first hit
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const int xs[3] = {w.m(x), x, w.p(x)}, ys[3] = {w.m(y), y, w.p(y)}, zs[3] = {w.m(z), z, w.p(z)};
        const uint8_t *other = cells + (cp > 0 ? V : 0);
        int found = 0;
        for (int c = 0; c < 3 && !found; c++)
            for (int b = 0; b < 3 && !found; b++) {
                const size_t row = (size_t)N * ((size_t)ys[b] + (size_t)N * zs[c]);
                found = other[row + xs[0]] | other[row + xs[1]] | other[row + xs[2]];
            }
        if (found) acc[cp > 0 ? 0 : 1] += 1.0;
    }
    block_reduce_store<2>(acc, 2, partials);
}

// Lagrangian, velocity-estimator and energy sums.  Partials:
// [sum L, sum kin L, sum grad L, sum kin V, sum grad V, sum V, sum kin, sum grad, sum elec, sum mag, sum pot]
__global__ void __launch_bounds__(RED_BLOCK) density_kernel(const float *pos, const float *mom, size_t V,
                                                            int N, DiagCoef k, double *partials)
{
    const Wrap w{N};
    const float4 *PA = reinterpret_cast<const float4 *>(pos), *PB = reinterpret_cast<const float4 *>(pos + 4 * V);
    const float2 *PC = reinterpret_cast<const float2 *>(pos + 8 * V);
    const float4 *MA = reinterpret_cast<const float4 *>(mom), *MB = reinterpret_cast<const float4 *>(mom + 4 * V);
    const float2 *MC = reinterpret_cast<const float2 *>(mom + 8 * V);
    double acc[11] = {0, 0, 0, 0, 0, 0, 0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V;
         lin += (size_t)gridDim.x * blockDim.x) {
        int x, y, z;
        site_xyz(lin, N, x, y, z);
        const size_t nb[3] = {w.at(w.p(x), y, z), w.at(x, w.p(y), z), w.at(x, y, w.p(z))};
        const float4 Ac = PA[lin], An[3] = {PA[nb[0]], PA[nb[1]], PA[nb[2]]};
        const float4 Bc = PB[lin], Bn[3] = {PB[nb[0]], PB[nb[1]], PB[nb[2]]};
        const float2 Cc = PC[lin], Cn[2] = {PC[nb[0]], PC[nb[1]]};
        const float4 ma = MA[lin], mb = MB[lin];
        const float2 mc = MC[lin];
        // per-site terms in fp32 (each a sum of <= 18 squares), everything that is accumulated over the lattice in fp64
        float kin = 0.f, grad = 0.f, elec = 0.f, mag = 0.f, m2[2];
        const float inv_dx2 = (float)k.inv_dx2;
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const float fr = s ? Ac.z : Ac.x, fi = s ? Ac.w : Ac.y;
            const float pr = s ? ma.z : ma.x, pi = s ? ma.w : ma.y;
            const float inv2e2 = (float)(1.0 / (2.0 * (s ? k.e2 * k.e2 : k.e1 * k.e1)));
            kin += pr * pr + pi * pi;
            m2[s] = fr * fr + fi * fi;
            const float thc[3] = {s ? Bc.z : Bc.x, s ? Bc.w : Bc.y, s ? Cc.y : Cc.x};
            const float ev[3] = {s ? mb.z : mb.x, s ? mb.w : mb.y, s ? mc.y : mc.x};
            float g2 = 0.f, e2 = 0.f, f2 = 0.f;
#pragma unroll
            for (int i = 0; i < 3; i++) {
                float sn, cs;
                sincosf(thc[i], &sn, &cs);
                const float ar = s ? An[i].z : An[i].x, ai = s ? An[i].w : An[i].y;
                const float dr = (cs * ar + sn * ai) - fr, di = (cs * ai - sn * ar) - fi;
                g2 += dr * dr + di * di;
                e2 += ev[i] * ev[i];
            }
            // theta_j(x + i) for the three plaquettes (i, j) = (x,y), (x,z), (y,z) and theta_i(x + j)
            const float ty_x = s ? Bn[0].w : Bn[0].y, tx_y = s ? Bn[1].z : Bn[1].x;
            const float tz_x = s ? Cn[0].y : Cn[0].x, tx_z = s ? Bn[2].z : Bn[2].x;
            const float tz_y = s ? Cn[1].y : Cn[1].x, ty_z = s ? Bn[2].w : Bn[2].y;
            const float Pl[3] = {thc[0] + ty_x - tx_y - thc[1], thc[0] + tz_x - tx_z - thc[2], thc[1] + tz_y - ty_z - thc[2]};
#pragma unroll
            for (int q = 0; q < 3; q++) f2 += Pl[q] * Pl[q];
            grad += g2 * inv_dx2;
            elec += e2 * inv2e2;
            mag += f2 * (inv_dx2 * inv_dx2) * inv2e2;
        }
        const double a2 = (double)m2[0] - k.sig1sq, b2 = (double)m2[1] - k.sig2sq;
        const double vint = k.kappa * a2 * b2;
        const double pot = 0.25 * k.lam1 * a2 * a2 + 0.25 * k.lam2 * b2 * b2 - vint;
        const double lag = (double)kin - (double)grad + ((double)elec - (double)mag) / k.c - k.c * pot;
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

cudaError_t launch_windings(const float *pos, size_t V, int N, uint8_t *codes, uint8_t *cells,
                            double *partials, double *result, cudaStream_t st)
{
    const int nb = red_blocks(V);
    const int ntx = (N + WTX - 1) / WTX, nty = (N + WTY - 1) / WTY, nzc = (N + WZC - 1) / WZC;
    const int nbw = ntx * nty * nzc < RED_MAX_BLOCKS ? ntx * nty * nzc : RED_MAX_BLOCKS;
    winding_tiled_kernel<<<nbw, RED_BLOCK, 0, st>>>(pos, V, N, codes, partials, ntx, nty, nzc);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nbw, 5, 4, result);
    cells_kernel<<<nb, RED_BLOCK, 0, st>>>(codes, V, N, cells, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 3, 3, result + 8);
    overlap_tol_kernel<<<nb, RED_BLOCK, 0, st>>>(cells, V, N, partials);
    fold_kernel<<<1, RED_BLOCK, 0, st>>>(partials, nb, 2, 2, result + 12);
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
