// step_ref.cu -- reference fused kick+drift kernel: one thread per site, every stencil operand
// fetched straight from global memory through the scalar accessor comp_off() (L1/L2 provide the
// reuse).  Kept as kernel_variant 1 (fp32) / 3 (fp64 arithmetic): the simplest correct CUDA statement
// of PAPER.md Eq. 17-26 (:108-158) and the A/B partner of the tiled kernel in step_tiled.cu.
// Curl in plaquette form, exactly as PAPER.md:139 Eq. 20 prints it.
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

struct Idx {
    int N;
    __device__ size_t operator()(int x, int y, int z) const
    {
        x = x < 0 ? x + N : (x >= N ? x - N : x);
        y = y < 0 ? y + N : (y >= N ? y - N : y);
        z = z < 0 ? z + N : (z >= N ? z - N : z);
        return (size_t)x + (size_t)N * ((size_t)y + (size_t)N * (size_t)z);
    }
};

__device__ inline int dxi(int d) { return d == 0; }
__device__ inline int dyi(int d) { return d == 1; }
__device__ inline int dzi(int d) { return d == 2; }

// P_ij at site (x,y,z) of the sector whose links are logical components t0..t0+2:
// theta_i(x) + theta_j(x+i) - theta_i(x+j) - theta_j(x)
template <typename R>
__device__ inline R plaq(const float *P, int t0, size_t V, Idx at, int x, int y, int z, int i, int j)
{
    return (R)P[comp_off(t0 + i, at(x, y, z), V)] +
           (R)P[comp_off(t0 + j, at(x + dxi(i), y + dyi(i), z + dzi(i)), V)] -
           (R)P[comp_off(t0 + i, at(x + dxi(j), y + dyi(j), z + dzi(j)), V)] -
           (R)P[comp_off(t0 + j, at(x, y, z), V)];
}

__device__ inline void sincos_r(float t, float *s, float *c) { sincosf(t, s, c); }
__device__ inline void sincos_r(double t, double *s, double *c) { sincos(t, s, c); }

template <typename R>
__global__ void __launch_bounds__(256) step_ref_kernel(Lattice L, StepCoef k)
{
    const int N = L.N;
    const int x = blockIdx.x * blockDim.x + threadIdx.x;
    const int y = blockIdx.y * blockDim.y + threadIdx.y;
    const int z = blockIdx.z;
    if (x >= N || y >= N) return;
    const size_t V = L.V;
    const Idx at{N};
    const size_t c = at(x, y, z);
    const float *P = L.pos_in;
    float *M = L.mom;
    float *O = L.pos_out;

    R mod2[2];
#pragma unroll
    for (int s = 0; s < 2; s++) {
        const R re = P[comp_off(2 * s, c, V)], im = P[comp_off(2 * s + 1, c, V)];
        mod2[s] = re * re + im * im;
    }

#pragma unroll
    for (int s = 0; s < 2; s++) {
        const int f0 = 2 * s, t0 = 4 + 3 * s;           // logical components of this sector
        const R fr = P[comp_off(f0, c, V)], fi = P[comp_off(f0 + 1, c, V)];
        R lap_re = (R)0, lap_im = (R)0, J[3], curl[3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const size_t ip = at(x + dxi(j), y + dyi(j), z + dzi(j));
            const size_t im_ = at(x - dxi(j), y - dyi(j), z - dzi(j));
            R sn, cs;
            sincos_r((R)P[comp_off(t0 + j, c, V)], &sn, &cs);                  // U = exp(-i theta)
            const R ar = P[comp_off(f0, ip, V)], ai = P[comp_off(f0 + 1, ip, V)];
            const R hr = cs * ar + sn * ai;                                     // U phi(x+j)
            const R hi = cs * ai - sn * ar;
            sincos_r((R)P[comp_off(t0 + j, im_, V)], &sn, &cs);
            const R br_ = P[comp_off(f0, im_, V)], bi_ = P[comp_off(f0 + 1, im_, V)];
            const R br = cs * br_ - sn * bi_;                                   // conj(U(x-j)) phi(x-j)
            const R bi = cs * bi_ + sn * br_;
            lap_re += hr + br - (R)2 * fr;
            lap_im += hi + bi - (R)2 * fi;
            J[j] = fr * hi - fi * hr;                                           // Im(conj(phi) U phi(x+j))
        }
#pragma unroll
        for (int i = 0; i < 3; i++) {
            R acc = (R)0;
#pragma unroll
            for (int j = 0; j < 3; j++) {
                if (j == i) continue;
                acc += plaq<R>(P, t0, V, at, x, y, z, i, j) -
                       plaq<R>(P, t0, V, at, x - dxi(j), y - dyi(j), z - dzi(j), i, j);
            }
            curl[i] = acc;
        }
        const R sig = s ? k.sig2sq : k.sig1sq, sigo = s ? k.sig1sq : k.sig2sq;
        const R lamh = s ? k.lamh2 : k.lamh1, cur = s ? k.cur2 : k.cur1;
        const R bracket = lamh * (mod2[s] - sig) - (R)k.kap * (mod2[1 - s] - sigo);
        // scalar kick (Eq. 17-18) and drift (Eq. 23-24)
        const size_t o0 = comp_off(f0, c, V), o1 = comp_off(f0 + 1, c, V);
        const R pr = (R)k.aS * (R)M[o0] + (R)k.bS * (lap_re * (R)k.inv_dx2 - fr * bracket);
        const R pi = (R)k.aS * (R)M[o1] + (R)k.bS * (lap_im * (R)k.inv_dx2 - fi * bracket);
        M[o0] = (float)pr;
        M[o1] = (float)pi;
        O[o0] = (float)(fr + (R)k.dtau * pr);
        O[o1] = (float)(fi + (R)k.dtau * pi);
        // gauge kick (Eq. 20-21) and drift (Eq. 25-26)
#pragma unroll
        for (int i = 0; i < 3; i++) {
            const size_t m = comp_off(t0 + i, c, V);
            const R e = (R)k.aG * (R)M[m] + (R)k.bG * (cur * J[i] - curl[i] * (R)k.inv_dx3);
            M[m] = (float)e;
            O[m] = (float)((R)P[m] + (R)k.dtau_dx * e);
        }
    }
}

}  // namespace

cudaError_t launch_step_ref(const Lattice &L, const StepCoef &k, cudaStream_t stream, bool fp64)
{
    dim3 block(64, 4, 1);
    dim3 grid((L.N + 63) / 64, (L.N + 3) / 4, L.N);
    if (fp64) step_ref_kernel<double><<<grid, block, 0, stream>>>(L, k);
    else step_ref_kernel<float><<<grid, block, 0, stream>>>(L, k);
    return cudaGetLastError();
}

}  // namespace u1u1
