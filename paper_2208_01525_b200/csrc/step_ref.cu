// step_ref.cu -- reference fused kick+drift kernel: one thread per site, every stencil operand
// fetched straight from global memory (L1/L2 provide the reuse).  Kept as kernel_variant = 1: it is
// the simplest correct CUDA statement of PAPER.md Eq. 17-26 (:108-158) and the A/B partner of the
// tiled kernel in step_tiled.cu.  Curl in plaquette form, exactly as PAPER.md:139 Eq. 20 prints it.
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

// P_ij at site (x,y,z): theta_i(x) + theta_j(x+i) - theta_i(x+j) - theta_j(x)
template <typename R>
__device__ inline R plaq(const float *th, size_t V, Idx at, int x, int y, int z, int i, int j)
{
    const float *ti = th + (size_t)i * V, *tj = th + (size_t)j * V;
    return (R)ti[at(x, y, z)] + (R)tj[at(x + dxi(i), y + dyi(i), z + dzi(i))] -
           (R)ti[at(x + dxi(j), y + dyi(j), z + dzi(j))] - (R)tj[at(x, y, z)];
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

    R mod2[2];
#pragma unroll
    for (int s = 0; s < 2; s++) {
        const R re = P[(size_t)(2 * s) * V + c], im = P[(size_t)(2 * s + 1) * V + c];
        mod2[s] = re * re + im * im;
    }

#pragma unroll
    for (int s = 0; s < 2; s++) {
        const float *fre = P + (size_t)(2 * s) * V, *fim = fre + V;
        const float *th = P + (size_t)(4 + 3 * s) * V;
        const R fr = fre[c], fi = fim[c];
        R lap_re = (R)0, lap_im = (R)0, J[3], curl[3];
#pragma unroll
        for (int j = 0; j < 3; j++) {
            const size_t ip = at(x + dxi(j), y + dyi(j), z + dzi(j));
            const size_t im_ = at(x - dxi(j), y - dyi(j), z - dzi(j));
            R sn, cs;
            sincos_r((R)th[(size_t)j * V + c], &sn, &cs);          // U = exp(-i theta)
            const R hr = cs * (R)fre[ip] + sn * (R)fim[ip];       // U phi(x+j)
            const R hi = cs * (R)fim[ip] - sn * (R)fre[ip];
            sincos_r((R)th[(size_t)j * V + im_], &sn, &cs);
            const R br = cs * (R)fre[im_] - sn * (R)fim[im_];     // conj(U(x-j)) phi(x-j)
            const R bi = cs * (R)fim[im_] + sn * (R)fre[im_];
            lap_re += hr + br - (R)2 * fr;
            lap_im += hi + bi - (R)2 * fi;
            J[j] = fr * hi - fi * hr;                           // Im(conj(phi) U phi(x+j))
        }
#pragma unroll
        for (int i = 0; i < 3; i++) {
            R acc = (R)0;
#pragma unroll
            for (int j = 0; j < 3; j++) {
                if (j == i) continue;
                acc += plaq<R>(th, V, at, x, y, z, i, j) -
                       plaq<R>(th, V, at, x - dxi(j), y - dyi(j), z - dzi(j), i, j);
            }
            curl[i] = acc;
        }
        const R sig = s ? k.sig2sq : k.sig1sq, sigo = s ? k.sig1sq : k.sig2sq;
        const R lamh = s ? k.lamh2 : k.lamh1, cur = s ? k.cur2 : k.cur1;
        const R bracket = lamh * (mod2[s] - sig) - k.kap * (mod2[1 - s] - sigo);
        float *M = L.mom;
        float *O = L.pos_out;
        // scalar kick (Eq. 17-18) and drift (Eq. 23-24)
        const R pr = (R)k.aS * (R)M[(size_t)(2 * s) * V + c] + k.bS * (lap_re * k.inv_dx2 - fr * bracket);
        const R pi = (R)k.aS * (R)M[(size_t)(2 * s + 1) * V + c] + k.bS * (lap_im * k.inv_dx2 - fi * bracket);
        M[(size_t)(2 * s) * V + c] = (float)pr;
        M[(size_t)(2 * s + 1) * V + c] = (float)pi;
        O[(size_t)(2 * s) * V + c] = (float)(fr + k.dtau * pr);
        O[(size_t)(2 * s + 1) * V + c] = (float)(fi + k.dtau * pi);
        // gauge kick (Eq. 20-21) and drift (Eq. 25-26)
#pragma unroll
        for (int i = 0; i < 3; i++) {
            const size_t m = (size_t)(4 + 3 * s + i) * V + c;
            const R e = (R)k.aG * (R)M[m] + k.bG * (cur * J[i] - curl[i] * k.inv_dx3);
            M[m] = (float)e;
            O[m] = (float)((R)th[(size_t)i * V + c] + k.dtau_dx * e);
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
