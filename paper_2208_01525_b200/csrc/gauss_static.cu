// gauss_static.cu -- u1u1_gauss_violation_static (include/u1u1.h): the Gauss-law monitor (PAPER.md:73-77 Eq. 9-10, :272)
// for callers that have no device memory to spare for this library and no way of getting any.
//
// Every other diagnostic call works through a context, and a context needs a caller-allocated scratch buffer
// (10 B/site) next to the 120 B/site state.  Some users of the monitor cannot provide one: a plug-in inside a host
// application whose memory pool already owns all of HBM (cudaMalloc fails, or has to be avoided because it would
// starve the pool), an in-situ checker called from a time-critical loop (cudaMalloc / cudaFree synchronise the whole
// device and stall every other stream), a post-processor that only holds a checkpoint in the public canonical layout.
// For them this file keeps the reduction scratch INSIDE the library image: a file-scope __device__ array of a fixed,
// modest size.  Nothing here calls cudaMalloc, cudaFree or any routine that allocates device memory.
//
// The kernel is a variant of gauss_kernel (diag.cu): same per-site fp64 arithmetic, but it reads the canonical
// float32 [20][N][N][N] layout directly (no context, no import), and its blocks are tied to the lattice geometry
// -- one block per (z plane, quarter of the y rows) -- so that the number of partial rows is 4 N and the array
// below bounds N.
#include <cmath>
#include <cstdio>
#include <cstring>
#include <mutex>

#include "../../include/u1u1.h"
#include "common.cuh"

using namespace u1u1;

namespace {

constexpr int YSPLIT = 4;                                  // blocks per z plane (N is a multiple of 4)
constexpr int ROW = 8;                                     // doubles per partial row: 6 sums + 2 maxima
constexpr int MAX_ROWS = YSPLIT * U1U1_STATIC_MAX_N;
constexpr int MAX_DEVICES = 64;

// The scratch: 4 * 1024 rows of 8 doubles = 256 KiB, resident on every GPU that loads libu1u1.so until the process
// exits.  In HOST code this name is only a handle for cudaGetSymbolAddress -- it is not a device address and must never
// be handed to a kernel as one; scratch_of_current_device() below asks the runtime for the real address.
static __device__ __align__(256) double g_gauss_scratch[MAX_ROWS * ROW];

std::mutex g_setup_lock;
double *g_scratch_addr[MAX_DEVICES];                       // device address of g_gauss_scratch, per device ordinal

// Once per device, with that device current: resolve the device address of the static array.
cudaError_t scratch_of_current_device(double **out, int *dev_out)
{
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    *dev_out = dev;
    if (dev < 0 || dev >= MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> hold(g_setup_lock);
    if (!g_scratch_addr[dev]) {
        double *p = nullptr;
        e = cudaGetSymbolAddress((void **)&p, g_gauss_scratch);
        if (e != cudaSuccess) return e;
        if (!p) return cudaErrorInvalidSymbol;
        g_scratch_addr[dev] = p;
    }
    *out = g_scratch_addr[dev];
    return cudaSuccess;
}

struct GaussArgs {
    const float *canon;      // float32 [20][N][N][N]
    size_t V;
    int N;
    double inv_dx;
    double rho_p, rho_q;     // 2 e_p0^2 cG, 2 e_q0^2 cG
};

// One block per (z, quarter of the rows); a thread takes four consecutive x sites at a time, so every component plane
// is read with 128-bit loads (N is a multiple of 4 and the state 16-byte aligned: every group of four is aligned).
// Row of partials: [sum g_p^2, rho_p^2, div_p^2, sum g_q^2, rho_q^2, div_q^2, max|g_p|, max|g_q|].  Every block writes
// its whole row, so no part of the scratch has to be cleared beforehand.
__device__ inline float4 ld4(const float *p) { return *reinterpret_cast<const float4 *>(p); }
__device__ inline float at4(const float4 &v, int j) { return j == 0 ? v.x : j == 1 ? v.y : j == 2 ? v.z : v.w; }

__global__ void __launch_bounds__(RED_BLOCK) gauss_canonical_kernel(GaussArgs a, double *rows)
{
    const int N = a.N, nq = N / 4, z = blockIdx.x / YSPLIT, y0 = (blockIdx.x % YSPLIT) * (N / YSPLIT);
    const int zm = z == 0 ? N - 1 : z - 1;
    const size_t V = a.V, NN = (size_t)N * N;
    const float *f = a.canon;
    double acc[ROW] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int i = threadIdx.x; i < (N / YSPLIT) * nq; i += RED_BLOCK) {
        const int y = y0 + i / nq, x = 4 * (i % nq);
        const int xm = x == 0 ? N - 1 : x - 1, ym = y == 0 ? N - 1 : y - 1;
        const size_t row = (size_t)N * y + NN * z, lin = row + x;
        const size_t lx = row + xm, ly = (size_t)N * ym + NN * z + x, lz = (size_t)N * y + NN * zm + x;
#pragma unroll
        for (int s = 0; s < 2; s++) {
            const float *fld = f + (size_t)(4 * s) * V;             // phi_re, phi_im, Pi_re, Pi_im | psi ..., Psi ...
            const float *el = f + (size_t)(11 + 6 * s) * V;         // E_xyz | H_xyz
            const float4 fr = ld4(fld + lin), fi = ld4(fld + V + lin), pr = ld4(fld + 2 * V + lin), pi = ld4(fld + 3 * V + lin);
            const float4 ex = ld4(el + lin), ey = ld4(el + V + lin), ez = ld4(el + 2 * V + lin);
            const float4 eym = ld4(el + V + ly), ezm = ld4(el + 2 * V + lz);
            const float exm[4] = {el[lx], ex.x, ex.y, ex.z};        // E_x of the site one to the left
            const double coef = s ? a.rho_q : a.rho_p;
#pragma unroll
            for (int j = 0; j < 4; j++) {
                double div = 0.0;
                div += ((double)at4(ex, j) - (double)exm[j]) * a.inv_dx;
                div += ((double)at4(ey, j) - (double)at4(eym, j)) * a.inv_dx;
                div += ((double)at4(ez, j) - (double)at4(ezm, j)) * a.inv_dx;
                const double rho = coef * ((double)at4(fr, j) * (double)at4(pi, j) - (double)at4(fi, j) * (double)at4(pr, j));
                const double g = div - rho;
                acc[3 * s + 0] += g * g;
                acc[3 * s + 1] += rho * rho;
                acc[3 * s + 2] += div * div;
                acc[6 + s] = fmax(acc[6 + s], fabs(g));
            }
        }
    }
    __shared__ double sm[ROW][RED_BLOCK / 32];
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
    for (int k = 0; k < ROW; k++) {
        const double r = k < 6 ? warp_sum(acc[k]) : warp_max(acc[k]);
        if (lane == 0) sm[k][warp] = r;
    }
    __syncthreads();
    if (threadIdx.x < ROW) {
        const int k = threadIdx.x;
        double r = sm[k][0];
        for (int w = 1; w < RED_BLOCK / 32; w++) r = k < 6 ? r + sm[k][w] : fmax(r, sm[k][w]);
        rows[(size_t)blockIdx.x * ROW + k] = r;
    }
}

// Fold the first `nrows` rows (fixed order: bit-reproducible) and write the eight norms of u1u1_gauss_violation.
__global__ void __launch_bounds__(RED_BLOCK) gauss_finish_kernel(const double *rows, int nrows, double *out)
{
    __shared__ double sm[ROW][RED_BLOCK];
    double r[ROW] = {0, 0, 0, 0, 0, 0, 0, 0};
    for (int b = threadIdx.x; b < nrows; b += RED_BLOCK)
#pragma unroll
        for (int k = 0; k < ROW; k++) {
            const double v = rows[(size_t)b * ROW + k];
            r[k] = k < 6 ? r[k] + v : fmax(r[k], v);
        }
#pragma unroll
    for (int k = 0; k < ROW; k++) sm[k][threadIdx.x] = r[k];
    __syncthreads();
    for (int o = RED_BLOCK / 2; o > 0; o >>= 1) {
        if (threadIdx.x < o)
#pragma unroll
            for (int k = 0; k < ROW; k++)
                sm[k][threadIdx.x] = k < 6 ? sm[k][threadIdx.x] + sm[k][threadIdx.x + o]
                                           : fmax(sm[k][threadIdx.x], sm[k][threadIdx.x + o]);
        __syncthreads();
    }
    if (threadIdx.x < 2) {
        const int s = threadIdx.x;
        const double l2g = sqrt(sm[3 * s][0]), l2r = sqrt(sm[3 * s + 1][0]), l2d = sqrt(sm[3 * s + 2][0]);
        out[4 * s + 0] = l2g;
        out[4 * s + 1] = l2r;
        out[4 * s + 2] = sm[6 + s][0];
        out[4 * s + 3] = l2g / fmax(fmax(l2r, l2d), 1e-300);
    }
}

int refuse(char *err, size_t err_len, int code, const char *msg)
{
    if (err && err_len) snprintf(err, err_len, "u1u1_gauss_violation_static: %s", msg);
    return code;
}

// false only for plain pageable host memory, which no kernel can read
bool gpu_can_reach(const void *p)
{
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
        cudaGetLastError();
        return false;
    }
    return at.type != cudaMemoryTypeUnregistered;
}

}  // namespace

extern "C" int u1u1_gauss_violation_static(const void *state_canonical_dev, int32_t N, double dx, double e1, double e2,
                                           double cG, double *out_dev, void *cuda_stream, char *err_host, size_t err_len)
{
    if (err_host && err_len) err_host[0] = 0;
    if (!state_canonical_dev || !out_dev) return refuse(err_host, err_len, U1U1_EINVAL, "state or out is NULL");
    if (N > U1U1_STATIC_MAX_N) {
        char msg[160];
        snprintf(msg, sizeof msg, "N = %d exceeds U1U1_STATIC_MAX_N = %d, the largest lattice the library's built-in scratch "
                 "array (%d rows) can reduce", (int)N, U1U1_STATIC_MAX_N, MAX_ROWS);
        return refuse(err_host, err_len, U1U1_ESIZE, msg);
    }
    if (N < 8 || (N % 4) != 0) return refuse(err_host, err_len, U1U1_ESIZE, "N must be a multiple of 4, at least 8");
    if (!(dx > 0) || !(e1 > 0) || !(e2 > 0) || !std::isfinite(cG))
        return refuse(err_host, err_len, U1U1_EPARAM, "need dx > 0, e1 > 0, e2 > 0 and a finite cG");
    if (((uintptr_t)state_canonical_dev & 15) || ((uintptr_t)out_dev & 7))
        return refuse(err_host, err_len, U1U1_EINVAL, "state must be 16-byte aligned and out 8-byte aligned");
    if (!gpu_can_reach(state_canonical_dev) || !gpu_can_reach(out_dev))
        return refuse(err_host, err_len, U1U1_EINVAL, "state and out must be memory the GPU can address (DEVICE pointers)");

    double *rows = nullptr;
    int dev = -1;
    cudaError_t e = scratch_of_current_device(&rows, &dev);
    if (e != cudaSuccess) {
        char msg[160];
        snprintf(msg, sizeof msg, "cudaGetSymbolAddress of the scratch array on device %d: %s", dev, cudaGetErrorString(e));
        return refuse(err_host, err_len, U1U1_ECUDA, msg);
    }

    GaussArgs a;
    a.canon = (const float *)state_canonical_dev;
    a.N = N;
    a.V = (size_t)N * N * N;
    a.inv_dx = 1.0 / dx;
    a.rho_p = 2.0 * e1 * e1 * cG;
    a.rho_q = 2.0 * e2 * e2 * cG;
    const int nrows = YSPLIT * N;
    cudaStream_t st = (cudaStream_t)cuda_stream;
    gauss_canonical_kernel<<<nrows, RED_BLOCK, 0, st>>>(a, rows);
    gauss_finish_kernel<<<1, RED_BLOCK, 0, st>>>(rows, nrows, out_dev);
    e = cudaGetLastError();
    if (e != cudaSuccess) {
        char msg[160];
        snprintf(msg, sizeof msg, "kernel launch: %s", cudaGetErrorString(e));
        return refuse(err_host, err_len, U1U1_ECUDA, msg);
    }
    return U1U1_OK;
}
