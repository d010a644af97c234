// segments.cu -- pq-segment identification on the GPU (the paper's "robust method", PAPER.md:240-256, :390-394,
// there done off-line with ParaView's overlap + connectivity filters): connected-component labelling of the cells
// pierced by both string types, segment count N_pq, segment length (N_cells - 1) dx (:248), length threshold.
// Union-find over the periodic 26-neighbourhood (cells that share at least a corner; reading R-21) with atomicMin
// root linking; labels are site indices, so the result is independent of the execution order.
#include "common.cuh"
#include "kernels.h"

namespace u1u1 {

namespace {

__device__ inline int wrap_p(int v, int N) { return v + 1 == N ? 0 : v + 1; }
__device__ inline int wrap_m(int v, int N) { return v == 0 ? N - 1 : v - 1; }

__device__ inline void xyz_of(size_t lin, int N, int &x, int &y, int &z)
{
    x = (int)(lin % (size_t)N);
    const size_t r = lin / (size_t)N;
    y = (int)(r % (size_t)N);
    z = (int)(r / (size_t)N);
}

// label[x] = x for pq cells, -1 elsewhere.  tolerant = 0: C^p > 0 and C^q > 0 at the same cell;
// 1: a pierced cell of one type with a pierced cell of the other type in its 3x3x3 neighbourhood (R-13b).
__global__ void seg_init_kernel(const uint8_t *cells, size_t V, int N, int tolerant, int *label)
{
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V; lin += (size_t)gridDim.x * blockDim.x) {
        const int cp = cells[lin], cq = cells[V + lin];
        int on = cp > 0 && cq > 0;
        if (!on && tolerant && (cp | cq)) {
            int x, y, z;
            xyz_of(lin, N, x, y, z);
            const int xs[3] = {wrap_m(x, N), x, wrap_p(x, N)}, ys[3] = {wrap_m(y, N), y, wrap_p(y, N)},
                      zs[3] = {wrap_m(z, N), z, wrap_p(z, N)};
            int anyp = 0, anyq = 0;
            for (int c = 0; c < 3; c++)
                for (int b = 0; b < 3; b++)
                    for (int a = 0; a < 3; a++) {
                        const size_t nb = (size_t)xs[a] + (size_t)N * ((size_t)ys[b] + (size_t)N * zs[c]);
                        anyp |= cells[nb];
                        anyq |= cells[V + nb];
                    }
            on = (cp > 0 && anyq > 0) || (cq > 0 && anyp > 0);
        }
        label[lin] = on ? (int)lin : -1;
    }
}

__device__ inline int find_root(const int *label, int x)
{
    int p = label[x];
    while (p != x) {
        x = p;
        p = label[x];
    }
    return x;
}

__device__ inline void unite(int *label, int a, int b)
{
    while (true) {
        a = find_root(label, a);
        b = find_root(label, b);
        if (a == b) return;
        if (a > b) { const int t = a; a = b; b = t; }       // link the larger root under the smaller
        const int old = atomicMin(&label[b], a);
        if (old == b) return;
        b = old;                                            // somebody re-linked b meanwhile: retry from there
    }
}

// 13 "forward" neighbours = half of the 26-neighbourhood; every unordered pair of adjacent cells is visited once
__global__ void seg_merge_kernel(int *label, size_t V, int N)
{
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V; lin += (size_t)gridDim.x * blockDim.x) {
        if (label[lin] < 0) continue;
        int x, y, z;
        xyz_of(lin, N, x, y, z);
        const int xs[3] = {wrap_m(x, N), x, wrap_p(x, N)}, ys[3] = {wrap_m(y, N), y, wrap_p(y, N)};
        const int zp = wrap_p(z, N);
        for (int k = 0; k < 13; k++) {
            // k = 0..8: the nine cells of plane z+1; 9..11: row y+1 of plane z; 12: (x+1, y, z)
            const int a = k < 9 ? k % 3 : (k < 12 ? k - 9 : 2), b = k < 9 ? k / 3 : (k < 12 ? 2 : 1);
            const size_t nb = (size_t)xs[a] + (size_t)N * ((size_t)ys[b] + (size_t)N * (k < 9 ? zp : z));
            if (nb != lin && label[nb] >= 0) unite(label, (int)lin, (int)nb);
        }
    }
}

// size[root] counts HALF cells: a cell adds (pierced by p) + (pierced by q), i.e. 2 for an exact-overlap cell and 1 for a
// cell that belongs to the region by the one-cell tolerance only (reading R-21b: a region's cell count is
// (its p cells + its q cells) / 2, so a displaced pair of lines is as long as a coincident one)
__global__ void seg_flatten_count_kernel(int *label, int *size, const uint8_t *cells, size_t V)
{
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V; lin += (size_t)gridDim.x * blockDim.x) {
        if (label[lin] < 0) continue;
        const int r = find_root(label, (int)lin);
        label[lin] = r;             // roots keep label == index; concurrent readers see either a valid ancestor or the root
        atomicAdd(&size[r], (cells[lin] > 0) + (cells[V + lin] > 0));
    }
}

// Partials: [segments with n >= min_cells, sum (n - 1) over them, cells n in them, all segments, all pq cells,
// cells of the union mask | largest n], n = size / 2 (may be a half-integer for tolerant regions)
__global__ void __launch_bounds__(RED_BLOCK) seg_reduce_kernel(const int *label, const int *size, size_t V,
                                                               int min_cells, double *partials)
{
    double acc[7] = {0, 0, 0, 0, 0, 0, 0};
    for (size_t lin = (size_t)blockIdx.x * blockDim.x + threadIdx.x; lin < V; lin += (size_t)gridDim.x * blockDim.x) {
        const int lab = label[lin];
        if (lab >= 0) acc[5] += 1.0;                 // plain cell count of the mask (the reading R-21b replaced)
        if (lab != (int)lin) continue;               // roots only
        const int n2 = size[lin];
        const double n = 0.5 * (double)n2;
        acc[3] += 1.0;
        acc[4] += n;
        acc[6] = fmax(acc[6], n);
        if (n2 >= 2 * min_cells) {
            acc[0] += 1.0;
            acc[1] += n - 1.0;
            acc[2] += n;
        }
    }
    block_reduce_store<7>(acc, 6, partials);
}

}  // namespace

cudaError_t launch_segments(const uint8_t *cells, size_t V, int N, int tolerant, int min_cells, int *label, int *size,
                            double *partials, double *result, cudaStream_t st)
{
    const size_t need = (V + RED_BLOCK - 1) / RED_BLOCK;
    const int nb = (int)(need < (size_t)RED_MAX_BLOCKS ? need : (size_t)RED_MAX_BLOCKS);
    seg_init_kernel<<<nb, RED_BLOCK, 0, st>>>(cells, V, N, tolerant, label);
    cudaError_t e = cudaMemsetAsync(size, 0, V * sizeof(int), st);
    if (e != cudaSuccess) return e;
    seg_merge_kernel<<<nb, RED_BLOCK, 0, st>>>(label, V, N);
    seg_flatten_count_kernel<<<nb, RED_BLOCK, 0, st>>>(label, size, cells, V);
    seg_reduce_kernel<<<nb, RED_BLOCK, 0, st>>>(label, size, V, min_cells, partials);
    e = launch_fold(partials, nb, 7, 6, result, st);
    return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace u1u1
