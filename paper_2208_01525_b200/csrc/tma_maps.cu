// tma_maps.cu -- host-side encoding of the TMA tensor maps of stage.cuh (cuTensorMapEncodeTiled, reached through
// cudaGetDriverEntryPoint so that libu1u1.so links against the runtime only).
#include <mutex>

#include "stage.cuh"

namespace u1u1 {

namespace {

typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn()
{
    static std::once_flag once;
    static EncodeTiledFn fn = nullptr;
    std::call_once(once, [] {
        void *p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    });
    return fn;
}

// A pack of W floats per site at `base`: 3-d float tensor (W x + component, y, z), box (W bx, by, 1): x and the
// component form ONE contiguous innermost run, so a box row is a single bx*W*4-byte request.  The box origin
// must be 16-byte aligned, i.e. (W x) a multiple of 4 floats: any x for W = 4, even x for W = 2.
// (Measured dead ends: a 4-d (component, x, y, z) map makes TMA issue 16-byte requests, 25 % slower; 8-byte element
// types and unaligned origins raise `illegal instruction` on sm_100a.)
bool encode_pack(CUtensorMap *m, const float *base, int W, int N, int NZ, int bx, int by)
{
    EncodeTiledFn fn = encode_fn();
    if (!fn) return false;
    const cuuint64_t n = (cuuint64_t)N, w = (cuuint64_t)W;
    const cuuint64_t dims[3] = {w * n, n, (cuuint64_t)NZ}, strides[2] = {4 * w * n, 4 * w * n * n};
    const cuuint32_t box[3] = {(cuuint32_t)(W * bx), (cuuint32_t)by, 1}, es[3] = {1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, (void *)base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
              CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// NZ = planes in the buffer (N for the cubic lattice, nz_own + 2 for a z slab); V = N * N * NZ
// rows = box height (ROWS = the 8-row tiles + halo)
bool encode_halo_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ, int rows)
{
    return encode_pack(&m->A, buf, 4, N, NZ, COLS, rows) && encode_pack(&m->B, buf + 4 * V, 4, N, NZ, COLS, rows) &&
           encode_pack(&m->C, buf + 8 * V, 2, N, NZ, CCOLS, rows);
}

bool encode_halo2_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ)
{
    return encode_pack(&m->A, buf, 4, N, NZ, P2_COLS, P2_ROWS) && encode_pack(&m->B, buf + 4 * V, 4, N, NZ, P2_COLS, P2_ROWS) &&
           encode_pack(&m->C, buf + 8 * V, 2, N, NZ, P2_COLS, P2_ROWS);
}

bool encode_tb_tile_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ)
{
    return encode_pack(&m->A, buf, 4, N, NZ, TX, TBY) && encode_pack(&m->B, buf + 4 * V, 4, N, NZ, TX, TBY) &&
           encode_pack(&m->C, buf + 8 * V, 2, N, NZ, TX, TBY);
}

bool encode_tile_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ)
{
    return encode_pack(&m->A, buf, 4, N, NZ, TX, TY) && encode_pack(&m->B, buf + 4 * V, 4, N, NZ, TX, TY) &&
           encode_pack(&m->C, buf + 8 * V, 2, N, NZ, TX, TY);
}

}  // namespace u1u1
