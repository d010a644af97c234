// stage.cuh -- shared-memory staging of xy tiles (+ one-site halo) of a 10-word buffer, used by the fused step
// kernel (step_tiled.cu) and the fused diagnostics sweep (diag_fused.cu).
//
// A buffer (positions or momenta) holds three packs (common.cuh): A float4[V], B float4[V], C float2[V].  One ring
// slot holds one z plane of a TX x TY tile with its halo: A and B as float4[ROWS][COLS] (sites x0-1 .. x0+TX,
// y0-1 .. y0+TY), C as float2[ROWS][CCOLS] staged from x0-2 (a TMA box origin must be 16-byte aligned), so that
// site column c of the tile row r sits at A/B index r*COLS + c and at C index r*CCOLS + c + 1.
//   * tiles whose halo lies inside the lattice: three TMA box loads per plane (cp.async.bulk.tensor.3d, issued by
//     one thread, completion on an mbarrier);
//   * boundary / ragged tiles (a TMA box cannot wrap periodically): per-thread cp.async (LDGSTS) with the wrap
//     resolved once per tile in a per-thread plan.
#pragma once
#include <cuda.h>

#include "common.cuh"

namespace u1u1 {

constexpr int TX = 32;              // tile width  (one warp along x)
constexpr int TY = 8;               // tile height (one warp per row)
constexpr int NTHREADS = TX * TY;
constexpr int ROWS = TY + 2;        // + halo rows y0-1, y0+wy
constexpr int COLS = TX + 2;        // + halo columns x0-1, x0+wx
constexpr int NELEM = ROWS * COLS;  // staged sites per plane (340)
constexpr int CCOLS = COLS + 2;
// one ring slot: A float4[NELEM] | B float4[NELEM] | C float2[ROWS * CCOLS], each 128-byte aligned (TMA destination)
constexpr int OFF_B = 5504, OFF_C = 11008, SLOT_BYTES = 13952;
constexpr int POS_TX_BYTES = NELEM * 32 + ROWS * CCOLS * 8;    // bytes one plane's three halo boxes deliver
constexpr int NITEM = (3 * NELEM + NTHREADS - 1) / NTHREADS;   // cp.async copies per thread per plane (4)
static_assert(NELEM * 16 <= OFF_B && OFF_B + NELEM * 16 <= OFF_C && OFF_C + ROWS * CCOLS * 8 <= SLOT_BYTES, "slot layout");

// The two-steps-per-pass kernel (step_tb.cu) stages positions with a TWO-site halo: A, B float4[P2_ROWS][P2_COLS], C
// float2[P2_ROWS][P2_COLS], all from site (x0-2, y0-2) (an even x, so pack C is 16-byte aligned as it is).
#ifndef TB_TY
#define TB_TY 16         // 8: 352 threads, 2 CTAs/SM, 80 registers; 16: 640 threads, 1 CTA/SM, 96 registers (faster)
#endif
constexpr int TBY = TB_TY;          // tile height of the two-steps-per-pass kernel
constexpr int P2_COLS = TX + 4, P2_ROWS = TBY + 4, P2_ELEM = P2_ROWS * P2_COLS;      // 36 x 20 = 720 sites
constexpr int P2_OFF_B = P2_ELEM * 16, P2_OFF_C = 2 * P2_ELEM * 16, P2_SLOT_BYTES = P2_OFF_C + P2_ELEM * 8;   // 28 800 B
static_assert(P2_OFF_B % 128 == 0 && P2_OFF_C % 128 == 0 && P2_SLOT_BYTES % 128 == 0, "TMA destinations");

// Tensor maps of the three packs of one buffer (halo boxes COLS x ROWS, or plain TX x TY tile boxes).
struct alignas(64) PackMaps {
    CUtensorMap A, B, C;
};

// Tensor maps of one step launch: halo boxes of the position buffer being read, tile boxes of the momenta.
struct alignas(64) StepMaps {
    PackMaps pos, mom;
};
// Tensor maps of one diagnostics sweep: halo boxes of the current positions and of the momenta.
struct alignas(64) DiagMaps {
    PackMaps pos, mom;
};

// Tensor maps of one two-step launch: two-site-halo boxes of the positions being read, tile boxes of the momenta.
struct alignas(64) TbMaps {
    PackMaps pos, mom;
};

// host (tma_maps.cu): false if cuTensorMapEncodeTiled is unavailable or rejects the layout
bool encode_halo_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ, int rows = ROWS);
bool encode_tile_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ);
bool encode_halo2_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ);
bool encode_tb_tile_maps(PackMaps *m, const float *buf, size_t V, int N, int NZ);

#ifdef __CUDACC__
__device__ inline unsigned smem_u32(const void *p) { return (unsigned)__cvta_generic_to_shared(p); }

__device__ inline void cp_async16(unsigned sdst, const void *gsrc)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;\n" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ inline void cp_async8(unsigned sdst, const void *gsrc)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;\n" ::"r"(sdst), "l"(gsrc) : "memory");
}
__device__ inline unsigned long long policy_evict_first()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;\n" : "=l"(pol));
    return pol;
}
__device__ inline unsigned long long policy_evict_last()
{
    unsigned long long pol;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;\n" : "=l"(pol));
    return pol;
}
__device__ inline void cp_async_commit() { asm volatile("cp.async.commit_group;\n" ::: "memory"); }
template <int N_>
__device__ inline void cp_async_wait() { asm volatile("cp.async.wait_group %0;\n" ::"n"(N_) : "memory"); }

__device__ inline void mbar_init(unsigned bar, unsigned count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;\n" ::"r"(bar), "r"(count) : "memory");
}
__device__ inline void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;\n" ::: "memory"); }
__device__ inline void mbar_expect_tx(unsigned bar, unsigned bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;\n" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ inline void mbar_wait(unsigned bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "WAIT_LOOP:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
        "@p bra WAIT_DONE;\n"
        "bra WAIT_LOOP;\n"
        "WAIT_DONE:\n"
        "}\n" ::"r"(bar), "r"(parity)
        : "memory");
}
// TMA box load of a 3-d (W x + component, y, z) float tensor with an L2 eviction policy: evict-first for data
// read exactly once, evict-last for planes that the neighbouring tiles re-read as halo
__device__ inline void tma_load_3d_hint(unsigned sdst, const CUtensorMap *map, int c0, int c1, int c2, unsigned bar,
                                        unsigned long long pol)
{
    asm volatile(
        "cp.async.bulk.tensor.3d.shared::cluster.global.tile.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3, %4}], [%5], %6;\n" ::
            "r"(sdst), "l"(map), "r"(c0), "r"(c1), "r"(c2), "r"(bar), "l"(pol)
        : "memory");
}

__device__ inline int wrapi(int v, int N) { return v < 0 ? v + N : (v >= N ? v - N : v); }

// cp.async path: in-plane site index of each of this thread's copies of one halo plane (-1: none)
struct CpPlan {
    int lin[NITEM];
};

__device__ inline void make_cp_plan(CpPlan &p, int tid, int x0, int y0, int wx, int wy, int N)
{
#pragma unroll
    for (int q = 0; q < NITEM; q++) {
        const int item = tid + q * NTHREADS;
        const int pack = item / NELEM, e = item - pack * NELEM, r = e / COLS, c = e - r * COLS;
        const int y = wrapi(r == wy + 1 ? y0 + wy : y0 - 1 + r, N), x = wrapi(c == wx + 1 ? x0 + wx : x0 - 1 + c, N);
        p.lin[q] = (pack < 3 && r <= wy + 1 && c <= wx + 1) ? y * N + x : -1;
    }
}

// every thread; `buf` = byte address of a 10 V-float buffer, zp = z * N * N; the caller commits the group
__device__ inline void stage_plane_cp(const CpPlan &p, int tid, const char *buf, size_t V, size_t zp, unsigned slot)
{
#pragma unroll
    for (int q = 0; q < NITEM; q++) {
        if (p.lin[q] < 0) continue;
        const int item = tid + q * NTHREADS;
        const int pack = item < NELEM ? 0 : item < 2 * NELEM ? 1 : 2, e = item - pack * NELEM;
        const size_t site = zp + (size_t)p.lin[q];
        if (pack == 0) cp_async16(slot + e * 16, buf + site * 16);
        else if (pack == 1) cp_async16(slot + OFF_B + e * 16, buf + 16 * V + site * 16);
        else cp_async8(slot + OFF_C + (e + 2 * (e / COLS) + 1) * 8, buf + 32 * V + site * 8);
    }
}

// every thread: pack B only (float4 per site with halo, laid out as float4[ROWS][COLS] at `slot`) of a 10 V-float buffer
__device__ inline void stage_packB_cp(const CpPlan &p, int tid, const char *buf, size_t V, size_t zp, unsigned slot)
{
#pragma unroll
    for (int q = 0; q < NITEM; q++) {
        const int item = tid + q * NTHREADS;
        if (p.lin[q] < 0 || item < NELEM || item >= 2 * NELEM) continue;
        cp_async16(slot + (item - NELEM) * 16, buf + 16 * V + (zp + (size_t)p.lin[q]) * 16);
    }
}

// one thread: the three halo boxes of plane z of the tile at (x0, y0) into `slot`, completion on `bar`
__device__ inline void stage_plane_tma(const PackMaps &m, int x0, int y0, int z, unsigned slot, unsigned bar,
                                       unsigned long long pol)
{
    mbar_expect_tx(bar, POS_TX_BYTES);
    tma_load_3d_hint(slot, &m.A, 4 * (x0 - 1), y0 - 1, z, bar, pol);
    tma_load_3d_hint(slot + OFF_B, &m.B, 4 * (x0 - 1), y0 - 1, z, bar, pol);
    tma_load_3d_hint(slot + OFF_C, &m.C, 2 * (x0 - 2), y0 - 1, z, bar, pol);
}

// a tile can take the TMA path iff its halo (and the x0-2 column of pack C) lies inside the lattice
__device__ inline bool tile_is_interior(int x0, int y0, int N)
{
    return x0 >= 2 && x0 + TX + 2 <= N && y0 >= 1 && y0 + TY + 1 <= N;
}
#endif  // __CUDACC__

}  // namespace u1u1
