// kernels.h -- host-side launchers of the CUDA kernels (internal to libu1u1.so).
#pragma once
#include "common.cuh"

namespace u1u1 {

// step_ref.cu / step_tiled.cu: one fused kick+drift step (Eq. 17-26)
cudaError_t launch_step_ref(const Lattice &L, const StepCoef &k, cudaStream_t st, bool fp64);
struct StepMaps;
cudaError_t launch_step_tiled(const Lattice &L, const StepCoef &k, cudaStream_t st, int mode, const StepMaps *maps, int sms);
bool step_tiled_supports(int N);
bool step_tiled_uses_tma(int N);

// step_tb.cu: TWO fused steps per pass (80 B of HBM traffic per site-update); momenta are read from one buffer and
// written to another, positions as in the one-step kernel
struct TbLattice {
    const float *pos_in;   // positions at tau (read, two-site halo)
    float *pos_out;        // positions at tau + 2 dtau
    const float *mom_in;   // momenta before the two kicks (read, one-site halo)
    float *mom_out;        // momenta after them
    size_t V;
    int N;
};
struct TbMaps;
cudaError_t launch_step_tb(const TbLattice &L, StepCoef k1, StepCoef k2, cudaStream_t st, const TbMaps *maps, int sms);
bool step_tb_supports(int N);

// diag_fused.cu: every in-loop diagnostic from one read of the state.  Partial / result slots:
enum {
    FR_GAUSS = 0,    // sum g^2, rho^2, div^2 of the p sector, then of the q sector
    FR_SUMW = 6,     // sum |W^p|, sum |W^q|
    FR_NEAR = 8,     // plaquettes with a link angle within 1e-5 of the cut, p, q
    FR_CELLS = 10,   // cells pierced by p, by q, by both
    FR_DENS = 13,    // sum L, kin L, grad L, kin V, grad V, V, kin, grad, elec, mag, pot
    FUSED_NSUM = 24, // slots below are sums, slots from here on maxima
    FR_GMAX = 24,    // max |g_p|, max |g_q|
    FR_MAXW = 26,    // max |W|
    FR_MAXTH = 27,   // max |theta|
    FUSED_NRES = 28
};
struct FusedCoef {
    double inv_dx, rho1, rho2;   // Gauss: 1/dx, 2 e_p0^2 cG, 2 e_q0^2 cG
    float inv_dx2;               // 1/dx^2
    float el1, el2;              // 1/(2 e^2)
    float mg1, mg2;              // 1/(2 e^2 dx^4)
    float lam1q, lam2q, kappa;   // lambda/4, kappa_0
    float sig1sq, sig2sq;
    float c, inv_c;              // a^{2 beta} and its inverse
    int flags;                   // 2 = no TMA (cp.async staging everywhere)
    int nz_own;                  // 0: cubic lattice, periodic in z; else a z slab: own planes 1 .. nz_own of nz_own + 2, no z wrap
};
struct DiagMaps;
cudaError_t launch_diag_fused(const float *pos, const float *mom, size_t V, int N, FusedCoef k, uint8_t *cells, uint8_t *codes,
                              double *partials, int *nblocks, const DiagMaps *maps, int sms, cudaStream_t st);
cudaError_t launch_overlap_tol(const uint8_t *cells, size_t V, int N, double *partials, double *result, cudaStream_t st);
cudaError_t launch_fold(const double *partials, int nblocks, int nval, int n_sum, double *result, cudaStream_t st);

// diag.cu
cudaError_t launch_gauss(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                         double *partials, double *result, cudaStream_t st);
cudaError_t launch_decode_windings(const uint8_t *codes, size_t n, int8_t *w_out, uint8_t *near_out,
                                   cudaStream_t st);

// segments.cu: connected components of the pq cells (labels = root site index, -1 = not a pq cell)
// counts are in HALF cells: a cell of a region adds (pierced by p) + (pierced by q) to its root (reading R-21b)
cudaError_t launch_segments(const uint8_t *cells, size_t V, int N, int tolerant, int min_cells, int *label, int *size,
                            double *partials, double *result, cudaStream_t st);

// init.cu
cudaError_t launch_init_random_phase(float *pos, size_t n_own, size_t lin_off, size_t gidx_off, uint64_t seed, double eta1,
                                     double eta2, cudaStream_t st);
cudaError_t launch_init_smoothed(float *pos, double *tmp_a, double *tmp_b, size_t V, int N, uint64_t seed,
                                 double width, int trunc, double eta1, double eta2, cudaStream_t st);
cudaError_t launch_export_block(const float *pos, const float *mom, size_t V, int N, int x0, int y0, int z0,
                                int bx, int by, int bz, float *dst, cudaStream_t st);
cudaError_t launch_import_tiled(float *pos, float *mom, const float *canon, size_t V, int N, int n, cudaStream_t st);
cudaError_t launch_relayout(float *pos, float *mom, float *canon, size_t V, size_t n_own, size_t lin_off, int c0, int ncomp,
                            int to_canonical, cudaStream_t st);

}  // namespace u1u1
