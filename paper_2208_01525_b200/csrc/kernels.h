// kernels.h -- host-side launchers of the CUDA kernels (internal to libu1u1.so).
#pragma once
#include "common.cuh"

namespace u1u1 {

// step_ref.cu / step_tiled.cu: one fused kick+drift step (Eq. 17-26)
cudaError_t launch_step_ref(const Lattice &L, const StepCoef &k, cudaStream_t st, bool fp64);
cudaError_t launch_step_tiled(const Lattice &L, const StepCoef &k, cudaStream_t st, int mode);
bool step_tiled_supports(int N);

// diag.cu
cudaError_t launch_gauss(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                         double *partials, double *result, cudaStream_t st);
cudaError_t launch_windings(const float *pos, size_t V, int N, uint8_t *codes, uint8_t *cells,
                            double *partials, double *result, cudaStream_t st);
cudaError_t launch_densities(const float *pos, const float *mom, size_t V, int N, const DiagCoef &k,
                             double *partials, double *result, cudaStream_t st);
cudaError_t launch_decode_windings(const uint8_t *codes, size_t n, int8_t *w_out, uint8_t *near_out,
                                   cudaStream_t st);

// segments.cu: connected components of the pq cells (labels = root site index, -1 = not a pq cell)
cudaError_t launch_segments(const uint8_t *cells, size_t V, int N, int tolerant, int min_cells, int *label, int *size,
                            double *partials, double *result, cudaStream_t st);

// init.cu
cudaError_t launch_init_random_phase(float *pos, size_t V, uint64_t seed, double eta1, double eta2,
                                     cudaStream_t st);
cudaError_t launch_init_smoothed(float *pos, float *tmp_a, float *tmp_b, size_t V, int N, uint64_t seed,
                                 double width, int trunc, double eta1, double eta2, cudaStream_t st);
cudaError_t launch_export_block(const float *pos, const float *mom, size_t V, int N, int x0, int y0, int z0,
                                int bx, int by, int bz, float *dst, cudaStream_t st);
cudaError_t launch_import_tiled(float *pos, float *mom, const float *canon, size_t V, int N, int n, cudaStream_t st);
cudaError_t launch_relayout(float *pos, float *mom, float *canon, size_t V, int c0, int ncomp, int to_canonical,
                            cudaStream_t st);

}  // namespace u1u1
