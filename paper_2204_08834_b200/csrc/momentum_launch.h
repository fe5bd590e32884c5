// momentum_launch.h -- what flutas.cu needs to know of the momentum kernel, which is compiled as a translation unit of its
// own (momentum.cu): with it in the same module the compiler generates slower code for the transform kernels
// (measured: 116 instead of 128 registers, 7 % more instructions, x transforms 0.43 instead of 0.35 ms at 512^3).
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace flutas {

struct MomentumParams {
    double mu1, mu2, sigma, gx, gy, gz;
    double f1, f2;            // Adams-Bashforth: 1 + r/2, r/2
    int with_kappa, with_p;   // surface tension on / off; splitting terms on (fused with the projection) / off (u' = u**)
};

constexpr int kMomTileX = 32, kMomTileYMin = 8;   // nx must be a multiple of the first, ny of the second

// enqueue momentum_rhs_kernel on the whole grid (kernels_momentum.cuh); ty16: tiles of 32 x 16 cells when ny allows
cudaError_t launch_momentum_rhs(const GridParams &g, const MomentumParams &mp, double dt, bool ty16, const double *u, const double *v,
                                const double *w, const double *phi, const double *kappa, const double *p, const double *po,
                                const double *const *m_old, double *const *m_new, double *rhs, double *us, double *vs, double *ws,
                                cudaStream_t st);

}  // namespace flutas
