// vof_launch.h -- what vof_noalloc.cu needs from flutas.cu: the kernels of the volume-of-fluid step are defined in headers that
// only one translation unit can include (they hold non-template kernels), so the entry point without allocations reaches
// them through this launcher and reports its errors through the library's one error slot.
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"

namespace flutas {

// Enqueue the seven kernels of one MTHINC step (kernels_vof.cuh; Algorithm 2) on `st`.  flux, px, py, pz:
// four caller-given device fields of nx*ny*nz doubles, all fully written before they are read.  Returns cudaGetLastError().
cudaError_t launch_vof_step(const GridParams &g, double beta, double dt, const double *phi, const double *u, const double *v,
                            const double *w, double *flux, double *px, double *py, double *pz, double *phi_out, cudaStream_t st);

// record a failure in the calling thread's flutas_last_error() / flutas_last_error_code(); returns code
int report_error(int code, const char *msg);

}  // namespace flutas
