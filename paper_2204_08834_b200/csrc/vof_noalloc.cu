// vof_noalloc.cu -- flutas_vof_step_noalloc: the MTHINC volume-of-fluid step of flutas_vof_step (kernels_vof.cuh; PAPER.md:104-132,
// eqs. 8-12, Appendix A) for callers that are not allowed to allocate device memory.  Part of libflutas_b200.so.
//
// Who that is: code that runs where a cudaMalloc is either forbidden or too disruptive to issue -- a solver embedded in a
// host application whose memory pool has already claimed the whole GPU (a cudaMalloc there simply fails), a plug-in that a
// real-time or in-situ pipeline calls between two of its own kernels (cudaMalloc synchronises the device and stalls every
// stream of the host application), or a component whose rules of use say "no allocation after start-up".  The ordinary
// entry point does not suit them: flutas_vof_step needs a plan, creating a plan allocates its tables, and the step borrows
// four fields of the plan's workspace.
//
// What is different here: there is no plan, and the four intermediate fields of the step (the face fluxes of the current
// sweep and phi after the x, y and z sweeps) live in ONE array of static storage in this file, g_vof_scratch below.  It is
// part of the library's device image: every GPU that loads this part of the library holds the array (64 MiB) from then
// until the process exits, however small the grids it is used for.  That is why it has a fixed, modest size, and the size
// fixes the largest grid the entry point can take (FLUTAS_VOF_NOALLOC_MAX_CELLS cells, e.g. 128^3); anything larger is
// refused, never truncated.
//
// The kernels and their launch sequence are those of flutas_vof_step (the very same device code, reached through
// launch_vof_step in flutas.cu, and the same GridParams arithmetic); flutas_vof_step itself is untouched.
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <mutex>

#include "flutas.h"
#include "vof_launch.h"

using namespace flutas;

static constexpr size_t kMaxCells = FLUTAS_VOF_NOALLOC_MAX_CELLS;

// The scratch: 4 fields of kMaxCells doubles, back to back.  In HOST code this name is only a handle for the runtime, not a
// device address -- a kernel that were handed `g_vof_scratch` from the host side would fault, or quietly use some host
// memory where the GPU can reach it.  Host code therefore asks the runtime for the device address (scratch_on_current_device).
static __device__ __align__(256) double g_vof_scratch[4 * kMaxCells];

// device address of g_vof_scratch per device ordinal (every device has its own copy of the array); nullptr = not asked yet
static constexpr int kMaxDevices = 64;
static double *g_scratch_addr[kMaxDevices];
static std::mutex g_scratch_mu;

static int failf(int code, const char *fmt, ...) {
    char msg[384];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(msg, sizeof(msg), fmt, ap);
    va_end(ap);
    return report_error(code, msg);
}

// Set-up, once per device, with that device current: the address under which kernels on THIS device see g_vof_scratch.
// The first request on a device makes the runtime load this file's device image there, which is when the array gets its
// place in that GPU's memory; later calls only read the cached pointer.
static int scratch_on_current_device(double **out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return failf(FLUTAS_ERR_CUDA, "cudaGetDevice: %s", cudaGetErrorString(e));
    if (dev < 0 || dev >= kMaxDevices) return failf(FLUTAS_ERR_CUDA, "device ordinal %d is beyond the %d this entry point keeps track of", dev, kMaxDevices);
    std::lock_guard<std::mutex> lock(g_scratch_mu);
    if (!g_scratch_addr[dev]) {
        void *ptr = nullptr;
        e = cudaGetSymbolAddress(&ptr, g_vof_scratch);
        if (e != cudaSuccess || !ptr)
            return failf(FLUTAS_ERR_CUDA, "cudaGetSymbolAddress(g_vof_scratch) on device %d: %s", dev, cudaGetErrorString(e));
        g_scratch_addr[dev] = (double *)ptr;
    }
    *out = g_scratch_addr[dev];
    return FLUTAS_OK;
}

extern "C" size_t flutas_vof_step_noalloc_max_cells(void) { return kMaxCells; }

extern "C" int flutas_vof_step_noalloc(int nx, int ny, int nz, double lx, double ly, double lz, const double *phi, const double *u,
                                       const double *v, const double *w, double *phi_out, double beta, double dt, void *stream) {
    if (nx < 3 || ny < 3 || nz < 3) return failf(FLUTAS_ERR_INVALID_ARG, "nx, ny, nz must be at least 3");
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0) || !std::isfinite(lx) || !std::isfinite(ly) || !std::isfinite(lz))
        return failf(FLUTAS_ERR_INVALID_ARG, "lx, ly, lz must be positive and finite");
    if (!(beta > 0.0) || !std::isfinite(beta) || !(dt > 0.0) || !std::isfinite(dt))
        return failf(FLUTAS_ERR_INVALID_ARG, "beta and dt must be positive and finite");
    const long long npts = (long long)nx * ny * nz;
    if (npts > (long long)kMaxCells)
        return failf(FLUTAS_ERR_UNSUPPORTED_SIZE,
                     "flutas_vof_step_noalloc: %lld cells exceed the %lld its static scratch array is sized for "
                     "(FLUTAS_VOF_NOALLOC_MAX_CELLS); use flutas_vof_step with a plan for larger grids", npts, (long long)kMaxCells);
    const void *ptrs[5] = {phi, u, v, w, phi_out};
    const int n = phi_out == phi ? 4 : 5;               // phi_out may be phi itself, nothing else
    const size_t fb = sizeof(double) * (size_t)npts;
    for (int a = 0; a < n; ++a) {
        if (!ptrs[a]) return failf(FLUTAS_ERR_INVALID_ARG, "NULL field pointer (argument %d)", a);
        if (((size_t)ptrs[a]) & 15) return failf(FLUTAS_ERR_ALIAS, "field pointer %d is not 16-byte aligned", a);
    }
    for (int a = 0; a < n; ++a)
        for (int b = a + 1; b < n; ++b) {
            const char *x = (const char *)ptrs[a], *y = (const char *)ptrs[b];
            if (x < y + fb && y < x + fb) return failf(FLUTAS_ERR_ALIAS, "field arguments %d and %d overlap", a, b);
        }
    double *scratch = nullptr;
    if (int rc = scratch_on_current_device(&scratch)) return rc;

    // the grid exactly as flutas_plan_create describes it to the kernels (the VoF kernels read the sizes and spacings only)
    GridParams g{};
    g.nx = nx; g.ny = ny; g.nz = nz;
    g.inv_dx = 1.0 / (lx / nx); g.inv_dy = 1.0 / (ly / ny); g.inv_dz = 1.0 / (lz / nz);
    // Fields packed for THIS grid (npts, not kMaxCells, apart): a small grid touches the first 4 npts doubles only.  Nothing
    // has to be cleared although the array still holds whatever the previous call left: each sweep's flux kernel writes every
    // face exactly once and each update kernel every cell, before the kernel after it reads them.
    double *flux = scratch, *px = scratch + npts, *py = scratch + 2 * npts, *pz = scratch + 3 * npts;
    const cudaError_t e = launch_vof_step(g, beta, dt, phi, u, v, w, flux, px, py, pz, phi_out, (cudaStream_t)stream);
    if (e != cudaSuccess) return failf(FLUTAS_ERR_CUDA, "launch of vof_step_noalloc failed: %s", cudaGetErrorString(e));
    return FLUTAS_OK;
}
