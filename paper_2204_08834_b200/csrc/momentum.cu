// momentum.cu -- the momentum-prediction kernel (kernels_momentum.cuh) and its launcher, a translation unit of its own
// (see momentum_launch.h for why).  Part of libflutas_b200.so.
#include "kernels_momentum.cuh"

namespace flutas {

template <int TY>
static cudaError_t launch_ty(const GridParams &g, const MomentumParams &mp, double dt, const double *u, const double *v, const double *w,
                             const double *phi, const double *kappa, const double *p, const double *po, const double *const *m_old,
                             double *const *m_new, double *rhs, double *us, double *vs, double *ws, cudaStream_t st) {
    using T = MomTile<TY>;
    const int kc = g.nz < 32 ? g.nz : 32;
    const dim3 grid(g.nx / T::TX, g.ny / T::TY, (g.nz + kc - 1) / kc);
    // the shared-memory attribute is a property of the kernel on a device: set once per device and tile size, not on every
    // step (a driver call on the host; a second thread that gets here at the same time sets it twice, which is harmless)
    static bool attr_set[64] = {};
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= 64 || !attr_set[dev]) {
        e = cudaFuncSetAttribute(momentum_rhs_kernel<TY>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)T::SMEM);
        if (e != cudaSuccess) return e;
        if (dev >= 0 && dev < 64) attr_set[dev] = true;
    }
    momentum_rhs_kernel<TY><<<grid, T::NT, T::SMEM, st>>>(g, mp, dt, kc, u, v, w, phi, kappa, p, po, m_old[0], m_old[1], m_old[2],
                                                          m_new[0], m_new[1], m_new[2], rhs, us, vs, ws);
    return cudaGetLastError();
}

cudaError_t launch_momentum_rhs(const GridParams &g, const MomentumParams &mp, double dt, bool ty16, const double *u, const double *v,
                                const double *w, const double *phi, const double *kappa, const double *p, const double *po,
                                const double *const *m_old, double *const *m_new, double *rhs, double *us, double *vs, double *ws,
                                cudaStream_t st) {
    // tiles of 32 x 16 cells (one CTA of 672 threads per SM); 32 x 8 when ny is not a multiple of 16
    if (ty16 && g.ny % 16 == 0) return launch_ty<16>(g, mp, dt, u, v, w, phi, kappa, p, po, m_old, m_new, rhs, us, vs, ws, st);
    return launch_ty<8>(g, mp, dt, u, v, w, phi, kappa, p, po, m_old, m_new, rhs, us, vs, ws, st);
}

}  // namespace flutas
