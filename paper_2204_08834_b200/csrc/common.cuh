// common.cuh -- what every translation unit of libflutas_b200.so shares: the grid description and the fast reciprocal.
#pragma once
#include <cuda_runtime.h>

namespace flutas {

struct GridParams {
    int nx, ny, nz, wall;
    double inv_dx, inv_dy, inv_dz;
    double rho1, rho2, rho0;
    double c_pn, c_po;   // p_hat = c_pn p^n - c_po p^(n-1); (2, 1) for constant dt, (1 + r, r) in general
    double flux_one;     // 1, or 0 when rho1 == rho2: the splitting coefficient 1 - rho0/rho_f is then exactly 0
    int wall_x, wall_y;  // walls (u_n = 0, dp/dn = 0) at both ends of x / y: the last stored face is the wall face (passes through),
                         // the first wall face is not stored and carries 0 (as `wall` along z)
};

// ------------------------------------------------------------------------------------------------
// a1-a3: fused density + splitting right-hand side (eqs. 2, 16, 17).
// Reads u*, v*, w*, phi, p, p_old once; writes rhs and the half-corrected velocity u', v', w'.
// ------------------------------------------------------------------------------------------------
// Reciprocal of a normal, positive double: hardware seed (MUFU.RCP64H, ~2^-23) + two Newton steps
// (relative error <= ~1 ulp, branch-free, 5 instructions instead of the ~30 of an IEEE division).
// Used only where the operand is a face density (rho > 0, far from the denormal / overflow ranges).
__device__ __forceinline__ double rcp_density(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}

}  // namespace flutas
