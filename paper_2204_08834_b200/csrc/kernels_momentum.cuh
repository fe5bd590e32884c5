// kernels_momentum.cuh -- SURVEY.md sec. 8(f) NEXT-5: the momentum prediction of eq. (15) (the
// operator of eq. (5)) FUSED with rows a1-a3 of the projection step, so that the provisional velocity never
// travels through HBM between the two:
//
//     M(u)  = - div(u u) + (1/rho_f) div[ mu (grad u + grad u^T) ]            central differences, staggered grid
//     u**   = u^n + dt [ (1 + r/2) M(u^n) - (r/2) M(u^(n-1)) + g + sigma kappa grad(phi) / rho_f ]          eq. (15)
//     u'    = u** + (dt / rho0) (1 - rho0/rho_f) grad p_hat                    (what splitting_rhs_kernel* call u')
//     rhs   = (rho0 / dt) div u'                                               = rho0/dt div u** + div[(1 - rho0/rho_f) grad p_hat]
//
// in : u^n, v^n, w^n, phi, kappa (optional), p^n, p^(n-1), M(u^(n-1))          10 (9) fields read
// out: M(u^n) (separate arrays: the caller swaps the two sets), u', v', w', rhs  7 fields written   = 136 (128) B / point
// against  momentum kernel (7 r + 6 w) + splitting_rhs (6 r + 4 w) = 184 B / point  when the two are separate.
//
// Triply periodic.  A block owns a tile of 32 x 8 cells and marches in z.  Per plane it evaluates the face values u' on
// 33 x 8 east faces (its own and the column to the west), v' on 32 x 9 north faces (its own and the row to the south)
// and w' on its 32 x 8 top faces as three lists of work items spread over 32 x 9 = 288 threads (one round per list: the
// halo costs a ninth warp instead of a second, almost empty round in every warp), leaves them in shared memory, and
// then the first 256 threads take the divergence of their cells; w' of the plane below stays in shared memory from the previous
// step.  Operands come through L1 / L2 (read-only path): this is the first, plain form of the kernel.
#pragma once
#include "kernels.cuh"

namespace flutas {

struct MomentumParams {
    double mu1, mu2, sigma, gx, gy, gz;
    double f1, f2;            // Adams-Bashforth: 1 + r/2, r/2
    int with_kappa, with_p;   // surface tension on / off; splitting terms on (fused with the projection) / off (u' = u**)
};

struct MomTile {
    static constexpr int TX = 32, TY = 8, NT = TX * (TY + 1);   // one more row of threads than cells: every item list fits in ONE round
};

// everything one face evaluation needs to find its neighbours: wrapped indices around (i, j, k)
struct Nbr {
    long long c;                         // linear index of (i, j, k)
    long long xm, xp, xpp, ym, yp, ypp, zm, zp, zpp;   // offsets to add to c for i-1, i+1, i+2, ... (periodic wrap resolved)
};
__device__ __forceinline__ Nbr neighbours(const GridParams &g, int i, int j, int k) {
    Nbr n;
    const long long sx = 1, sy = g.nx, sz = (long long)g.nx * g.ny;
    n.c = i + sy * j + sz * k;
    n.xm = (i == 0 ? g.nx - 1 : -1) * sx;
    n.xp = (i == g.nx - 1 ? -(g.nx - 1) : 1) * sx;
    n.xpp = (i >= g.nx - 2 ? 2 - g.nx : 2) * sx;
    n.ym = (j == 0 ? g.ny - 1 : -1) * sy;
    n.yp = (j == g.ny - 1 ? -(g.ny - 1) : 1) * sy;
    n.ypp = (j >= g.ny - 2 ? 2 - g.ny : 2) * sy;
    n.zm = (k == 0 ? g.nz - 1 : -1) * sz;
    n.zp = (k == g.nz - 1 ? -(g.nz - 1) : 1) * sz;
    n.zpp = (k >= g.nz - 2 ? 2 - g.nz : 2) * sz;
    return n;
}

struct FaceOut { double m, up; };       // M(u^n) on the face and u'

// One velocity component on its own face.  The three components are the same stencil with the axes rotated: `a` is the
// component being advanced (along axis A), b and c the other two (axes B, C); oA / oB / oC give the index offsets of one
// step along each axis (p = +1, pp = +2, m = -1), hA, hB, hC the inverse spacings.
struct AxisOff { long long m, p, pp; };

__device__ __forceinline__ FaceOut
face_component(const double *__restrict__ a, const double *__restrict__ b, const double *__restrict__ c,
               const double *__restrict__ phi, const double *__restrict__ kappa, const double *__restrict__ p,
               const double *__restrict__ po, const double *__restrict__ mold, long long q, AxisOff oA, AxisOff oB, AxisOff oC,
               double hA, double hB, double hC, double grav, const GridParams &g, const MomentumParams &mp, double dt) {
    auto L = [](const double *f, long long idx) { return __ldg(f + idx); };
    // the component itself: centre and its six neighbours
    const double a0 = L(a, q), aAm = L(a, q + oA.m), aAp = L(a, q + oA.p), aBm = L(a, q + oB.m), aBp = L(a, q + oB.p),
                 aCm = L(a, q + oC.m), aCp = L(a, q + oC.p);
    // the transporting components on the four edges around the face (b lives on B faces, c on C faces)
    const double b0 = L(b, q), bA = L(b, q + oA.p), bm = L(b, q + oB.m), bmA = L(b, q + oB.m + oA.p);
    const double c0 = L(c, q), cA = L(c, q + oA.p), cm = L(c, q + oC.m), cmA = L(c, q + oC.m + oA.p);
    // viscosity at the two cell centres of the normal stress and (four-cell means) on the four edges of the shear stresses
    const double dmu = mp.mu1 - mp.mu2;
    auto mu_of = [&](double f) { return fma(dmu, f, mp.mu2); };
    const double f0 = L(phi, q), fA = L(phi, q + oA.p);
    const double fBp = L(phi, q + oB.p), fABp = L(phi, q + oA.p + oB.p), fBm = L(phi, q + oB.m), fABm = L(phi, q + oA.p + oB.m);
    const double fCp = L(phi, q + oC.p), fACp = L(phi, q + oA.p + oC.p), fCm = L(phi, q + oC.m), fACm = L(phi, q + oA.p + oC.m);
    const double mu0 = mu_of(f0), muA = mu_of(fA);
    const double mu_Bp = 0.25 * (mu0 + muA + mu_of(fBp) + mu_of(fABp)), mu_Bm = 0.25 * (mu_of(fBm) + mu_of(fABm) + mu0 + muA);
    const double mu_Cp = 0.25 * (mu0 + muA + mu_of(fCp) + mu_of(fACp)), mu_Cm = 0.25 * (mu_of(fCm) + mu_of(fACm) + mu0 + muA);

    // convection, divergence form with two-point means
    const double aa_p = 0.5 * (a0 + aAp), aa_m = 0.5 * (aAm + a0);
    const double ab_p = 0.5 * (a0 + aBp) * (0.5 * (b0 + bA)), ab_m = 0.5 * (aBm + a0) * (0.5 * (bm + bmA));
    const double ac_p = 0.5 * (a0 + aCp) * (0.5 * (c0 + cA)), ac_m = 0.5 * (aCm + a0) * (0.5 * (cm + cmA));
    const double conv = -((aa_p * aa_p - aa_m * aa_m) * hA + (ab_p - ab_m) * hB + (ac_p - ac_m) * hC);
    // stresses
    const double tAA_p = 2.0 * muA * ((aAp - a0) * hA), tAA_m = 2.0 * mu0 * ((a0 - aAm) * hA);
    const double tAB_p = mu_Bp * ((aBp - a0) * hB + (bA - b0) * hA), tAB_m = mu_Bm * ((a0 - aBm) * hB + (bmA - bm) * hA);
    const double tAC_p = mu_Cp * ((aCp - a0) * hC + (cA - c0) * hA), tAC_m = mu_Cm * ((a0 - aCm) * hC + (cmA - cm) * hA);
    const double drho = g.rho1 - g.rho2;
    const double rsum = fma(drho, f0, g.rho2) + fma(drho, fA, g.rho2);      // 2 rho_f
    const double r2 = rcp_density(rsum);                                     // 1 / (2 rho_f)
    const double inv_rf = r2 + r2;
    const double diff = ((tAA_p - tAA_m) * hA + (tAB_p - tAB_m) * hB + (tAC_p - tAC_m) * hC) * inv_rf;
    double src = grav;
    if (mp.with_kappa) src = fma(mp.sigma * (0.5 * (L(kappa, q) + L(kappa, q + oA.p))) * ((fA - f0) * hA), inv_rf, src);
    FaceOut o;
    o.m = conv + diff;
    double us = a0 + dt * (mp.f1 * o.m - mp.f2 * L(mold, q) + src);
    if (mp.with_p) {   // the splitting term of eq. (16), as flux_coef / c_up in kernels.cuh
        const double ph0 = fma(g.c_pn, L(p, q), -(g.c_po * L(po, q))), phA = fma(g.c_pn, L(p, q + oA.p), -(g.c_po * L(po, q + oA.p)));
        const double coef = fma(-2.0 * g.rho0 * g.flux_one, r2, g.flux_one);
        us = fma(dt / g.rho0, coef * ((phA - ph0) * hA), us);
    }
    o.up = us;
    return o;
}

__global__ void __launch_bounds__(MomTile::NT, 3)
momentum_rhs_kernel(GridParams g, MomentumParams mp, double dt, int kc, const double *__restrict__ u, const double *__restrict__ v,
                    const double *__restrict__ w, const double *__restrict__ phi, const double *__restrict__ kappa,
                    const double *__restrict__ p, const double *__restrict__ po, const double *__restrict__ mu_old,
                    const double *__restrict__ mv_old, const double *__restrict__ mw_old, double *__restrict__ mu_new,
                    double *__restrict__ mv_new, double *__restrict__ mw_new, double *__restrict__ rhs,
                    double *__restrict__ up, double *__restrict__ vp, double *__restrict__ wp) {
    using T = MomTile;
    __shared__ double su[T::TY][T::TX + 1], sv[T::TY + 1][T::TX], sw[2][T::TY][T::TX];
    const int tid = threadIdx.y * T::TX + threadIdx.x;
    const int x0 = blockIdx.x * T::TX, j0 = blockIdx.y * T::TY;
    const int k0 = blockIdx.z * kc, k1 = min(k0 + kc, g.nz);
    const double c_div = g.rho0 / dt;

    auto do_u = [&](int item, int k) {            // item in [0, 33 * 8): column -1 .. 31, row 0 .. 7
        const int jj = item / (T::TX + 1), ii = item % (T::TX + 1) - 1;
        const int i = ii < 0 ? (x0 == 0 ? g.nx - 1 : x0 - 1) : x0 + ii, j = j0 + jj;
        const Nbr n = neighbours(g, i, j, k);
        const FaceOut o = face_component(u, v, w, phi, kappa, p, po, mu_old, n.c, AxisOff{n.xm, n.xp, n.xpp}, AxisOff{n.ym, n.yp, n.ypp},
                                         AxisOff{n.zm, n.zp, n.zpp}, g.inv_dx, g.inv_dy, g.inv_dz, mp.gx, g, mp, dt);
        su[jj][ii + 1] = o.up;
        if (ii >= 0) { mu_new[n.c] = o.m; up[n.c] = o.up; }
    };
    auto do_v = [&](int item, int k) {            // item in [0, 32 * 9): row -1 .. 7
        const int jj = item / T::TX - 1, ii = item % T::TX;
        const int i = x0 + ii, j = jj < 0 ? (j0 == 0 ? g.ny - 1 : j0 - 1) : j0 + jj;
        const Nbr n = neighbours(g, i, j, k);
        const FaceOut o = face_component(v, w, u, phi, kappa, p, po, mv_old, n.c, AxisOff{n.ym, n.yp, n.ypp}, AxisOff{n.zm, n.zp, n.zpp},
                                         AxisOff{n.xm, n.xp, n.xpp}, g.inv_dy, g.inv_dz, g.inv_dx, mp.gy, g, mp, dt);
        sv[jj + 1][ii] = o.up;
        if (jj >= 0) { mv_new[n.c] = o.m; vp[n.c] = o.up; }
    };
    auto do_w = [&](int k, int slot, bool store) {
        if (threadIdx.y >= T::TY) return;
        const int kk = k < 0 ? g.nz - 1 : k;
        const Nbr n = neighbours(g, x0 + threadIdx.x, j0 + threadIdx.y, kk);
        const FaceOut o = face_component(w, u, v, phi, kappa, p, po, mw_old, n.c, AxisOff{n.zm, n.zp, n.zpp}, AxisOff{n.xm, n.xp, n.xpp},
                                         AxisOff{n.ym, n.yp, n.ypp}, g.inv_dz, g.inv_dx, g.inv_dy, mp.gz, g, mp, dt);
        sw[slot][threadIdx.y][threadIdx.x] = o.up;
        if (store) { mw_new[n.c] = o.m; wp[n.c] = o.up; }
    };

    // M(u^(n-1)) and M(u^n) are separate arrays: the halo items (west column, south row, the plane below the chunk) read old
    // values on faces whose new value another block writes.
    do_w(k0 - 1, 0, false);                       // top faces of the plane below the chunk
    int cur = 1;
    for (int k = k0; k < k1; ++k, cur ^= 1) {
        if (tid < (T::TX + 1) * T::TY) do_u(tid, k);
        do_v(tid, k);                              // 32 x 9 items = all threads
        do_w(k, cur, true);
        __syncthreads();
        const int tx = threadIdx.x, ty = threadIdx.y;
        if (ty < T::TY) {
            const long long q = (x0 + tx) + (long long)g.nx * ((j0 + ty) + (long long)g.ny * k);
            rhs[q] = c_div * ((su[ty][tx + 1] - su[ty][tx]) * g.inv_dx + (sv[ty + 1][tx] - sv[ty][tx]) * g.inv_dy +
                              (sw[cur][ty][tx] - sw[cur ^ 1][ty][tx]) * g.inv_dz);
        }
        __syncthreads();
    }
}

}  // namespace flutas
