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
// Triply periodic.  Second form of the kernel: finite-volume bookkeeping in shared memory.  M(u) is a difference of
// fluxes that neighbouring faces share -- the normal fluxes (u^2, 2 mu du/dx) live at cell centres and belong to two
// faces each, the shear fluxes (u v, mu (du/dy + dv/dx)) live on edges and belong to FOUR (two faces of each of two
// components) -- so every flux is evaluated once, left in shared memory, and the faces take differences:
//
//   a block owns TX x TY cells and marches in z; its threads are the POSITIONS of a padded (TX + 3) x (TY + 3) plane
//   (two halo cells to the west / south, one to the east / north), one thread per position, the same position in every array: a neighbour is an
//   immediate offset (+-1, +-PX) from the thread's own index, no index arithmetic, no bank conflicts;
//   per plane k:  (0) the thread's own element of u, v, w, phi, kappa, p, p_old of plane k + 2 is requested from
//                     global memory into registers (consumed at the end of the step: one DRAM latency per plane);
//                 (A) fluxes: XX, YY at the cell centres of plane k, ZZ of plane k + 1, XY on the edges of plane k,
//                     XZ, YZ on the edges between planes k and k + 1 (convective and viscous part separately: the
//                     viscous one is divided by the face density);
//                 (B) faces: M(u^n), u** and u' on the east / north / top faces incl. the column west and the row south of
//                     the tile (the divergence needs them); M and u' to global memory, u' to shared memory;
//                 (C) rhs = rho0/dt div u'; the registers of (0) go into the slot plane k has just left.
//   XZ, YZ, ZZ and w' of the level below are carried from the previous step in the other of two slots.
// Against the first form (every face evaluated on its own from ~45 global loads): 2.1 x fewer instructions per cell.
#pragma once
#include "common.cuh"
#include "momentum_launch.h"

namespace flutas {

template <int TY_> struct MomTile {
    static constexpr int TX = 32, TY = TY_;
    static constexpr int PX = TX + 3, PY = TY + 3, NP = PX * PY;        // padded plane: i = -2 .. TX, j = -2 .. TY
    static constexpr int NT = (NP + 31) / 32 * 32;
    // shared-memory arrays of NP doubles: 6 input fields x 2 plane slots, 6 in-plane flux arrays, 6 x 2 carried flux
    // arrays, u', v', 2 x w'
    static constexpr int N_ARRAYS = 12 + 6 + 12 + 4;
    static constexpr size_t SMEM = (size_t)N_ARRAYS * NP * sizeof(double);
};

template <int TY_>
__global__ void __launch_bounds__(MomTile<TY_>::NT, TY_ == 8 ? 2 : 1)
momentum_rhs_kernel(GridParams g, MomentumParams mp, double dt, int kc, const double *__restrict__ u, const double *__restrict__ v,
                    const double *__restrict__ w, const double *__restrict__ phi, const double *__restrict__ kappa,
                    const double *__restrict__ p, const double *__restrict__ po, const double *__restrict__ mu_old,
                    const double *__restrict__ mv_old, const double *__restrict__ mw_old, double *__restrict__ mu_new,
                    double *__restrict__ mv_new, double *__restrict__ mw_new, double *__restrict__ rhs,
                    double *__restrict__ up, double *__restrict__ vp, double *__restrict__ wp) {
    using T = MomTile<TY_>;
    constexpr int PX = T::PX, NP = T::NP, TX = T::TX, TY = T::TY;
    extern __shared__ double sm[];
    // inputs, slot = plane & 1
    double *sU = sm, *sV = sU + 2 * NP, *sW = sV + 2 * NP, *sF = sW + 2 * NP, *sK = sF + 2 * NP, *sP = sK + 2 * NP;
    // fluxes of the plane (c = convective, t = viscous) ...
    double *XXc = sP + 2 * NP, *XXt = XXc + NP, *YYc = XXt + NP, *YYt = YYc + NP, *XYc = YYt + NP, *XYt = XYc + NP;
    // ... and those carried from level to level, slot = level & 1 (XZ, YZ: level k + 1/2 in slot k & 1; ZZ: plane k in slot k & 1)
    double *XZc = XYt + NP, *XZt = XZc + 2 * NP, *YZc = XZt + 2 * NP, *YZt = YZc + 2 * NP, *ZZc = YZt + 2 * NP, *ZZt = ZZc + 2 * NP;
    double *su = ZZt + 2 * NP, *sv = su + NP, *sw = sv + NP;           // u', v' of the plane; w' of level k + 1/2 in slot k & 1

    const int tid = threadIdx.x;
    const bool live = tid < NP;
    const int pos = live ? tid : 0;
    const int i = pos % PX - 2, j = pos / PX - 2;                       // this thread's position relative to the tile
    const int x0 = blockIdx.x * TX, j0 = blockIdx.y * TY;
    const int k0 = blockIdx.z * kc, k1 = min(k0 + kc, g.nz);
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    int gi = x0 + i, gj = j0 + j;
    gi += gi < 0 ? nx : (gi >= nx ? -nx : 0);
    gj += gj < 0 ? ny : (gj >= ny ? -ny : 0);
    const int goff = gj * nx + gi;                                      // wrapped offset inside a plane (nx ny <= 2^22)
    const long long plane = (long long)nx * ny;
    auto plane_of = [&](int k) { return k < 0 ? k + nz : (k >= nz ? k - nz : k); };

    const double hx = g.inv_dx, hy = g.inv_dy, hz = g.inv_dz;
    const double dmu = mp.mu1 - mp.mu2, drho = g.rho1 - g.rho2;
    auto mu_of = [&](double f) { return fma(dmu, f, mp.mu2); };
    const double c_div = g.rho0 / dt, c_split = dt / g.rho0, m2rho0 = -2.0 * g.rho0 * g.flux_one;
    const bool in_x = i >= 0 && i < TX, in_y = j >= 0 && j < TY;        // inside the tile along x / y
    const bool west1 = i >= -1 && i < TX, south1 = j >= -1 && j < TY;   // ... or one position before it

    // M(u^(n-1)) on this thread's three faces: requested one plane ahead as well (a face would otherwise wait for DRAM)
    double mo_u = 0.0, mo_v = 0.0, mo_w = 0.0, mn_u = 0.0, mn_v = 0.0, mn_w = 0.0;
    const bool face_u = west1 && in_y, face_v = in_x && south1, face_w = in_x && in_y;
    auto request_m = [&](int k) {
        const long long q = (long long)plane_of(k) * plane + goff;
        if (face_u) mn_u = __ldg(mu_old + q);
        if (face_v) mn_v = __ldg(mv_old + q);
        if (face_w) mn_w = __ldg(mw_old + q);
    };
    // ---- staging: every thread moves its own element of the seven fields
    double r_u, r_v, r_w, r_f, r_k = 0.0, r_p = 0.0, r_po = 0.0;
    auto request = [&](int k) {
        const long long q = (long long)plane_of(k) * plane + goff;
        r_u = __ldg(u + q); r_v = __ldg(v + q); r_w = __ldg(w + q); r_f = __ldg(phi + q);
        if (mp.with_kappa) r_k = __ldg(kappa + q);
        if (mp.with_p) { r_p = __ldg(p + q); r_po = __ldg(po + q); }
    };
    auto deposit = [&](int k) {
        const int o = (k & 1) * NP + pos;
        sU[o] = r_u; sV[o] = r_v; sW[o] = r_w; sF[o] = r_f; sK[o] = r_k;
        sP[o] = fma(g.c_pn, r_p, -(g.c_po * r_po));                     // p_hat
    };

    // ---- phase A for plane k (s0) and the level above it (s1 = plane k + 1)
    auto fluxes = [&](int k, bool in_plane) {
        const int s0 = (k & 1) * NP + pos, s1 = ((k + 1) & 1) * NP + pos;
        if (in_plane) {
            if (i >= -1 && i <= TX && in_y) {                           // XX at the centre of cell (i, j)
                const double um = sU[s0 - 1], ue = sU[s0], ub = 0.5 * (um + ue);
                XXc[pos] = ub * ub;
                XXt[pos] = 2.0 * mu_of(sF[s0]) * ((ue - um) * hx);
            }
            if (in_x && j >= -1 && j <= TY) {                           // YY
                const double vm = sV[s0 - PX], vn = sV[s0], vb = 0.5 * (vm + vn);
                YYc[pos] = vb * vb;
                YYt[pos] = 2.0 * mu_of(sF[s0]) * ((vn - vm) * hy);
            }
            if (west1 && south1) {                                      // XY on the edge (i + 1/2, j + 1/2)
                const double u0 = sU[s0], un = sU[s0 + PX], v0 = sV[s0], ve = sV[s0 + 1];
                const double m4 = 0.25 * (mu_of(sF[s0]) + mu_of(sF[s0 + 1]) + mu_of(sF[s0 + PX]) + mu_of(sF[s0 + PX + 1]));
                XYc[pos] = 0.5 * (u0 + un) * (0.5 * (v0 + ve));
                XYt[pos] = m4 * ((un - u0) * hy + (ve - v0) * hx);
            }
        }
        const int lv = (k & 1) * NP + pos, lz = ((k + 1) & 1) * NP + pos;
        if (in_x && in_y) {                                             // ZZ at the centre of cell (i, j, k + 1)
            const double wb_ = sW[s0], wt = sW[s1], wm = 0.5 * (wb_ + wt);
            ZZc[lz] = wm * wm;
            ZZt[lz] = 2.0 * mu_of(sF[s1]) * ((wt - wb_) * hz);
        }
        if (west1 && in_y) {                                            // XZ on the edge (i + 1/2, j, k + 1/2)
            const double u0 = sU[s0], ut = sU[s1], w0 = sW[s0], we = sW[s0 + 1];
            const double m4 = 0.25 * (mu_of(sF[s0]) + mu_of(sF[s0 + 1]) + mu_of(sF[s1]) + mu_of(sF[s1 + 1]));
            XZc[lv] = 0.5 * (u0 + ut) * (0.5 * (w0 + we));
            XZt[lv] = m4 * ((ut - u0) * hz + (we - w0) * hx);
        }
        if (in_x && south1) {                                           // YZ on the edge (i, j + 1/2, k + 1/2)
            const double v0 = sV[s0], vt = sV[s1], w0 = sW[s0], wn = sW[s0 + PX];
            const double m4 = 0.25 * (mu_of(sF[s0]) + mu_of(sF[s0 + PX]) + mu_of(sF[s1]) + mu_of(sF[s1 + PX]));
            YZc[lv] = 0.5 * (v0 + vt) * (0.5 * (w0 + wn));
            YZt[lv] = m4 * ((vt - v0) * hz + (wn - w0) * hy);
        }
    };

    // one face: a0 the velocity on it, dc / dtv the divergences of the convective / viscous fluxes, (s, sa) the two cells it
    // separates (s + sa the one ahead), hA the inverse spacing across it.  Returns M; us = u'
    auto face = [&](double a0, double dc, double dtv, int s, int sa, double hA, double grav, double m_old, double &us) {
        const double f0 = sF[s], fA = sF[s + sa];
        const double r2 = rcp_density(fma(drho, f0, g.rho2) + fma(drho, fA, g.rho2));     // 1 / (2 rho_f)
        const double inv_rf = r2 + r2;
        double src = grav;
        if (mp.with_kappa) src = fma(mp.sigma * (0.5 * (sK[s] + sK[s + sa])) * ((fA - f0) * hA), inv_rf, src);
        const double m = -dc + dtv * inv_rf;
        us = a0 + dt * (mp.f1 * m - mp.f2 * m_old + src);
        if (mp.with_p) {                                                // the splitting term of eq. (16)
            const double coef = fma(m2rho0, r2, g.flux_one);
            us = fma(c_split, coef * ((sP[s + sa] - sP[s]) * hA), us);
        }
        return m;
    };

    // ---- phase B: the faces of plane k (u, v) and of level k + 1/2 (w)
    auto faces = [&](int k, bool only_w) {
        const int s0 = (k & 1) * NP + pos, s1 = ((k + 1) & 1) * NP + pos;
        const int lv = (k & 1) * NP + pos, lp = ((k + 1) & 1) * NP + pos;      // this level / the one below (and ZZ of plane k + 1 / k)
        const long long q = (long long)k * plane + goff;
        if (!only_w && west1 && in_y) {                                 // east face of cell (i, j): A = x, B = y, C = z
            const double dc = (XXc[pos + 1] - XXc[pos]) * hx + (XYc[pos] - XYc[pos - PX]) * hy + (XZc[lv] - XZc[lp]) * hz;
            const double dv = (XXt[pos + 1] - XXt[pos]) * hx + (XYt[pos] - XYt[pos - PX]) * hy + (XZt[lv] - XZt[lp]) * hz;
            double us;
            const double m = face(sU[s0], dc, dv, s0, 1, hx, mp.gx, mo_u, us);
            su[pos] = us;
            if (i >= 0) { mu_new[q] = m; up[q] = us; }
        }
        if (!only_w && in_x && south1) {                                // north face: A = y, B = z, C = x
            const double dc = (YYc[pos + PX] - YYc[pos]) * hy + (YZc[lv] - YZc[lp]) * hz + (XYc[pos] - XYc[pos - 1]) * hx;
            const double dv = (YYt[pos + PX] - YYt[pos]) * hy + (YZt[lv] - YZt[lp]) * hz + (XYt[pos] - XYt[pos - 1]) * hx;
            double us;
            const double m = face(sV[s0], dc, dv, s0, PX, hy, mp.gy, mo_v, us);
            sv[pos] = us;
            if (j >= 0) { mv_new[q] = m; vp[q] = us; }
        }
        if (in_x && in_y) {                                             // top face: A = z, B = x, C = y
            const double dc = (ZZc[lp] - ZZc[lv]) * hz + (XZc[lv] - XZc[lv - 1]) * hx + (YZc[lv] - YZc[lv - PX]) * hy;
            const double dv = (ZZt[lp] - ZZt[lv]) * hz + (XZt[lv] - XZt[lv - 1]) * hx + (YZt[lv] - YZt[lv - PX]) * hy;
            double us;
            // the cell above is the same position in the other slot: s1 - s0
            const double m = face(sW[s0], dc, dv, s0, s1 - s0, hz, mp.gz, mo_w, us);
            sw[lv] = us;
            if (!only_w) { mw_new[q] = m; wp[q] = us; }
        }
    };

    // ---- prologue: planes k0 - 1 and k0; ZZ of plane k0 - 1 (it needs w of plane k0 - 2); the fluxes of level k0 - 1/2 and
    //      w' on it; then plane k0 + 1 takes the slot of plane k0 - 1
    if (live) { request(k0 - 1); deposit(k0 - 1); request(k0); deposit(k0); }
    __syncthreads();
    if (live) {
        if (in_x && in_y) {
            const int s = ((k0 - 1) & 1) * NP + pos;
            const double wb_ = __ldg(w + (long long)plane_of(k0 - 2) * plane + goff), wt = sW[s], wm = 0.5 * (wb_ + wt);
            ZZc[s] = wm * wm;
            ZZt[s] = 2.0 * mu_of(sF[s]) * ((wt - wb_) * hz);
        }
        fluxes(k0 - 1, false);
    }
    __syncthreads();
    if (live) {
        // M(u^(n-1)) of the plane below is not needed for w' there?  It is: u** contains it.
        const int s0 = ((k0 - 1) & 1) * NP + pos, s1 = (k0 & 1) * NP + pos;
        if (in_x && in_y) {
            const int lv = s0, lp = s1;
            const double dc = (ZZc[lp] - ZZc[lv]) * hz + (XZc[lv] - XZc[lv - 1]) * hx + (YZc[lv] - YZc[lv - PX]) * hy;
            const double dv = (ZZt[lp] - ZZt[lv]) * hz + (XZt[lv] - XZt[lv - 1]) * hx + (YZt[lv] - YZt[lv - PX]) * hy;
            double us;
            face(sW[s0], dc, dv, s0, s1 - s0, hz, mp.gz, __ldg(mw_old + (long long)plane_of(k0 - 1) * plane + goff), us);
            sw[lv] = us;
        }
        request(k0 + 1);
        request_m(k0);
    }
    __syncthreads();
    if (live) deposit(k0 + 1);
    __syncthreads();

    for (int k = k0; k < k1; ++k) {
        const bool more = k + 1 < k1;
        if (live) {
            mo_u = mn_u; mo_v = mn_v; mo_w = mn_w;
            if (more) { request(k + 2); request_m(k + 1); }
            fluxes(k, true);
        }
        __syncthreads();
        if (live) faces(k, false);
        __syncthreads();
        if (live) {
            if (in_x && in_y) {
                const int lv = (k & 1) * NP + pos, lp = ((k + 1) & 1) * NP + pos;
                rhs[(long long)k * plane + goff] = c_div * ((su[pos] - su[pos - 1]) * hx + (sv[pos] - sv[pos - PX]) * hy + (sw[lv] - sw[lp]) * hz);
            }
            if (more) deposit(k + 2);                                   // plane k + 2 into the slot plane k has left
        }
        __syncthreads();
    }
}

}  // namespace flutas
