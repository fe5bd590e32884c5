// kernels.cuh -- the device kernels of the projection step (sm_100a, fp64).
//
//   splitting_rhs_kernel   a1-a3  density from colour, p_hat, splitting RHS; also stores the
//                                 half-corrected velocity u' = u* - dt (1/rho_f - 1/rho0) grad p_hat
//   fft_x_r2c_kernel       a4     real-to-complex transform along x (8 contiguous lines per CTA)
//   fft_strided_kernel     a5/a7  complex transform along y (tile = C columns of kx x all j)
//                          a6p    and, in SOLVE mode, forward-z / divide by eigenvalues / inverse-z
//   thomas_kernel          a6w    tridiagonal solve along z per (kx,ky), one thread per column
//   thomas_singular_kernel a6w    the (0,0) column: pin the last unknown, remove the mean
//   fft_x_c2r_kernel       a8     complex-to-real transform along x, normalisation, writes p^(n+1)
//   correction_kernel      a9     u = u' - dt/rho0 grad p^(n+1)
//
// Row labels are those of SURVEY.md sec. 8(a); the paper passages are cited in include/flutas.h.
#pragma once
#include <cuda_runtime.h>

#include "fft_core.cuh"

namespace flutas {

// Where the x transforms find the rows of the half-spectrum: row (j, k) starts at k * plane + j * pitch (a plane holds
// ny rows + padding); a launch covers lines line0, line0 + 1, ... of the real field (line = j + ny k).
struct SpecRows {
    int ny;
    long long plane, line0;
};
__device__ __forceinline__ long long spec_row_offset(const SpecRows &r, long long line, int pitch) {
    const long long g = r.line0 + line;
    return (g / r.ny) * r.plane + (g % r.ny) * pitch;
}

struct GridParams {
    int nx, ny, nz, wall;
    double inv_dx, inv_dy, inv_dz;
    double rho1, rho2, rho0;
    double c_pn, c_po;   // p_hat = c_pn p^n - c_po p^(n-1); (2, 1) for constant dt, (1 + r, r) in general
};

// ------------------------------------------------------------------------------------------------
// a1-a3: fused density + splitting right-hand side (eqs. 2, 16, 17).
// Reads u*, v*, w*, phi, p, p_old once; writes rhs and the half-corrected velocity u', v', w'.
//
// 2.5-D register-marching stencil: a block is (bx threads along x, 2 points each) x (ty rows of j); each
// thread marches over `kc` planes in z carrying, in registers, the centre and top values of rho_c and p_hat,
// the bottom-face flux (= the previous plane's top-face flux) and w below.  x neighbours come from warp
// shuffles (edge lanes load them), y neighbours from L1/L2 (the rows were loaded one iteration earlier by
// the neighbouring threads).  Per point: 4 reciprocals, no integer division, 32-bit index arithmetic.
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

struct Flux { double f, r; };   // f = (1 - rho0/rho_f) * g,  r = 1/rho_f
__device__ __forceinline__ Flux face_flux(double rc_a, double rc_b, double g, double rho0) {
    Flux o;
    o.r = rcp_density(0.5 * (rc_a + rc_b));
    o.f = (1.0 - rho0 * o.r) * g;
    return o;
}

__global__ void __launch_bounds__(256, 2)
splitting_rhs_kernel(GridParams g, double dt, int kc, const double *__restrict__ u, const double *__restrict__ v,
                     const double *__restrict__ w, const double *__restrict__ phi,
                     const double *__restrict__ p, const double *__restrict__ po,
                     double *__restrict__ rhs, double *__restrict__ up, double *__restrict__ vp,
                     double *__restrict__ wp) {
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int i0 = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(k0 + kc, nz);
    const int jn = (j + 1 == ny) ? 0 : j + 1, js = (j == 0) ? ny - 1 : j - 1;
    const int iw = (i0 == 0) ? nx - 1 : i0 - 1, ie = (i0 + 2 == nx) ? 0 : i0 + 2;
    // shuffle neighbourhood: a "row" of lanes is min(32, blockDim.x) wide
    const int lane = (threadIdx.x + threadIdx.y * blockDim.x) & 31;
    const int rw = blockDim.x < 32 ? blockDim.x : 32;
    const bool edge_l = (lane % rw) == 0, edge_r = (lane % rw) == rw - 1;
    const long long plane = (long long)nx * ny;
    const long long col = (long long)j * nx + i0, col_n = (long long)jn * nx + i0, col_s = (long long)js * nx + i0;
    const long long row_j = (long long)j * nx;
    const double rho1 = g.rho1, rho2 = g.rho2, rho0 = g.rho0, inv_rho0 = 1.0 / g.rho0;
    const double c_div = g.rho0 / dt;

    auto ld2 = [](const double *f, long long q) { return *reinterpret_cast<const double2 *>(f + q); };
    auto rho_of = [&](double f) { return rho1 * f + rho2 * (1.0 - f); };
    auto rho2_of = [&](double2 f) { return make_double2(rho_of(f.x), rho_of(f.y)); };
    const double c_pn = g.c_pn, c_po = g.c_po;
    auto phat2 = [&](double2 a, double2 b) { return make_double2(fma(c_pn, a.x, -(c_po * b.x)), fma(c_pn, a.y, -(c_po * b.y))); };

    // prologue: centre plane k0, bottom flux and w below
    long long qk = (long long)k0 * plane;
    double2 rc_c = rho2_of(ld2(phi, qk + col)), ph_c = phat2(ld2(p, qk + col), ld2(po, qk + col));
    double2 fb = make_double2(0.0, 0.0), wb = make_double2(0.0, 0.0);
    if (!(g.wall && k0 == 0)) {
        const long long qb = (long long)((k0 == 0) ? nz - 1 : k0 - 1) * plane + col;
        const double2 rc_b = rho2_of(ld2(phi, qb)), ph_b = phat2(ld2(p, qb), ld2(po, qb));
        fb.x = face_flux(rc_b.x, rc_c.x, (ph_c.x - ph_b.x) * g.inv_dz, rho0).f;
        fb.y = face_flux(rc_b.y, rc_c.y, (ph_c.y - ph_b.y) * g.inv_dz, rho0).f;
        wb = ld2(w, qb);
    }

    for (int k = k0; k < k1; ++k, qk += plane) {
        const bool top = g.wall && (k + 1 == nz);
        // next plane (becomes the centre of the next iteration)
        double2 rc_t = rc_c, ph_t = ph_c;
        if (!top) {
            const long long qt = (long long)((k + 1 == nz) ? 0 : k + 1) * plane + col;
            rc_t = rho2_of(ld2(phi, qt));
            ph_t = phat2(ld2(p, qt), ld2(po, qt));
        }
        // y neighbours of the centre plane
        const double2 rc_n = rho2_of(ld2(phi, qk + col_n)), ph_n = phat2(ld2(p, qk + col_n), ld2(po, qk + col_n));
        const double2 rc_s = rho2_of(ld2(phi, qk + col_s)), ph_s = phat2(ld2(p, qk + col_s), ld2(po, qk + col_s));
        const double2 uc = ld2(u, qk + col), vc = ld2(v, qk + col), wc = ld2(w, qk + col), vs = ld2(v, qk + col_s);

        // x faces: m between (i0, i0+1), e between (i0+1, i0+2), wf between (i0-1, i0)
        double rc_e = __shfl_down_sync(0xffffffffu, rc_c.x, 1), ph_e = __shfl_down_sync(0xffffffffu, ph_c.x, 1);
        if (edge_r) {
            const long long qe = qk + row_j + ie;
            rc_e = rho_of(phi[qe]);
            ph_e = fma(c_pn, p[qe], -(c_po * po[qe]));
        }
        const Flux fm = face_flux(rc_c.x, rc_c.y, (ph_c.y - ph_c.x) * g.inv_dx, rho0);
        const Flux fe = face_flux(rc_c.y, rc_e, (ph_e - ph_c.y) * g.inv_dx, rho0);
        double f_w = __shfl_up_sync(0xffffffffu, fe.f, 1), u_w = __shfl_up_sync(0xffffffffu, uc.y, 1);
        if (edge_l) {
            const long long qw = qk + row_j + iw;
            f_w = face_flux(rho_of(phi[qw]), rc_c.x, (ph_c.x - fma(c_pn, p[qw], -(c_po * po[qw]))) * g.inv_dx, rho0).f;
            u_w = u[qw];
        }
        // y faces
        const Flux fn0 = face_flux(rc_c.x, rc_n.x, (ph_n.x - ph_c.x) * g.inv_dy, rho0);
        const Flux fn1 = face_flux(rc_c.y, rc_n.y, (ph_n.y - ph_c.y) * g.inv_dy, rho0);
        const double fs0 = face_flux(rc_s.x, rc_c.x, (ph_c.x - ph_s.x) * g.inv_dy, rho0).f;
        const double fs1 = face_flux(rc_s.y, rc_c.y, (ph_c.y - ph_s.y) * g.inv_dy, rho0).f;
        // z faces (wall faces carry zero flux)
        Flux ft0{0.0, 0.0}, ft1{0.0, 0.0};
        double gz0 = 0.0, gz1 = 0.0;
        if (!top) {
            gz0 = (ph_t.x - ph_c.x) * g.inv_dz;
            gz1 = (ph_t.y - ph_c.y) * g.inv_dz;
            ft0 = face_flux(rc_c.x, rc_t.x, gz0, rho0);
            ft1 = face_flux(rc_c.y, rc_t.y, gz1, rho0);
        }

        double2 out;
        out.x = c_div * ((uc.x - u_w) * g.inv_dx + (vc.x - vs.x) * g.inv_dy + (wc.x - wb.x) * g.inv_dz) +
                ((fm.f - f_w) * g.inv_dx + (fn0.f - fs0) * g.inv_dy + (ft0.f - fb.x) * g.inv_dz);
        out.y = c_div * ((uc.y - uc.x) * g.inv_dx + (vc.y - vs.y) * g.inv_dy + (wc.y - wb.y) * g.inv_dz) +
                ((fe.f - fm.f) * g.inv_dx + (fn1.f - fs1) * g.inv_dy + (ft1.f - fb.y) * g.inv_dz);
        *reinterpret_cast<double2 *>(rhs + qk + col) = out;

        out.x = uc.x - dt * ((fm.r - inv_rho0) * ((ph_c.y - ph_c.x) * g.inv_dx));
        out.y = uc.y - dt * ((fe.r - inv_rho0) * ((ph_e - ph_c.y) * g.inv_dx));
        *reinterpret_cast<double2 *>(up + qk + col) = out;
        out.x = vc.x - dt * ((fn0.r - inv_rho0) * ((ph_n.x - ph_c.x) * g.inv_dy));
        out.y = vc.y - dt * ((fn1.r - inv_rho0) * ((ph_n.y - ph_c.y) * g.inv_dy));
        *reinterpret_cast<double2 *>(vp + qk + col) = out;
        out.x = top ? wc.x : wc.x - dt * ((ft0.r - inv_rho0) * gz0);
        out.y = top ? wc.y : wc.y - dt * ((ft1.r - inv_rho0) * gz1);
        *reinterpret_cast<double2 *>(wp + qk + col) = out;

        fb = make_double2(ft0.f, ft1.f);
        wb = wc;
        rc_c = rc_t;
        ph_c = ph_t;
    }
}

// ------------------------------------------------------------------------------------------------
// Second form of the same kernel: identical decomposition (thread = 2 x-points, marching in z), but
//  * software-pipelined: the operands that miss in cache (phi, p, p_old of plane k+2 and u*, v*, w* of plane
//    k+1) are requested one iteration before they are used, so a warp waits on DRAM once per kernel instead
//    of once per plane; the row / edge neighbours of the current plane (L1 / L2 hits) are requested at the top
//    of the iteration and consumed last;
//  * trimmed arithmetic: rho_c = fma(rho1 - rho2, phi, rho2); 1 - rho0/rho_f = 1 - 2 rho0 / (rho_a + rho_b);
//    u' = u* + (dt/rho0) F, because (1/rho_f - 1/rho0) = -(1 - rho0/rho_f)/rho0, so the face flux F already
//    computed for the right-hand side is all the half-corrected velocity needs.
// ------------------------------------------------------------------------------------------------
__device__ __forceinline__ double2 ldg2(const double *f, long long q) {
    return __ldg(reinterpret_cast<const double2 *>(f + q));
}
__device__ __forceinline__ void stcs2(double *f, long long q, double2 v) {
    __stcs(reinterpret_cast<double2 *>(f + q), v);
}
// (1 - rho0/rho_f) for the face between cells of density ra and rb
__device__ __forceinline__ double flux_coef(double ra, double rb, double m2rho0) {
    return fma(m2rho0, rcp_density(ra + rb), 1.0);
}

template <bool WALL>
__global__ void __launch_bounds__(256, 2)
splitting_rhs_kernel2(GridParams g, double dt, int kc, const double *__restrict__ u, const double *__restrict__ v,
                      const double *__restrict__ w, const double *__restrict__ phi,
                      const double *__restrict__ p, const double *__restrict__ po,
                      double *__restrict__ rhs, double *__restrict__ up, double *__restrict__ vp,
                      double *__restrict__ wp) {
    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int i0 = 2 * (blockIdx.x * blockDim.x + threadIdx.x);
    const int j = blockIdx.y * blockDim.y + threadIdx.y;
    const int k0 = blockIdx.z * kc, k1 = min(k0 + kc, nz);
    const int jn = (j + 1 == ny) ? 0 : j + 1, js = (j == 0) ? ny - 1 : j - 1;
    const int iw = (i0 == 0) ? nx - 1 : i0 - 1, ie = (i0 + 2 == nx) ? 0 : i0 + 2;
    const int lane = (threadIdx.x + threadIdx.y * blockDim.x) & 31;
    const int rw = blockDim.x < 32 ? blockDim.x : 32;
    const bool edge_l = (lane % rw) == 0, edge_r = (lane % rw) == rw - 1;
    const long long plane = (long long)nx * ny;
    const long long col = (long long)j * nx + i0, col_n = (long long)jn * nx + i0, col_s = (long long)js * nx + i0;
    const long long q_e = (long long)j * nx + ie, q_w = (long long)j * nx + iw;
    const double drho = g.rho1 - g.rho2, rho2 = g.rho2, m2rho0 = -2.0 * g.rho0;
    const double c_div = g.rho0 / dt, c_up = dt / g.rho0;
    const double idx = g.inv_dx, idy = g.inv_dy, idz = g.inv_dz;

    auto rho_of = [&](double f) { return fma(drho, f, rho2); };
    auto rho2_of = [&](double2 f) { return make_double2(rho_of(f.x), rho_of(f.y)); };
    const double c_pn = g.c_pn, c_po = g.c_po;
    auto phat = [&](double a, double b) { return fma(c_pn, a, -(c_po * b)); };   // c_po = 1: exactly 2a - b
    auto phat2 = [&](double2 a, double2 b) { return make_double2(phat(a.x, b.x), phat(a.y, b.y)); };

    // prologue: centre plane k0, the bottom-face flux and w below
    long long qk = (long long)k0 * plane;
    double2 rc_c = rho2_of(ldg2(phi, qk + col)), ph_c = phat2(ldg2(p, qk + col), ldg2(po, qk + col));
    double2 fb = make_double2(0.0, 0.0), wb = make_double2(0.0, 0.0);
    if (!(WALL && k0 == 0)) {
        const long long qb = (long long)((k0 == 0) ? nz - 1 : k0 - 1) * plane + col;
        const double2 rc_b = rho2_of(ldg2(phi, qb)), ph_b = phat2(ldg2(p, qb), ldg2(po, qb));
        fb.x = flux_coef(rc_b.x, rc_c.x, m2rho0) * ((ph_c.x - ph_b.x) * idz);
        fb.y = flux_coef(rc_b.y, rc_c.y, m2rho0) * ((ph_c.y - ph_b.y) * idz);
        wb = ldg2(w, qb);
    }
    // pipeline registers: plane k+1 (phi, p, p_old at the centre column) and plane k (u*, v*, w*, v* south)
    auto plane_of = [&](int k) { return WALL ? min(k, nz - 1) : (k >= nz ? k - nz : k); };
    long long qt = (long long)plane_of(k0 + 1) * plane + col;
    double2 a_phi = ldg2(phi, qt), a_p = ldg2(p, qt), a_po = ldg2(po, qt);
    double2 uc = ldg2(u, qk + col), vc = ldg2(v, qk + col), wc = ldg2(w, qk + col), vs = ldg2(v, qk + col_s);

    for (int k = k0; k < k1; ++k, qk += plane) {
        const bool top = WALL && (k + 1 == nz);
        // ---- requests for the NEXT iteration (DRAM latency, consumed one iteration later)
        double2 n_phi = a_phi, n_p = a_p, n_po = a_po, n_uc = uc, n_vc = vc, n_wc = wc, n_vs = vs;
        if (k + 1 < k1) {
            const long long q2 = (long long)plane_of(k + 2) * plane + col, q1 = qk + plane;
            n_phi = ldg2(phi, q2); n_p = ldg2(p, q2); n_po = ldg2(po, q2);
            n_uc = ldg2(u, q1 + col); n_vc = ldg2(v, q1 + col); n_wc = ldg2(w, q1 + col); n_vs = ldg2(v, q1 + col_s);
        }
        // ---- requests for THIS iteration that hit in L1 / L2: row neighbours and the two edge columns
        const double2 r_nphi = ldg2(phi, qk + col_n), r_np = ldg2(p, qk + col_n), r_npo = ldg2(po, qk + col_n);
        const double2 r_sphi = ldg2(phi, qk + col_s), r_sp = ldg2(p, qk + col_s), r_spo = ldg2(po, qk + col_s);
        double e_phi = 0.0, e_p = 0.0, e_po = 0.0, w_phi = 0.0, w_p = 0.0, w_po = 0.0, w_u = 0.0;
        if (edge_r) { e_phi = __ldg(phi + qk + q_e); e_p = __ldg(p + qk + q_e); e_po = __ldg(po + qk + q_e); }
        if (edge_l) { w_phi = __ldg(phi + qk + q_w); w_p = __ldg(p + qk + q_w); w_po = __ldg(po + qk + q_w); w_u = __ldg(u + qk + q_w); }

        // ---- z faces (top of this plane; wall faces carry zero flux)
        double2 rc_t = rc_c, ph_t = ph_c, ft = make_double2(0.0, 0.0);
        if (!top) {
            rc_t = rho2_of(a_phi);
            ph_t = phat2(a_p, a_po);
            ft.x = flux_coef(rc_c.x, rc_t.x, m2rho0) * ((ph_t.x - ph_c.x) * idz);
            ft.y = flux_coef(rc_c.y, rc_t.y, m2rho0) * ((ph_t.y - ph_c.y) * idz);
        }
        // ---- x faces: m between (i0, i0+1), e between (i0+1, i0+2), west face from the left lane
        double rc_e = __shfl_down_sync(0xffffffffu, rc_c.x, 1), ph_e = __shfl_down_sync(0xffffffffu, ph_c.x, 1);
        if (edge_r) { rc_e = rho_of(e_phi); ph_e = phat(e_p, e_po); }
        const double fm = flux_coef(rc_c.x, rc_c.y, m2rho0) * ((ph_c.y - ph_c.x) * idx);
        const double fe = flux_coef(rc_c.y, rc_e, m2rho0) * ((ph_e - ph_c.y) * idx);
        double f_w = __shfl_up_sync(0xffffffffu, fe, 1), u_w = __shfl_up_sync(0xffffffffu, uc.y, 1);
        if (edge_l) {
            f_w = flux_coef(rho_of(w_phi), rc_c.x, m2rho0) * ((ph_c.x - phat(w_p, w_po)) * idx);
            u_w = w_u;
        }
        // ---- y faces
        const double2 rc_n = rho2_of(r_nphi), ph_n = phat2(r_np, r_npo);
        const double2 rc_s = rho2_of(r_sphi), ph_s = phat2(r_sp, r_spo);
        const double fn0 = flux_coef(rc_c.x, rc_n.x, m2rho0) * ((ph_n.x - ph_c.x) * idy);
        const double fn1 = flux_coef(rc_c.y, rc_n.y, m2rho0) * ((ph_n.y - ph_c.y) * idy);
        const double fs0 = flux_coef(rc_s.x, rc_c.x, m2rho0) * ((ph_c.x - ph_s.x) * idy);
        const double fs1 = flux_coef(rc_s.y, rc_c.y, m2rho0) * ((ph_c.y - ph_s.y) * idy);

        double2 out;
        out.x = c_div * ((uc.x - u_w) * idx + (vc.x - vs.x) * idy + (wc.x - wb.x) * idz) +
                ((fm - f_w) * idx + (fn0 - fs0) * idy + (ft.x - fb.x) * idz);
        out.y = c_div * ((uc.y - uc.x) * idx + (vc.y - vs.y) * idy + (wc.y - wb.y) * idz) +
                ((fe - fm) * idx + (fn1 - fs1) * idy + (ft.y - fb.y) * idz);
        stcs2(rhs, qk + col, out);
        stcs2(up, qk + col, make_double2(fma(c_up, fm, uc.x), fma(c_up, fe, uc.y)));
        stcs2(vp, qk + col, make_double2(fma(c_up, fn0, vc.x), fma(c_up, fn1, vc.y)));
        stcs2(wp, qk + col, make_double2(fma(c_up, ft.x, wc.x), fma(c_up, ft.y, wc.y)));   // top wall: ft = 0

        fb = ft; wb = wc; rc_c = rc_t; ph_c = ph_t;
        a_phi = n_phi; a_p = n_p; a_po = n_po; uc = n_uc; vc = n_vc; wc = n_wc; vs = n_vs;
    }
}

// ------------------------------------------------------------------------------------------------
// a9: u = u' - dt/rho0 grad p^(n+1)   (eq. 18; p^(n+1) was already stored by a8)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
correction_kernel(GridParams g, double dt, long long q0, long long q1, const double *__restrict__ pn,
                  const double *__restrict__ up, const double *__restrict__ vp, const double *__restrict__ wp,
                  double *__restrict__ u, double *__restrict__ v, double *__restrict__ w) {
    // two consecutive x points per thread (nx is even and q0 a multiple of nx): 16-byte loads and streaming stores
    const long long q = q0 + 2 * ((long long)blockIdx.x * blockDim.x + threadIdx.x);   // this launch covers points q0 .. q1 - 1
    if (q >= q1) return;
    const int i = (int)(q % g.nx);
    const long long r = q / g.nx;
    const int j = (int)(r % g.ny), k = (int)(r / g.ny);
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    const long long qip = (i + 2 == g.nx) ? q - (g.nx - 2) : q + 2;
    const long long qjp = (j + 1 == g.ny) ? q - (g.ny - 1) * sy : q + sy;
    const long long qkp = (k + 1 == g.nz) ? q - (g.nz - 1) * sz : q + sz;
    const bool top = g.wall && (k + 1 == g.nz);
    const double c = dt / g.rho0;
    auto ld2 = [](const double *f, long long a) { return *reinterpret_cast<const double2 *>(f + a); };
    const double2 pc = ld2(pn, q), pj = ld2(pn, qjp), pk = ld2(pn, qkp);
    const double pe = pn[qip];
    const double2 a = ld2(up, q), b = ld2(vp, q), d = ld2(wp, q);
    stcs2(u, q, make_double2(a.x - c * ((pc.y - pc.x) * g.inv_dx), a.y - c * ((pe - pc.y) * g.inv_dx)));
    stcs2(v, q, make_double2(b.x - c * ((pj.x - pc.x) * g.inv_dy), b.y - c * ((pj.y - pc.y) * g.inv_dy)));
    stcs2(w, q, top ? d : make_double2(d.x - c * ((pk.x - pc.x) * g.inv_dz), d.y - c * ((pk.y - pc.y) * g.inv_dz)));
}

// ------------------------------------------------------------------------------------------------
// FFT of a tile held in shared memory: all passes, one __syncthreads between passes.
// NT threads cooperate; thread (l = tid % C, t = tid / C + m * NT/C) owns butterfly t of line l.
// ------------------------------------------------------------------------------------------------
template <int N, int C, bool SWZ, int NT, int DIR>
__device__ __forceinline__ void tile_fft(double2 *s, const double2 *__restrict__ tw, int tws, int tid) {
    constexpr int P = Fact<N>::P;
    const int l = tid % C;
#pragma unroll
    for (int pp = 0; pp < P; ++pp) {
        const int p = DIR < 0 ? pp + 1 : P - pp;
        for (int t = tid / C; t < N / 8; t += NT / C) {
            int pos[8], n2;
            double2 v[8];
            pass_positions<N>(p, t, pos, n2);
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = s[tile_index<C, SWZ>(pos[e], l)];
            if (DIR < 0) fwd_pass_regs<N>(p, n2, v, tw, tws);
            else inv_pass_regs<N>(p, n2, v, tw, tws);
#pragma unroll
            for (int e = 0; e < 8; ++e) s[tile_index<C, SWZ>(pos[e], l)] = v[e];
        }
        if (pp + 1 < P) __syncthreads();
    }
}

// ------------------------------------------------------------------------------------------------
// a5 / a7 / a6p: transform along a strided direction.  A tile is C consecutive kx columns x the whole
// line (N positions, `row_stride` elements apart); blockIdx.x = tx + n_tiles_x * outer.
// ------------------------------------------------------------------------------------------------
enum { MODE_FWD = 0, MODE_INV = 1, MODE_SOLVE = 2 };

struct StridedArgs {
    double2 *data;
    long long row_stride;    // elements between line positions r and r+1
    long long outer_stride;  // elements between outer indices (k for the y pass, j for the z pass)
    int n_tiles_x;           // tiles along kx
    int nxh;                 // valid kx columns (nx/2 + 1)
    const double2 *tw;       // e^{-2 pi i m / N}
    // SOLVE only: eigenvalues in storage (permuted) order
    const double *lam_x, *lam_outer, *lam_pos;
};

// The first pass reads its 8 elements straight from global memory into registers and the last pass
// writes them straight back (the permuted order makes every pass in place), so shared memory is only
// the exchange buffer between passes: P-1 exchanges, P-1 barriers, no staging copies.
template <int N, int C, int MODE, int NT>
__global__ void __launch_bounds__(NT, (N * C * 16 <= 72 * 1024 && NT == 256) ? 3 : 1) fft_strided_kernel(StridedArgs a) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    constexpr int P = Fact<N>::P;
    const int tid = threadIdx.x;
    const int tx = blockIdx.x % a.n_tiles_x, outer = blockIdx.x / a.n_tiles_x;
    const int l = tid % C;
    const int kx = tx * C + l;
    const bool valid = kx < a.nxh;
    double2 *gp = a.data + (long long)outer * a.outer_stride + kx;
    const long long rs = a.row_stride;

    auto load8 = [&](bool from_global, const int *pos, double2 *v) {
        if (from_global) {
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = valid ? gp[(long long)pos[e] * rs] : make_double2(0.0, 0.0);
        } else {
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = s[pos[e] * C + l];
        }
    };
    auto store8 = [&](bool to_global, const int *pos, const double2 *v) {
        if (to_global) {
            if (valid) {
#pragma unroll
                for (int e = 0; e < 8; ++e) gp[(long long)pos[e] * rs] = v[e];
            }
        } else {
#pragma unroll
            for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
        }
    };

    if (MODE == MODE_FWD || MODE == MODE_INV) {
#pragma unroll
        for (int pp = 0; pp < P; ++pp) {
            const int p = (MODE == MODE_FWD) ? pp + 1 : P - pp;
            for (int t = tid / C; t < N / 8; t += NT / C) {
                int pos[8], n2;
                double2 v[8];
                pass_positions<N>(p, t, pos, n2);
                load8(pp == 0, pos, v);
                if (MODE == MODE_FWD) fwd_pass_regs<N>(p, n2, v, a.tw, 1);
                else inv_pass_regs<N>(p, n2, v, a.tw, 1);
                store8(pp == P - 1, pos, v);
            }
            if (pp + 1 < P) __syncthreads();
        }
    } else {
        // forward passes 1..P-1
#pragma unroll
        for (int p = 1; p < P; ++p) {
            for (int t = tid / C; t < N / 8; t += NT / C) {
                int pos[8], n2;
                double2 v[8];
                pass_positions<N>(p, t, pos, n2);
                load8(p == 1, pos, v);
                fwd_pass_regs<N>(p, n2, v, a.tw, 1);
                store8(false, pos, v);
            }
            __syncthreads();
        }
        // last forward pass, division by the eigenvalue sum, first inverse pass: all in registers
        const double lam_xy = a.lam_x[valid ? kx : 0] + a.lam_outer[outer];
        for (int t = tid / C; t < N / 8; t += NT / C) {
            int pos[8], n2;
            double2 v[8];
            pass_positions<N>(P, t, pos, n2);
            load8(P == 1, pos, v);
            fwd_pass_regs<N>(P, n2, v, a.tw, 1);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const double den = lam_xy + a.lam_pos[pos[e]];
                const double inv = (den == 0.0) ? 0.0 : 1.0 / den;     // the (0,0,0) mode is dropped (zero-mean gauge)
                v[e] = cscale(v[e], inv);
            }
            inv_pass_regs<N>(P, n2, v, a.tw, 1);
            store8(P == 1, pos, v);
        }
#pragma unroll
        for (int p = P - 1; p >= 1; --p) {
            __syncthreads();
            for (int t = tid / C; t < N / 8; t += NT / C) {
                int pos[8], n2;
                double2 v[8];
                pass_positions<N>(p, t, pos, n2);
                load8(false, pos, v);
                inv_pass_regs<N>(p, n2, v, a.tw, 1);
                store8(p == 1, pos, v);
            }
        }
    }
}

// ------------------------------------------------------------------------------------------------
// Cooperative copy of TOT contiguous elements with B loads in flight per thread: all loads of a batch are
// issued before the first use, so a CTA pays one memory latency per batch instead of one per element.
// ------------------------------------------------------------------------------------------------
template <int TOT, int NT, int B, typename T, typename Load, typename Store>
__device__ __forceinline__ void batched_copy(int tid, Load load, Store store) {
    for (int base = 0; base < TOT; base += NT * B) {
        T vals[B];
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int idx = base + b * NT + tid;
            if (idx < TOT) vals[b] = load(idx);
        }
#pragma unroll
        for (int b = 0; b < B; ++b) {
            const int idx = base + b * NT + tid;
            if (idx < TOT) store(idx, vals[b]);
        }
    }
}

// ------------------------------------------------------------------------------------------------
// a4: real-to-complex along x.  CTA = 8 consecutive lines (contiguous in memory), N2 = nx/2.
// Output row (line) layout: kx = 0..N2 in natural order; row pitch = N2 + 8,
// so the 8 output rows of a CTA are one contiguous block as well.
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT, NT == 256 ? 2 : 1)
fft_x_r2c_kernel(const double *__restrict__ rhs, double2 *__restrict__ spec,
                 const double2 *__restrict__ tw /* e^{-2 pi i m / nx} */, SpecRows sr) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    constexpr int PITCH = N2 + 8;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    const double2 *src = reinterpret_cast<const double2 *>(rhs) + line0 * N2;
    batched_copy<8 * N2, NT, 8, double2>(
        tid, [&](int idx) { return src[idx]; },
        [&](int idx, double2 val) { s[tile_index<8, true>(idx % N2, idx / N2)] = val; });
    __syncthreads();
    tile_fft<N2, 8, true, NT, -1>(s, tw, 2, tid);
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) r2c_post_item<N2, 8, true>(s, item / 8, item % 8, tw);
    __syncthreads();
    double2 *dst = spec + spec_row_offset(sr, line0, PITCH);
    for (int idx = tid; idx < 8 * PITCH; idx += NT) {
        const int l = idx / PITCH, k = idx % PITCH;     // spectrum rows are stored in natural kx order
        if (k <= N2) dst[idx] = s[tile_index<8, true>(k == N2 ? N2 : pos_of_freq<N2>(k), l)];
    }
}

// ------------------------------------------------------------------------------------------------
// a8: complex-to-real along x with the normalisation of the whole transform chain; writes p^(n+1).
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT, NT == 256 ? 2 : 1)
fft_x_c2r_kernel(const double2 *__restrict__ spec, double *__restrict__ out,
                 const double2 *__restrict__ tw, double scale, SpecRows sr) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    constexpr int PITCH = N2 + 8;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    const double2 *src = spec + spec_row_offset(sr, line0, PITCH);
    batched_copy<8 * PITCH, NT, 9, double2>(
        tid, [&](int idx) { return src[idx]; },
        [&](int idx, double2 val) {
            const int l = idx / PITCH, k = idx % PITCH;
            if (k <= N2) s[tile_index<8, true>(k == N2 ? N2 : pos_of_freq<N2>(k), l)] = val;
        });
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) c2r_pre_item<N2, 8, true>(s, item / 8, item % 8, tw);
    __syncthreads();
    tile_fft<N2, 8, true, NT, +1>(s, tw, 2, tid);
    __syncthreads();
    double2 *dst = reinterpret_cast<double2 *>(out) + line0 * N2;
    for (int idx = tid; idx < 8 * N2; idx += NT)
        dst[idx] = cscale(s[tile_index<8, true>(idx % N2, idx / N2)], scale);
}

// ------------------------------------------------------------------------------------------------
// a6w: Gauss elimination along z.  One thread per (kx, ky) column, marching in k;
// consecutive threads are consecutive kx, so every access is coalesced.
//   a x_{k-1} + b_k x_k + a x_{k+1} = d_k,  a = 1/dz^2,  b_k = -2a + lam_xy (interior), -a + lam_xy (ends)
// Forward sweep stores d'_k in place and c'_k in `cp`; the backward sweep reads both.
// The singular column (0,0) is skipped here and handled by thomas_singular_kernel.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
thomas_kernel(double2 *__restrict__ spec, double *__restrict__ cp, int pitch, int ny, int nz, int nxh,
              const double *__restrict__ lam_x, const double *__restrict__ lam_y, double inv_dz2, long long plane) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long ncol = (long long)pitch * ny;
    if (c >= ncol || c == 0) return;
    const int kx = (int)(c % pitch), jy = (int)(c / pitch);
    if (kx >= nxh) return;
    const double lam = lam_x[kx] + lam_y[jy];
    const double a = inv_dz2, b_end = -inv_dz2 + lam, b_in = -2.0 * inv_dz2 + lam;
    double inv = 1.0 / b_end;
    double cpv = a * inv;
    double2 d = spec[c];
    double2 dp = make_double2(d.x * inv, d.y * inv);
    spec[c] = dp;
    cp[c] = cpv;
#pragma unroll 4
    for (int k = 1; k < nz; ++k) {
        const long long q = c + (long long)k * plane;
        d = spec[q];
        const double b = (k == nz - 1) ? b_end : b_in;
        inv = 1.0 / (b - a * cpv);
        cpv = a * inv;
        dp = make_double2((d.x - a * dp.x) * inv, (d.y - a * dp.y) * inv);
        spec[q] = dp;
        cp[q] = cpv;
    }
    double2 x = dp;  // x_{nz-1} = d'_{nz-1}
#pragma unroll 4
    for (int k = nz - 2; k >= 0; --k) {
        const long long q = c + (long long)k * plane;
        const double2 dk = spec[q];
        const double ck = cp[q];
        x = make_double2(dk.x - ck * x.x, dk.y - ck * x.y);
        spec[q] = x;
    }
}

// The (kx,ky) = (0,0) column: lam_xy = 0, the system is singular (pure Neumann).  Eliminate rows
// 0..nz-2, pin x_{nz-1} = 0, back-substitute, then remove the mean over k (zero-mean gauge, R5).
__global__ void thomas_singular_kernel(double2 *__restrict__ spec, long long col_stride, int nz,
                                       const double *__restrict__ coef /* inv_k, c'_k interleaved: 2 nz doubles */) {
    extern __shared__ double sm[];
    double *dr = sm, *di = sm + nz, *cf = sm + 2 * nz, *mean = sm + 4 * nz;
    for (int k = threadIdx.x; k < nz; k += blockDim.x) {
        const double2 d = spec[(long long)k * col_stride];
        dr[k] = d.x;
        di[k] = d.y;
        cf[2 * k] = coef[2 * k];
        cf[2 * k + 1] = coef[2 * k + 1];
    }
    __syncthreads();
    if (threadIdx.x < 2) {                      // thread 0: real parts, thread 1: imaginary parts
        double *x = threadIdx.x == 0 ? dr : di;
        const double a = cf[2 * nz - 1];        // slot of c'_{nz-1} (never used as such) carries a = 1/dz^2
        double prev = x[0] * cf[0];
        x[0] = prev;
        for (int k = 1; k <= nz - 2; ++k) {
            prev = (x[k] - a * prev) * cf[2 * k];
            x[k] = prev;
        }
        double nxt = 0.0, sum = 0.0;            // x_{nz-1} = 0 (the pinned unknown, R5)
        x[nz - 1] = 0.0;
        for (int k = nz - 2; k >= 0; --k) {
            nxt = x[k] - cf[2 * k + 1] * nxt;
            x[k] = nxt;
        }
        for (int k = 0; k < nz; ++k) sum += x[k];
        mean[threadIdx.x] = sum / nz;
    }
    __syncthreads();
    const double mr = mean[0], mi = mean[1];
    for (int k = threadIdx.x; k < nz; k += blockDim.x)
        spec[(long long)k * col_stride] = make_double2(dr[k] - mr, di[k] - mi);
}

}  // namespace flutas
