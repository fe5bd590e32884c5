// kernels_rhs.cuh -- third form of the fused density + splitting right-hand side kernel (rows a1-a3 of the step;
// eqs. 2, 16, 17: PAPER.md:76, 153-155, 161), fed by the bulk-copy engine.
//
// Same decomposition as splitting_rhs_kernel2 in kernels.cuh (block = 64 x-threads x 2 points x TY rows of j, marching in z; TY = 8: 57 KB per slab,
// one CTA of 512 threads per SM, 25 % less halo traffic from L2 than TY = 4 and 3 % faster), but
// the operands no longer travel through registers: one warp asks the copy engine (cp.async.bulk -> mbarrier
// complete_tx) for whole row segments of the plane two steps ahead, which land in a three-slot ring of plane
// slabs in shared memory -- phi, p, p_old with their j-1 / j+TY rows and i-1 / i+X columns, u* with its west
// column, v* with its south row, w*.  Periodic wrap (x, y, z) is resolved when the copy is issued, so the
// compute loop has no edge lanes, no shuffles and no global loads at all: every neighbour is a shared-memory
// read, a warp waits on an mbarrier for data requested two planes earlier, and the only registers carried from
// plane to plane are rho_c, p_hat of the centre plane, the bottom-face flux and w below.
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

namespace flutas {

struct Rhs3Geom {
    static constexpr int X = 128, TY = 8, NTX = X / 2;        // tile: X cells along x, TY rows of j; thread = 2 cells
    static constexpr int RP = X + 4;                           // row pitch with the two halo pairs (doubles)
    static constexpr int O_PHI = 0, O_P = (TY + 2) * RP, O_PO = 2 * (TY + 2) * RP, O_U = 3 * (TY + 2) * RP;
    static constexpr int O_V = O_U + TY * RP, O_W = O_V + (TY + 1) * X;
    static constexpr int STAGE = O_W + TY * X;                 // doubles per plane slab
    static constexpr int NSLOT = 3;
    static constexpr int NROWCOPY = 3 * (TY + 2) + TY + (TY + 1) + TY;   // 55 row copies per slab
    static_assert(NROWCOPY <= 4 * (NTX * TY / 32), "four lanes of every warp issue one row copy each");
    static_assert((STAGE * 8) % 16 == 0 && (RP * 8) % 16 == 0, "bulk copies need 16-byte granules");
    static constexpr size_t SMEM = (size_t)NSLOT * STAGE * 8 + 128;
};

enum { RHS3_LOAD_SCALARS = 1, RHS3_LOAD_UV = 2, RHS3_LOAD_W = 4, RHS3_LOAD_ALL = 7 };

template <bool WALL>
__global__ void __launch_bounds__(Rhs3Geom::NTX * Rhs3Geom::TY, Rhs3Geom::TY == 4 ? 2 : 1)
splitting_rhs_kernel3(GridParams g, double dt, int kc, int k_base, int k_end, const double *__restrict__ u, const double *__restrict__ v,
                      const double *__restrict__ w, const double *__restrict__ phi,
                      const double *__restrict__ p, const double *__restrict__ po,
                      double *__restrict__ rhs, double *__restrict__ up, double *__restrict__ vp,
                      double *__restrict__ wp) {
    using G = Rhs3Geom;
    extern __shared__ unsigned char smem_raw[];
    double *ring = reinterpret_cast<double *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    __shared__ uint64_t full[G::NSLOT];

    const int nx = g.nx, ny = g.ny, nz = g.nz;
    const int tx = threadIdx.x, ty = threadIdx.y;
    const int tid = ty * G::NTX + tx;
    const int x0 = blockIdx.x * G::X, j0 = blockIdx.y * G::TY;
    const int k0 = k_base + blockIdx.z * kc, k1 = min(k0 + kc, k_end);   // this launch covers planes k_base .. k_end - 1
    const long long plane = (long long)nx * ny;

    if (tid == 0) {
#pragma unroll
        for (int s = 0; s < G::NSLOT; ++s) mbar_init(&full[s], 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    // ---- producer side: the first four lanes of every warp own one row copy of a slab each (a bulk copy costs its
    //      issuing warp ~65 cycles, so the copies are spread over all warps); wrap in x, y, z is resolved here
    const double *r_src = nullptr;      // field base + row offset (plane added per slab)
    int r_dst = 0, r_kind = 0, r_mask = 0;   // kind: 2 = both halo pairs, 1 = west pair only, 0 = none
    if ((tid & 31) < 4 && (tid >> 5) * 4 + (tid & 31) < G::NROWCOPY) {
        const int r = (tid >> 5) * 4 + (tid & 31);
        auto wrap_j = [&](int j) { return j < 0 ? j + ny : (j >= ny ? j - ny : j); };
        if (r < 3 * (G::TY + 2)) {
            const int f = r / (G::TY + 2), rr = r % (G::TY + 2);
            r_src = (f == 0 ? phi : (f == 1 ? p : po)) + (long long)wrap_j(j0 - 1 + rr) * nx;
            r_dst = f * (G::TY + 2) * G::RP + rr * G::RP;
            r_kind = 2; r_mask = RHS3_LOAD_SCALARS;
        } else if (r < 3 * (G::TY + 2) + G::TY) {
            const int rr = r - 3 * (G::TY + 2);
            r_src = u + (long long)(j0 + rr) * nx;
            r_dst = G::O_U + rr * G::RP;
            r_kind = 1; r_mask = RHS3_LOAD_UV;
        } else if (r < 3 * (G::TY + 2) + 2 * G::TY + 1) {
            const int rr = r - (3 * (G::TY + 2) + G::TY);
            r_src = v + (long long)wrap_j(j0 - 1 + rr) * nx;
            r_dst = G::O_V + rr * G::X;
            r_kind = 0; r_mask = RHS3_LOAD_UV;
        } else {
            const int rr = r - (3 * (G::TY + 2) + 2 * G::TY + 1);
            r_src = w + (long long)(j0 + rr) * nx;
            r_dst = G::O_W + rr * G::X;
            r_kind = 0; r_mask = RHS3_LOAD_W;
        }
    }
    const bool x_interior = x0 > 0 && x0 + G::X < nx;
    const int xw = x0 == 0 ? nx - 2 : x0 - 2, xe = x0 + G::X == nx ? 0 : x0 + G::X;
    auto plane_of = [&](int k) { return WALL ? max(0, min(k, nz - 1)) : (k < 0 ? k + nz : (k >= nz ? k - nz : k)); };

    // called by every thread
    auto issue_slab = [&](int k, int slot, int mask) {
        if (tid == 0) {
            const uint32_t total = ((mask & RHS3_LOAD_SCALARS) ? 3 * (G::TY + 2) * (G::X + 4) * 8 : 0) +
                                   ((mask & RHS3_LOAD_UV) ? G::TY * (G::X + 2) * 8 + (G::TY + 1) * G::X * 8 : 0) +
                                   ((mask & RHS3_LOAD_W) ? G::TY * G::X * 8 : 0);
            mbar_arrive_expect_tx(&full[slot], total);     // the phase cannot complete before this arrival
        }
        if (r_src != nullptr && (r_mask & mask)) {
            const double *src = r_src + (long long)plane_of(k) * plane;
            double *dst = ring + slot * G::STAGE + r_dst;
            if (r_kind == 0) {
                bulk_load(dst, src + x0, G::X * 8, &full[slot]);
            } else if (r_kind == 2 && x_interior) {
                bulk_load(dst, src + x0 - 2, (G::X + 4) * 8, &full[slot]);
            } else {
                bulk_load(dst, src + xw, 16, &full[slot]);
                bulk_load(dst + 2, src + x0, G::X * 8, &full[slot]);
                if (r_kind == 2) bulk_load(dst + 2 + G::X, src + xe, 16, &full[slot]);
            }
        }
    };

    // ---- slabs: m = 0 .. m_last holds plane k0 - 1 + m; the first is only the plane below (rho_c, p_hat, w*),
    //      the last only the plane above (rho_c, p_hat) of the chunk
    const int m_last = k1 - k0 + 1;
    auto mask_of = [&](int m) { return m == 0 ? (RHS3_LOAD_SCALARS | RHS3_LOAD_W) : (m == m_last ? RHS3_LOAD_SCALARS : RHS3_LOAD_ALL); };
#pragma unroll
    for (int m = 0; m < G::NSLOT; ++m)
        if (m <= m_last) issue_slab(k0 - 1 + m, m, mask_of(m));

    const double drho = g.rho1 - g.rho2, rho2 = g.rho2, one = g.flux_one, m2rho0 = -2.0 * g.rho0 * g.flux_one;
    const double c_div = g.rho0 / dt, c_up = dt / g.rho0;
    const double idx = g.inv_dx, idy = g.inv_dy, idz = g.inv_dz;
    const double c_pn = g.c_pn, c_po = g.c_po;
    auto rho_of = [&](double f) { return fma(drho, f, rho2); };
    auto phat = [&](double a, double b) { return fma(c_pn, a, -(c_po * b)); };   // c_po = 1: exactly 2a - b
    auto ld2s = [](const double *q) { return *reinterpret_cast<const double2 *>(q); };

    const int col = 2 + 2 * tx;                         // column of cell i0 inside a haloed row
    const int c_row = (ty + 1) * G::RP + col;           // centre row of phi / p / p_old
    const long long out0 = (long long)(j0 + ty) * nx + x0 + 2 * tx;
    const bool wall_w = g.wall_x && x0 + 2 * tx == 0, wall_e = g.wall_x && x0 + 2 * tx + 2 == nx;
    const bool wall_s = g.wall_y && j0 + ty == 0, wall_n = g.wall_y && j0 + ty + 1 == ny;

    // carried from plane to plane
    double2 rc_b = make_double2(1.0, 1.0), ph_b = make_double2(0.0, 0.0);   // rho_c, p_hat of the plane below
    double2 fb = make_double2(0.0, 0.0), wb = make_double2(0.0, 0.0);       // its top-face flux and w*
    double2 part = make_double2(0.0, 0.0);                                  // in-plane part of rhs of the plane below

    for (int m = 0; m <= m_last; ++m) {
        const int q = k0 - 1 + m, slot = m % G::NSLOT;
        const double *S = ring + slot * G::STAGE;
        mbar_wait(&full[slot], (m / G::NSLOT) & 1);

        const double2 a_phi = ld2s(S + G::O_PHI + c_row), a_p = ld2s(S + G::O_P + c_row), a_po = ld2s(S + G::O_PO + c_row);
        const double2 rc = make_double2(rho_of(a_phi.x), rho_of(a_phi.y));
        const double2 ph = make_double2(phat(a_p.x, a_po.x), phat(a_p.y, a_po.y));

        // z face between planes q-1 and q (wall faces carry zero flux)
        double2 fz = make_double2(0.0, 0.0);
        if (m >= 1 && !(WALL && (q == 0 || q == nz))) {
            fz.x = flux_coef(rc_b.x, rc.x, m2rho0, one) * ((ph.x - ph_b.x) * idz);
            fz.y = flux_coef(rc_b.y, rc.y, m2rho0, one) * ((ph.y - ph_b.y) * idz);
        }
        if (m >= 2) {   // plane q-1 is complete: its top-face flux is fz, its bottom-face flux fb
            const long long o = (long long)(q - 1) * plane + out0;
            stcs2(rhs, o, make_double2(part.x + (fz.x - fb.x) * idz, part.y + (fz.y - fb.y) * idz));
            stcs2(wp, o, make_double2(fma(c_up, fz.x, wb.x), fma(c_up, fz.y, wb.y)));     // top wall: fz = 0
        }
        if (m == 0) {
            if (!(WALL && q < 0)) wb = ld2s(S + G::O_W + ty * G::X + 2 * tx);
        } else if (m < m_last) {
            // ---- in-plane faces of plane q
            const int n_row = c_row + G::RP, s_row = c_row - G::RP;
            const double2 n_phi = ld2s(S + G::O_PHI + n_row), n_p = ld2s(S + G::O_P + n_row), n_po = ld2s(S + G::O_PO + n_row);
            const double2 s_phi = ld2s(S + G::O_PHI + s_row), s_p = ld2s(S + G::O_P + s_row), s_po = ld2s(S + G::O_PO + s_row);
            const double e_phi = S[G::O_PHI + c_row + 2], e_p = S[G::O_P + c_row + 2], e_po = S[G::O_PO + c_row + 2];
            const double w_phi = S[G::O_PHI + c_row - 1], w_p = S[G::O_P + c_row - 1], w_po = S[G::O_PO + c_row - 1];
            const double2 uc = ld2s(S + G::O_U + ty * G::RP + col);
            double u_w = S[G::O_U + ty * G::RP + col - 1];
            const double2 vc = ld2s(S + G::O_V + (ty + 1) * G::X + 2 * tx);
            double2 vs = ld2s(S + G::O_V + ty * G::X + 2 * tx);
            const double2 wc = ld2s(S + G::O_W + ty * G::X + 2 * tx);

            const double fm = flux_coef(rc.x, rc.y, m2rho0, one) * ((ph.y - ph.x) * idx);
            double fe = flux_coef(rc.y, rho_of(e_phi), m2rho0, one) * ((phat(e_p, e_po) - ph.y) * idx);
            double fw = flux_coef(rho_of(w_phi), rc.x, m2rho0, one) * ((ph.x - phat(w_p, w_po)) * idx);
            const double2 rc_n = make_double2(rho_of(n_phi.x), rho_of(n_phi.y)), ph_n = make_double2(phat(n_p.x, n_po.x), phat(n_p.y, n_po.y));
            const double2 rc_s = make_double2(rho_of(s_phi.x), rho_of(s_phi.y)), ph_s = make_double2(phat(s_p.x, s_po.x), phat(s_p.y, s_po.y));
            double fn0 = flux_coef(rc.x, rc_n.x, m2rho0, one) * ((ph_n.x - ph.x) * idy);
            double fn1 = flux_coef(rc.y, rc_n.y, m2rho0, one) * ((ph_n.y - ph.y) * idy);
            double fs0 = flux_coef(rc_s.x, rc.x, m2rho0, one) * ((ph.x - ph_s.x) * idy);
            double fs1 = flux_coef(rc_s.y, rc.y, m2rho0, one) * ((ph.y - ph_s.y) * idy);
            // walls along x / y: wall faces carry no flux and the unstored first wall face no velocity;
            // the halo the copies wrapped around periodically is then simply not used
            if (wall_e) fe = 0.0;
            if (wall_w) { fw = 0.0; u_w = 0.0; }
            if (wall_n) fn0 = fn1 = 0.0;
            if (wall_s) { fs0 = fs1 = 0.0; vs = make_double2(0.0, 0.0); }

            part.x = c_div * ((uc.x - u_w) * idx + (vc.x - vs.x) * idy + (wc.x - wb.x) * idz) +
                     ((fm - fw) * idx + (fn0 - fs0) * idy);
            part.y = c_div * ((uc.y - uc.x) * idx + (vc.y - vs.y) * idy + (wc.y - wb.y) * idz) +
                     ((fe - fm) * idx + (fn1 - fs1) * idy);
            const long long o = (long long)q * plane + out0;
            stcs2(up, o, make_double2(fma(c_up, fm, uc.x), fma(c_up, fe, uc.y)));
            stcs2(vp, o, make_double2(fma(c_up, fn0, vc.x), fma(c_up, fn1, vc.y)));
            wb = wc;
        }
        fb = fz; rc_b = rc; ph_b = ph;

        __syncthreads();                                  // every warp is done with this slot: refill it
        if (m + G::NSLOT <= m_last) issue_slab(q + G::NSLOT, slot, mask_of(m + G::NSLOT));
    }
}

}  // namespace flutas
