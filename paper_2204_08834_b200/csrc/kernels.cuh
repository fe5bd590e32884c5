// kernels.cuh -- the device kernels of the projection step (sm_100a, fp64).
//
//   splitting_rhs_kernel2  a1-a3  density from colour, p_hat, splitting RHS; also stores the
//                                 half-corrected velocity u' = u* - dt (1/rho_f - 1/rho0) grad p_hat
//                                 (register-marching form for small grids; kernels_rhs.cuh holds the production form)
//   fft_x_r2c_kernel       a4     real-to-complex transform along x (8 contiguous lines per CTA; nx outside 128..1024)
//   fft_x8_r2c/c2r_kernel  a4/a8  the degenerate length nx = 8
//   thomas_kernel          a6w    tridiagonal solve along z per (kx,ky), one thread per column (two sweeps; nz > 512)
//   thomas_singular_kernel a6w    the (0,0) column: pin the last unknown, remove the mean
//   fft_x_c2r_kernel       a8     complex-to-real transform along x, normalisation, writes p^(n+1)
//   correction_kernel      a9     u = u' - dt/rho0 grad p^(n+1)
//
// Row labels are those of SURVEY.md sec. 8(a); the paper passages are cited in include/flutas.h.
#pragma once
#include <cuda_runtime.h>

#include "common.cuh"
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

// ------------------------------------------------------------------------------------------------
// Register-marching form (small grids: nx < 128 or ny < 8).  2.5-D stencil: a block is (bx threads along x, 2 points
// each) x (ty rows of j); each thread marches over `kc` planes in z carrying, in registers, the centre and top values of
// rho_c and p_hat, the bottom-face flux and w below.  x neighbours come from warp shuffles (edge lanes load them),
// y neighbours from L1/L2.
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
// (1 - rho0/rho_f) for the face between cells of density ra and rb: one = 1, m2rho0 = -2 rho0
// (one = m2rho0 = 0 when rho1 == rho2: exactly 0, the constant-density projection)
__device__ __forceinline__ double flux_coef(double ra, double rb, double m2rho0, double one) {
    return fma(m2rho0, rcp_density(ra + rb), one);
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
    const double drho = g.rho1 - g.rho2, rho2 = g.rho2, one = g.flux_one, m2rho0 = -2.0 * g.rho0 * g.flux_one;
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
        fb.x = flux_coef(rc_b.x, rc_c.x, m2rho0, one) * ((ph_c.x - ph_b.x) * idz);
        fb.y = flux_coef(rc_b.y, rc_c.y, m2rho0, one) * ((ph_c.y - ph_b.y) * idz);
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
            ft.x = flux_coef(rc_c.x, rc_t.x, m2rho0, one) * ((ph_t.x - ph_c.x) * idz);
            ft.y = flux_coef(rc_c.y, rc_t.y, m2rho0, one) * ((ph_t.y - ph_c.y) * idz);
        }
        // ---- x faces: m between (i0, i0+1), e between (i0+1, i0+2), west face from the left lane
        double rc_e = __shfl_down_sync(0xffffffffu, rc_c.x, 1), ph_e = __shfl_down_sync(0xffffffffu, ph_c.x, 1);
        if (edge_r) { rc_e = rho_of(e_phi); ph_e = phat(e_p, e_po); }
        const double fm = flux_coef(rc_c.x, rc_c.y, m2rho0, one) * ((ph_c.y - ph_c.x) * idx);
        double fe = flux_coef(rc_c.y, rc_e, m2rho0, one) * ((ph_e - ph_c.y) * idx);
        if (g.wall_x && i0 + 2 == nx) fe = 0.0;
        double f_w = __shfl_up_sync(0xffffffffu, fe, 1), u_w = __shfl_up_sync(0xffffffffu, uc.y, 1);
        if (edge_l) {
            f_w = flux_coef(rho_of(w_phi), rc_c.x, m2rho0, one) * ((ph_c.x - phat(w_p, w_po)) * idx);
            u_w = w_u;
        }
        const bool wall_w = g.wall_x && i0 == 0, wall_e = g.wall_x && i0 + 2 == nx;
        const bool wall_s = g.wall_y && j == 0, wall_n = g.wall_y && j + 1 == ny;
        if (wall_w) { f_w = 0.0; u_w = 0.0; }
        // ---- y faces
        const double2 rc_n = rho2_of(r_nphi), ph_n = phat2(r_np, r_npo);
        const double2 rc_s = rho2_of(r_sphi), ph_s = phat2(r_sp, r_spo);
        double fn0 = flux_coef(rc_c.x, rc_n.x, m2rho0, one) * ((ph_n.x - ph_c.x) * idy);
        double fn1 = flux_coef(rc_c.y, rc_n.y, m2rho0, one) * ((ph_n.y - ph_c.y) * idy);
        if (wall_n) fn0 = fn1 = 0.0;
        double fs0 = flux_coef(rc_s.x, rc_c.x, m2rho0, one) * ((ph_c.x - ph_s.x) * idy);
        double fs1 = flux_coef(rc_s.y, rc_c.y, m2rho0, one) * ((ph_c.y - ph_s.y) * idy);
        if (wall_s) { fs0 = fs1 = 0.0; vs = make_double2(0.0, 0.0); }

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
    const bool east = g.wall_x && (i + 2 == g.nx), north = g.wall_y && (j + 1 == g.ny);   // wall faces pass through
    const double c = dt / g.rho0;
    auto ld2 = [](const double *f, long long a) { return *reinterpret_cast<const double2 *>(f + a); };
    const double2 pc = ld2(pn, q), pj = ld2(pn, qjp), pk = ld2(pn, qkp);
    const double pe = pn[qip];
    const double2 a = ld2(up, q), b = ld2(vp, q), d = ld2(wp, q);
    stcs2(u, q, make_double2(a.x - c * ((pc.y - pc.x) * g.inv_dx), east ? a.y : a.y - c * ((pe - pc.y) * g.inv_dx)));
    stcs2(v, q, north ? b : make_double2(b.x - c * ((pj.x - pc.x) * g.inv_dy), b.y - c * ((pj.y - pc.y) * g.inv_dy)));
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

// modes of the strided transform kernels (kernels_tma.cuh, kernels_y16.cuh)
enum { MODE_FWD = 0, MODE_INV = 1, MODE_SOLVE = 2, MODE_R2R_FWD = 3, MODE_R2R_INV = 4,
       MODE_FWD_SCAT = 5, MODE_SOLVE_SCAT = 6 };   // MODE_FWD / MODE_SOLVE whose last pass stores into the peers' arrays

// ------------------------------------------------------------------------------------------------
// z-slab decomposition over several GPUs: the two all-to-all
// transposes around the z stage are the STORE stage of the transform before them.  The last pass of a transform
// along a line whose positions are dealt out to the ranks in equal blocks writes position r of the line
//     to   base[r / rows_per_peer] + ((r % rows_per_peer) + lead) * row_stride + (outer + outer_off) * outer_stride + kx
// (base[]: the same array of every rank, mapped into this process: NVLink peer memory, or plain device memory when
// the ranks share a device).  halo = 1: the first / last position of every block is also written one row past the
// end / before the start of the neighbouring rank's block (the plane above / below a slab: what the velocity
// correction and the next step's right-hand side need from the neighbour), wrapping around when wrap = 1.
// ------------------------------------------------------------------------------------------------
constexpr int kMaxRanks = 16;
struct PeerScatter {
    int shift;                 // log2(rows_per_peer)
    int lead;                  // rows before a rank's block in its array (1 with halo planes, else 0)
    int halo, wrap, n_peers;
    long long row_stride, outer_stride, outer_off;   // of the destination arrays, in elements
    double2 *base[kMaxRanks];
};
// The descriptor is read where it is used, through a volatile pointer (shared memory in the transform kernels), so that
// it does not sit in registers across the butterfly passes (those kernels are at their register limit).
struct ScatterRegs {
    const volatile PeerScatter *d;
    __device__ __forceinline__ void load(const PeerScatter *desc) { d = desc; }
    __device__ __forceinline__ double2 *base(int peer) const { return d->base[peer]; }
};
__device__ __forceinline__ void scatter_store(const ScatterRegs &sc, int r, long long outer, int kx, double2 v) {
    const int shift = sc.d->shift, lead = sc.d->lead;
    const int rpp = 1 << shift, peer = r >> shift, loc = r & (rpp - 1);
    const long long row_stride = sc.d->row_stride;
    const long long off = (outer + sc.d->outer_off) * sc.d->outer_stride + kx;
    sc.base(peer)[(long long)(loc + lead) * row_stride + off] = v;
    if (sc.d->halo) {
        const int n_peers = sc.d->n_peers, wrap = sc.d->wrap;
        if (loc == 0) {                                    // the plane above the slab of the rank below
            const int q = peer > 0 ? peer - 1 : (wrap ? n_peers - 1 : -1);
            if (q >= 0) sc.base(q)[(long long)(rpp + lead) * row_stride + off] = v;
        }
        if (loc == rpp - 1) {                              // the plane below the slab of the rank above
            const int q = peer + 1 < n_peers ? peer + 1 : (wrap ? 0 : -1);
            if (q >= 0) sc.base(q)[off] = v;
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
// a4 / a8 for the degenerate length nx = 8: one thread per line, the 8-point transform in registers (a complex radix-8
// butterfly on real input: natural order in and out), rows written / read in natural kx order (kx = 0..4).
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128)
fft_x8_r2c_kernel(const double *__restrict__ rhs, double2 *__restrict__ spec, long long nlines, SpecRows sr) {
    const long long line = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (line >= nlines) return;
    double2 v[8];
#pragma unroll
    for (int e = 0; e < 4; ++e) {
        const double2 x = reinterpret_cast<const double2 *>(rhs + line * 8)[e];
        v[2 * e] = make_double2(x.x, 0.0);
        v[2 * e + 1] = make_double2(x.y, 0.0);
    }
    radix8<-1>(v);
    double2 *dst = spec + spec_row_offset(sr, line, 4 + 8);
#pragma unroll
    for (int k = 0; k <= 4; ++k) dst[k] = (k == 0 || k == 4) ? make_double2(v[k].x, 0.0) : v[k];
}

__global__ void __launch_bounds__(128)
fft_x8_c2r_kernel(const double2 *__restrict__ spec, double *__restrict__ out, double scale, long long nlines, SpecRows sr) {
    const long long line = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (line >= nlines) return;
    const double2 *src = spec + spec_row_offset(sr, line, 4 + 8);
    double2 v[8];
    v[0] = make_double2(src[0].x, 0.0);          // the imaginary parts of the DC and Nyquist columns do not enter
    v[4] = make_double2(src[4].x, 0.0);
#pragma unroll
    for (int k = 1; k < 4; ++k) { v[k] = src[k]; v[8 - k] = cconj(src[k]); }
    radix8<+1>(v);
#pragma unroll
    for (int e = 0; e < 4; ++e)
        reinterpret_cast<double2 *>(out + line * 8)[e] = make_double2(v[2 * e].x * scale, v[2 * e + 1].x * scale);
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
              const double *__restrict__ lam_x, const double *__restrict__ lam_y, double inv_dz2, long long plane,
              double end_coef /* 1 Neumann, 3 Dirichlet */, int has_null) {
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long ncol = (long long)pitch * ny;
    if (c >= ncol || (has_null && c == 0)) return;
    const int kx = (int)(c % pitch), jy = (int)(c / pitch);
    if (kx >= nxh) return;
    const double lam = lam_x[kx] + lam_y[jy];
    const double a = inv_dz2, b_end = -end_coef * inv_dz2 + lam, b_in = -2.0 * inv_dz2 + lam;
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
// re_only: with non-periodic x the imaginary part of column 0 is another (regular) mode and is left alone.
// sc != nullptr (z-slab decomposition): the solved column goes to the ranks that own its planes instead of back in place.
__global__ void thomas_singular_kernel(double2 *__restrict__ spec, long long col_stride, int nz,
                                       const double *__restrict__ coef /* inv_k, c'_k interleaved: 2 nz doubles */, int re_only,
                                       const PeerScatter *__restrict__ sc) {
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
    if (threadIdx.x == 1 && re_only) mean[1] = 0.0;
    if (threadIdx.x < (re_only ? 1 : 2)) {      // thread 0: real parts, thread 1: imaginary parts
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
    if (sc) {
        ScatterRegs scr;
        scr.load(sc);
        for (int k = threadIdx.x; k < nz; k += blockDim.x) scatter_store(scr, k, 0, 0, make_double2(dr[k] - mr, di[k] - mi));
        return;
    }
    for (int k = threadIdx.x; k < nz; k += blockDim.x)
        spec[(long long)k * col_stride] = make_double2(dr[k] - mr, di[k] - mi);
}

}  // namespace flutas
