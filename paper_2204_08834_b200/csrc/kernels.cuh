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

struct GridParams {
    int nx, ny, nz, wall;
    double inv_dx, inv_dy, inv_dz;
    double rho1, rho2, rho0;
};

// ------------------------------------------------------------------------------------------------
// a1-a3: fused density + splitting right-hand side (eqs. 2, 16, 17)
// One thread per grid point.  Reads u*, v*, w*, phi, p, p_old; writes rhs and u', v', w'.
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
splitting_rhs_kernel(GridParams g, double dt, const double *__restrict__ u, const double *__restrict__ v,
                     const double *__restrict__ w, const double *__restrict__ phi,
                     const double *__restrict__ p, const double *__restrict__ po,
                     double *__restrict__ rhs, double *__restrict__ up, double *__restrict__ vp,
                     double *__restrict__ wp) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int i = (int)(q % g.nx);
    const long long r = q / g.nx;
    const int j = (int)(r % g.ny), k = (int)(r / g.ny);
    const long long sx = 1, sy = g.nx, sz = (long long)g.nx * g.ny;
    const long long qip = (i + 1 == g.nx) ? q - (g.nx - 1) * sx : q + sx;
    const long long qim = (i == 0) ? q + (g.nx - 1) * sx : q - sx;
    const long long qjp = (j + 1 == g.ny) ? q - (g.ny - 1) * sy : q + sy;
    const long long qjm = (j == 0) ? q + (g.ny - 1) * sy : q - sy;
    const long long qkp = (k + 1 == g.nz) ? q - (g.nz - 1) * sz : q + sz;
    const long long qkm = (k == 0) ? q + (g.nz - 1) * sz : q - sz;
    const bool top = g.wall && (k + 1 == g.nz), bot = g.wall && (k == 0);

    auto rho_c = [&](long long a) { const double f = phi[a]; return g.rho1 * f + g.rho2 * (1.0 - f); };
    auto p_hat = [&](long long a) { return 2.0 * p[a] - po[a]; };

    const double rc = rho_c(q), ph = p_hat(q);
    // east / west faces
    const double r_e = 1.0 / (0.5 * (rc + rho_c(qip))), r_w = 1.0 / (0.5 * (rc + rho_c(qim)));
    const double g_e = (p_hat(qip) - ph) * g.inv_dx, g_w = (ph - p_hat(qim)) * g.inv_dx;
    // north / south
    const double r_n = 1.0 / (0.5 * (rc + rho_c(qjp))), r_s = 1.0 / (0.5 * (rc + rho_c(qjm)));
    const double g_n = (p_hat(qjp) - ph) * g.inv_dy, g_s = (ph - p_hat(qjm)) * g.inv_dy;
    // top / bottom (wall faces carry zero flux)
    const double r_t = top ? 0.0 : 1.0 / (0.5 * (rc + rho_c(qkp)));
    const double r_b = bot ? 0.0 : 1.0 / (0.5 * (rc + rho_c(qkm)));
    const double g_t = top ? 0.0 : (p_hat(qkp) - ph) * g.inv_dz;
    const double g_b = bot ? 0.0 : (ph - p_hat(qkm)) * g.inv_dz;

    const double f_e = (1.0 - g.rho0 * r_e) * g_e, f_w = (1.0 - g.rho0 * r_w) * g_w;
    const double f_n = (1.0 - g.rho0 * r_n) * g_n, f_s = (1.0 - g.rho0 * r_s) * g_s;
    const double f_t = (1.0 - g.rho0 * r_t) * g_t, f_b = (1.0 - g.rho0 * r_b) * g_b;

    const double uc = u[q], vc = v[q], wc = w[q];
    const double um = u[qim], vm = v[qjm], wm = bot ? 0.0 : w[qkm];
    const double div_u = (uc - um) * g.inv_dx + (vc - vm) * g.inv_dy + (wc - wm) * g.inv_dz;
    const double div_f = (f_e - f_w) * g.inv_dx + (f_n - f_s) * g.inv_dy + (f_t - f_b) * g.inv_dz;
    rhs[q] = g.rho0 / dt * div_u + div_f;

    const double inv_rho0 = 1.0 / g.rho0;
    up[q] = uc - dt * ((r_e - inv_rho0) * g_e);
    vp[q] = vc - dt * ((r_n - inv_rho0) * g_n);
    wp[q] = top ? wc : wc - dt * ((r_t - inv_rho0) * g_t);
}

// ------------------------------------------------------------------------------------------------
// a9: u = u' - dt/rho0 grad p^(n+1)   (eq. 18; p^(n+1) was already stored by a8)
// ------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
correction_kernel(GridParams g, double dt, const double *__restrict__ pn, const double *__restrict__ up,
                  const double *__restrict__ vp, const double *__restrict__ wp, double *__restrict__ u,
                  double *__restrict__ v, double *__restrict__ w) {
    const long long n = (long long)g.nx * g.ny * g.nz;
    const long long q = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (q >= n) return;
    const int i = (int)(q % g.nx);
    const long long r = q / g.nx;
    const int j = (int)(r % g.ny), k = (int)(r / g.ny);
    const long long sy = g.nx, sz = (long long)g.nx * g.ny;
    const long long qip = (i + 1 == g.nx) ? q - (g.nx - 1) : q + 1;
    const long long qjp = (j + 1 == g.ny) ? q - (g.ny - 1) * sy : q + sy;
    const long long qkp = (k + 1 == g.nz) ? q - (g.nz - 1) * sz : q + sz;
    const bool top = g.wall && (k + 1 == g.nz);
    const double c = dt / g.rho0;
    const double pc = pn[q];
    u[q] = up[q] - c * ((pn[qip] - pc) * g.inv_dx);
    v[q] = vp[q] - c * ((pn[qjp] - pc) * g.inv_dy);
    w[q] = top ? wp[q] : wp[q] - c * ((pn[qkp] - pc) * g.inv_dz);
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

template <int N, int C, int MODE, int NT>
__global__ void __launch_bounds__(NT) fft_strided_kernel(StridedArgs a) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    const int tid = threadIdx.x;
    const int tx = blockIdx.x % a.n_tiles_x, outer = blockIdx.x / a.n_tiles_x;
    const int l = tid % C;
    const int kx = tx * C + l;
    const bool valid = kx < a.nxh;
    double2 *gp = a.data + (long long)outer * a.outer_stride + kx;

#pragma unroll 8
    for (int r = tid / C; r < N; r += NT / C)
        s[r * C + l] = valid ? gp[(long long)r * a.row_stride] : make_double2(0.0, 0.0);
    __syncthreads();

    if (MODE == MODE_FWD) {
        tile_fft<N, C, false, NT, -1>(s, a.tw, 1, tid);
    } else if (MODE == MODE_INV) {
        tile_fft<N, C, false, NT, +1>(s, a.tw, 1, tid);
    } else {
        // forward passes 1..P-1 through shared memory
        constexpr int P = Fact<N>::P;
#pragma unroll
        for (int p = 1; p < P; ++p) {
            for (int t = tid / C; t < N / 8; t += NT / C) {
                int pos[8], n2;
                double2 v[8];
                pass_positions<N>(p, t, pos, n2);
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] = s[pos[e] * C + l];
                fwd_pass_regs<N>(p, n2, v, a.tw, 1);
#pragma unroll
                for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
            }
            __syncthreads();
        }
        // last forward pass, division by the eigenvalue sum, first inverse pass: all in registers
        const double lam_xy = a.lam_x[valid ? kx : 0] + a.lam_outer[outer];
        for (int t = tid / C; t < N / 8; t += NT / C) {
            int pos[8], n2;
            double2 v[8];
            pass_positions<N>(P, t, pos, n2);
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = s[pos[e] * C + l];
            fwd_pass_regs<N>(P, n2, v, a.tw, 1);
#pragma unroll
            for (int e = 0; e < 8; ++e) {
                const double den = lam_xy + a.lam_pos[pos[e]];
                const double inv = (den == 0.0) ? 0.0 : 1.0 / den;     // the (0,0,0) mode is dropped (zero-mean gauge)
                v[e] = cscale(v[e], inv);
            }
            inv_pass_regs<N>(P, n2, v, a.tw, 1);
#pragma unroll
            for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
        }
        if (P > 1) __syncthreads();
#pragma unroll
        for (int p = P - 1; p >= 1; --p) {
            for (int t = tid / C; t < N / 8; t += NT / C) {
                int pos[8], n2;
                double2 v[8];
                pass_positions<N>(p, t, pos, n2);
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] = s[pos[e] * C + l];
                inv_pass_regs<N>(p, n2, v, a.tw, 1);
#pragma unroll
                for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
            }
            if (p > 1) __syncthreads();
        }
    }
    __syncthreads();

    if (valid) {
#pragma unroll 8
        for (int r = tid / C; r < N; r += NT / C) gp[(long long)r * a.row_stride] = s[r * C + l];
    }
}

// ------------------------------------------------------------------------------------------------
// a4: real-to-complex along x.  CTA = 8 consecutive lines (contiguous in memory), N2 = nx/2.
// Output row (line) layout: positions 0..N2-1 in permuted order, Nyquist at N2; row pitch `pitch`.
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT)
fft_x_r2c_kernel(const double *__restrict__ rhs, double2 *__restrict__ spec, int pitch,
                 const double2 *__restrict__ tw /* e^{-2 pi i m / nx} */) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    const double2 *src = reinterpret_cast<const double2 *>(rhs) + line0 * N2;
#pragma unroll 4
    for (int idx = tid; idx < 8 * N2; idx += NT) {
        const int l = idx / N2, i = idx % N2;
        s[tile_index<8, true>(i, l)] = src[idx];
    }
    __syncthreads();
    tile_fft<N2, 8, true, NT, -1>(s, tw, 2, tid);
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) r2c_post_item<N2, 8, true>(s, item / 8, item % 8, tw);
    __syncthreads();
    for (int l = 0; l < 8; ++l) {
        double2 *dst = spec + (line0 + l) * pitch;
        for (int pos = tid; pos <= N2; pos += NT) dst[pos] = s[tile_index<8, true>(pos, l)];
    }
}

// ------------------------------------------------------------------------------------------------
// a8: complex-to-real along x with the normalisation of the whole transform chain; writes p^(n+1).
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT)
fft_x_c2r_kernel(const double2 *__restrict__ spec, double *__restrict__ out, int pitch,
                 const double2 *__restrict__ tw, double scale) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    for (int l = 0; l < 8; ++l) {
        const double2 *src = spec + (line0 + l) * pitch;
        for (int pos = tid; pos <= N2; pos += NT) s[tile_index<8, true>(pos, l)] = src[pos];
    }
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) c2r_pre_item<N2, 8, true>(s, item / 8, item % 8, tw);
    __syncthreads();
    tile_fft<N2, 8, true, NT, +1>(s, tw, 2, tid);
    __syncthreads();
    double2 *dst = reinterpret_cast<double2 *>(out) + line0 * N2;
#pragma unroll 4
    for (int idx = tid; idx < 8 * N2; idx += NT) {
        const int l = idx / N2, i = idx % N2;
        dst[idx] = cscale(s[tile_index<8, true>(i, l)], scale);
    }
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
              const double *__restrict__ lam_x, const double *__restrict__ lam_y, double inv_dz2) {
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
        const long long q = c + (long long)k * ncol;
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
        const long long q = c + (long long)k * ncol;
        const double2 dk = spec[q];
        const double ck = cp[q];
        x = make_double2(dk.x - ck * x.x, dk.y - ck * x.y);
        spec[q] = x;
    }
}

// The (kx,ky) = (0,0) column: lam_xy = 0, the system is singular (pure Neumann).  Eliminate rows
// 0..nz-2, pin x_{nz-1} = 0, back-substitute, then remove the mean over k (zero-mean gauge, R5).
__global__ void thomas_singular_kernel(double2 *__restrict__ spec, long long col_stride, int nz, double inv_dz2) {
    extern __shared__ double sm[];
    double *dr = sm, *di = sm + nz, *cpv = sm + 2 * nz;
    for (int k = threadIdx.x; k < nz; k += blockDim.x) {
        const double2 d = spec[(long long)k * col_stride];
        dr[k] = d.x;
        di[k] = d.y;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        const double a = inv_dz2, b_end = -inv_dz2, b_in = -2.0 * inv_dz2;
        double inv = 1.0 / b_end;
        cpv[0] = a * inv;
        dr[0] *= inv;
        di[0] *= inv;
        for (int k = 1; k <= nz - 2; ++k) {
            inv = 1.0 / (b_in - a * cpv[k - 1]);
            cpv[k] = a * inv;
            dr[k] = (dr[k] - a * dr[k - 1]) * inv;
            di[k] = (di[k] - a * di[k - 1]) * inv;
        }
        dr[nz - 1] = 0.0;
        di[nz - 1] = 0.0;
        for (int k = nz - 2; k >= 0; --k) {
            dr[k] = dr[k] - cpv[k] * dr[k + 1];
            di[k] = di[k] - cpv[k] * di[k + 1];
        }
        double mr = 0.0, mi = 0.0;
        for (int k = 0; k < nz; ++k) { mr += dr[k]; mi += di[k]; }
        cpv[0] = mr / nz;
        cpv[1] = mi / nz;     // nz >= 2
    }
    __syncthreads();
    const double mr = cpv[0], mi = cpv[1];
    for (int k = threadIdx.x; k < nz; k += blockDim.x)
        spec[(long long)k * col_stride] = make_double2(dr[k] - mr, di[k] - mi);
}

}  // namespace flutas
