// kernels_r2r.cuh -- the expansions along x for NON-PERIODIC x ("all the
// possible homogeneous pressure boundary conditions", "fast discrete cosine and sine transforms ...
// using real-to-complex / complex-to-real FFTs ..., with pre- and post-processing of the input and output signals").
//
// Neumann x (walls): the eigenvectors of the cell-centred second difference are cos(pi m (2i+1) / (2 nx)), so the
// forward expansion of a real line x[0..N) is the DCT-II  X[m] = 2 sum_i x[i] cos(pi m (2i+1) / (2N))  and the
// backward one its inverse; Dirichlet x: sin(pi (m+1) (2i+1) / (2N)), the DST-II, which is the DCT-II of
// (-1)^i x[i] read backwards (X_s[m] = X'[N-1-m]).  Both are computed with the machinery of the periodic case
// (fft_core.cuh: an N/2-point complex FFT of a packed real line + the real-FFT split), wrapped in
//   pre :  v[n] = x[2n], v[N-1-n] = (+-) x[2n+1]   (the even samples, then the odd samples backwards),   V = FFT_N(v)
//   post:  X[k] = 2 Re(w_k V[k]),  X[N-k] = -2 Im(w_k V[k]),   w_k = e^{-i pi k / (2N)},  k = 0 .. N/2
// fused into the load of the tile and into the split, so a line crosses HBM once in and once out as before.
//
// Output layout ("split columns"): N/2 complex columns per line, column k = (X[k], X[N-k]) for k >= 1 and column 0 =
// (X[0], X[N/2]): the real and the imaginary part of a column are two DIFFERENT modes along x.  Every later stage is
// real-linear per component (cosine / sine / half-complex expansion along y, elimination along z with real
// coefficients), so it treats a column as a pair of independent real numbers with their own eigenvalues
// (lam_x2[2 k + component]).
//
// These are staged kernels (8 contiguous lines per CTA, one tile in shared memory beside a landing area), not the
// persistent bulk-copy-fed form of kernels_x.cuh: first version of a new row, measured in DESIGN.md sec. 6.
#pragma once
#include "kernels.cuh"

namespace flutas {

constexpr double kSqrt2 = 1.41421356237309504880168872420969807857;

// split of the packed transform + the cosine post-twiddle, in place: Z[q], Z[N2-q] -> columns q, N2-q
template <int N2>
__device__ __forceinline__ void r2r_post_item(double2 *s, int q, int l, const double2 *__restrict__ tw /* e^{-2 pi i m / N} */,
                                              const double2 *__restrict__ wq /* e^{-i pi k / (2N)} */) {
    if (q == 0) {
        const double2 z = s[tile_index<8, true>(0, l)];
        s[tile_index<8, true>(0, l)] = make_double2(2.0 * (z.x + z.y), kSqrt2 * (z.x - z.y));   // (X[0], X[N/2])
    } else if (2 * q == N2) {
        const int ia = tile_index<8, true>(pos_of_freq<N2>(q), l);
        const double2 y = cmul(wq[q], cconj(s[ia]));                                       // w_q V[q], V[q] = conj Z[q]
        s[ia] = make_double2(2.0 * y.x, -2.0 * y.y);
    } else {
        const int ia = tile_index<8, true>(pos_of_freq<N2>(q), l);
        const int ib = tile_index<8, true>(pos_of_freq<N2>(N2 - q), l);
        const double2 zk = s[ia], zc = cconj(s[ib]);
        const double2 a = cadd(zk, zc), t = cmul(tw[q], csub(zk, zc));
        const double2 va = make_double2(0.5 * (a.x + t.y), 0.5 * (a.y - t.x));             // V[q]
        const double2 vb = make_double2(0.5 * (a.x - t.y), -0.5 * (a.y + t.x));            // V[N2 - q]
        const double2 ya = cmul(wq[q], va), yb = cmul(wq[N2 - q], vb);
        s[ia] = make_double2(2.0 * ya.x, -2.0 * ya.y);
        s[ib] = make_double2(2.0 * yb.x, -2.0 * yb.y);
    }
}

// the inverse, up to the scale of the unnormalised inverse FFT: columns q, N2-q -> Z'[q], Z'[N2-q]
template <int N2>
__device__ __forceinline__ void r2r_pre_item(double2 *s, int q, int l, const double2 *__restrict__ tw,
                                             const double2 *__restrict__ wq) {
    if (q == 0) {
        const double2 c = s[tile_index<8, true>(0, l)];
        const double v0 = 0.5 * c.x, vn = c.y * (0.5 * kSqrt2);                            // V[0], V[N/2] (both real)
        s[tile_index<8, true>(0, l)] = make_double2(v0 + vn, v0 - vn);
    } else if (2 * q == N2) {
        const int ia = tile_index<8, true>(pos_of_freq<N2>(q), l);
        const double2 c = s[ia];
        const double2 v = cmulc(make_double2(0.5 * c.x, -0.5 * c.y), wq[q]);               // V = conj(w_q) (X[q] - i X[N-q]) / 2
        s[ia] = make_double2(2.0 * v.x, -2.0 * v.y);
    } else {
        const int ia = tile_index<8, true>(pos_of_freq<N2>(q), l);
        const int ib = tile_index<8, true>(pos_of_freq<N2>(N2 - q), l);
        const double2 ca = s[ia], cb = s[ib];
        const double2 xk = cmulc(make_double2(0.5 * ca.x, -0.5 * ca.y), wq[q]);            // V[q]
        const double2 xc = cconj(cmulc(make_double2(0.5 * cb.x, -0.5 * cb.y), wq[N2 - q]));   // conj V[N2 - q]
        const double2 a = cadd(xk, xc), sv = cmulc(csub(xk, xc), tw[q]);
        s[ia] = make_double2(a.x - sv.y, a.y + sv.x);
        s[ib] = make_double2(a.x + sv.y, sv.x - a.y);
    }
}

// ------------------------------------------------------------------------------------------------
// forward: 8 real lines -> 8 rows of N2 split columns (natural order k = 0 .. N2-1)
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT, 1)
fft_x_r2r_fwd_kernel(const double *__restrict__ rhs, double2 *__restrict__ spec, const double2 *__restrict__ tw,
                     const double2 *__restrict__ wq, int neg_odd, SpecRows sr) {
    extern __shared__ double2 smem[];
    double2 *s = smem;                                           // N2 positions x 8 lines, swizzled
    double *land = reinterpret_cast<double *>(smem + 8 * N2);    // 8 lines x N reals as they are in memory
    constexpr int N = 2 * N2, PITCH = N2 + 8;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    const double2 *src = reinterpret_cast<const double2 *>(rhs) + line0 * N2;
    batched_copy<8 * N2, NT, 8, double2>(
        tid, [&](int idx) { return src[idx]; },
        [&](int idx, double2 val) { reinterpret_cast<double2 *>(land)[idx] = val; });
    __syncthreads();
    // z[i] = (v[2i], v[2i+1]) of the reordered line: even samples forwards, odd samples backwards
    for (int idx = tid; idx < 8 * N2; idx += NT) {
        const int i = idx % N2, l = idx / N2;
        const double *L = land + l * N;
        double a, b;
        if (i < N2 / 2) { a = L[4 * i]; b = L[4 * i + 2]; }
        else {
            a = L[2 * N - 4 * i - 1]; b = L[2 * N - 4 * i - 3];
            if (neg_odd) { a = -a; b = -b; }
        }
        s[tile_index<8, true>(i, l)] = make_double2(a, b);
    }
    __syncthreads();
    tile_fft<N2, 8, true, NT, -1>(s, tw, 2, tid);
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) r2r_post_item<N2>(s, item / 8, item % 8, tw, wq);
    __syncthreads();
    double2 *dst = spec + spec_row_offset(sr, line0, PITCH);
    for (int idx = tid; idx < 8 * PITCH; idx += NT) {
        const int l = idx / PITCH, k = idx % PITCH;
        if (k < N2) dst[idx] = s[tile_index<8, true>(pos_of_freq<N2>(k), l)];
    }
}

// ------------------------------------------------------------------------------------------------
// backward: 8 rows of split columns -> 8 real lines, scaled
// ------------------------------------------------------------------------------------------------
template <int N2, int NT>
__global__ void __launch_bounds__(NT, 1)
fft_x_r2r_inv_kernel(const double2 *__restrict__ spec, double *__restrict__ out, const double2 *__restrict__ tw,
                     const double2 *__restrict__ wq, int neg_odd, double scale, SpecRows sr) {
    extern __shared__ double2 smem[];
    double2 *s = smem;
    double *land = reinterpret_cast<double *>(smem + 8 * N2);
    constexpr int N = 2 * N2, PITCH = N2 + 8;
    const int tid = threadIdx.x;
    const long long line0 = (long long)blockIdx.x * 8;
    const double2 *src = spec + spec_row_offset(sr, line0, PITCH);
    batched_copy<8 * PITCH, NT, 9, double2>(
        tid, [&](int idx) { return src[idx]; },
        [&](int idx, double2 val) {
            const int l = idx / PITCH, k = idx % PITCH;
            if (k < N2) s[tile_index<8, true>(pos_of_freq<N2>(k), l)] = val;
        });
    __syncthreads();
    for (int item = tid; item < 8 * (N2 / 2 + 1); item += NT) r2r_pre_item<N2>(s, item / 8, item % 8, tw, wq);
    __syncthreads();
    tile_fft<N2, 8, true, NT, +1>(s, tw, 2, tid);
    __syncthreads();
    const double so = neg_odd ? -scale : scale;
    for (int idx = tid; idx < 8 * N2; idx += NT) {
        const int i = idx % N2, l = idx / N2;
        const double2 z = s[tile_index<8, true>(i, l)];
        double *L = land + l * N;
        if (i < N2 / 2) { L[4 * i] = z.x * scale; L[4 * i + 2] = z.y * scale; }
        else { L[2 * N - 4 * i - 1] = z.x * so; L[2 * N - 4 * i - 3] = z.y * so; }
    }
    __syncthreads();
    double2 *dst = reinterpret_cast<double2 *>(out) + line0 * N2;
    for (int idx = tid; idx < 8 * N2; idx += NT) dst[idx] = reinterpret_cast<const double2 *>(land)[idx];
}

}  // namespace flutas
