// fft_core.cuh -- radix-8 in-register butterflies and the in-place, permuted-order FFT passes
// used by every transform kernel of the Poisson solve (Fourier expansion
// along x and y, and along z in the triply periodic case).
//
// Design:
//  * A tile holds C lines of length N interleaved in shared memory: element (pos, l) of line l is
//    at s[pos*C + slot(pos,l)], 16 bytes each (double2 = re, im).  With C = 8 a quarter-warp that
//    touches the 8 lines of one position covers one 128-byte row: every access pattern of every
//    pass is bank-conflict free without padding.  slot() optionally XOR-swizzles the line index
//    with the position so that the x-direction kernels can also fill the tile with lanes running
//    along pos (coalesced in global memory) without conflicts.
//  * The forward transform is decimation-in-frequency: pass p does radix-R_p butterflies on
//    elements M_p apart, then multiplies by W^(n2*k1); each thread keeps 8 elements in registers
//    and writes them back where it read them (in place, one __syncthreads per exchange).
//    The result is left in digit-reversed ("permuted") order: position pos holds frequency
//    freq_of_pos(pos).  The inverse transform is the exact transpose (decimation-in-time):
//    it takes permuted input and returns natural order.  Nothing is ever re-sorted: the spectral
//    arrays of the solver live in permuted order in all three directions and the eigenvalue
//    tables are permuted once on the host.
//  * N = 8^a * r, r in {1,2,4}: a radix-8 passes followed (forward) by one pass of 8/r
//    independent radix-r butterflies per thread.
//
// Everything here is __host__ __device__ and free of CUDA intrinsics so that the same code is
// exercised by a host emulation harness during development.
#pragma once

#ifdef __CUDACC__
#define FL_HD __host__ __device__ __forceinline__
#define FL_CE __host__ __device__ constexpr
#else
#define FL_HD inline
#define FL_CE constexpr
struct double2 { double x, y; };
static inline double2 make_double2(double x, double y) { double2 r; r.x = x; r.y = y; return r; }
#endif

namespace flutas {

constexpr double kInvSqrt2 = 0.70710678118654752440084436210484903928;

FL_HD double2 cadd(double2 a, double2 b) { return make_double2(a.x + b.x, a.y + b.y); }
FL_HD double2 csub(double2 a, double2 b) { return make_double2(a.x - b.x, a.y - b.y); }
FL_HD double2 cmul(double2 a, double2 b) { return make_double2(a.x * b.x - a.y * b.y, a.x * b.y + a.y * b.x); }
FL_HD double2 cmulc(double2 a, double2 b) {  // a * conj(b)
    return make_double2(a.x * b.x + a.y * b.y, a.y * b.x - a.x * b.y);
}
FL_HD double2 cconj(double2 a) { return make_double2(a.x, -a.y); }
FL_HD double2 cscale(double2 a, double s) { return make_double2(a.x * s, a.y * s); }
// multiply by -i (DIR = -1, forward) or by +i (DIR = +1, inverse)
template <int DIR> FL_HD double2 mul_dir_i(double2 a) {
    return DIR < 0 ? make_double2(a.y, -a.x) : make_double2(-a.y, a.x);
}

FL_CE int ilog2(int n) { return n <= 1 ? 0 : 1 + ilog2(n / 2); }
FL_CE int ipow8(int p) { return p <= 0 ? 1 : 8 * ipow8(p - 1); }

// compile-time factorisation N = 8^(P-1) * R_last
template <int N> struct Fact {
    static_assert(N >= 8 && (N & (N - 1)) == 0, "FFT length must be a power of two >= 8");
    static constexpr int LOG = ilog2(N);
    static constexpr int P = (LOG + 2) / 3;                  // number of passes
    static constexpr int RLAST = 1 << (LOG - 3 * (P - 1));   // 2, 4 or 8
};

// radix of pass p (1-based) and the stride M_p = N / (R_1 ... R_p)
template <int N> FL_HD int pass_radix(int p) { return p < Fact<N>::P ? 8 : Fact<N>::RLAST; }
template <int N> FL_HD int pass_stride(int p) { return p < Fact<N>::P ? N / ipow8(p) : 1; }

// position (storage index after the forward transform) <-> frequency.  All radices are powers of two, so
// the digit exchange is shifts and masks (no division): digit p (p < P) of the frequency is 3 bits wide and
// weighs N / 8^p in the position; the last digit (radix RLAST) weighs 1.
template <int N> FL_HD int freq_of_pos(int pos) {
    constexpr int P = Fact<N>::P;
    int k = (pos & (Fact<N>::RLAST - 1)) << (3 * (P - 1));
#pragma unroll
    for (int p = 1; p < P; ++p) k += ((pos >> (Fact<N>::LOG - 3 * p)) & 7) << (3 * (p - 1));
    return k;
}
template <int N> FL_HD int pos_of_freq(int k) {
    constexpr int P = Fact<N>::P;
    int pos = k >> (3 * (P - 1));
#pragma unroll
    for (int p = 1; p < P; ++p) pos += ((k >> (3 * (p - 1))) & 7) << (Fact<N>::LOG - 3 * p);
    return pos;
}

// ---- butterflies: v[k] <- sum_n v[n] * exp(DIR * 2 pi i n k / R), natural order in and out -------

template <int DIR> FL_HD void radix2(double2 &a, double2 &b) {
    double2 t = csub(a, b);
    a = cadd(a, b);
    b = t;
}

template <int DIR> FL_HD void radix4(double2 &c0, double2 &c1, double2 &c2, double2 &c3) {
    double2 s0 = cadd(c0, c2), s1 = csub(c0, c2), s2 = cadd(c1, c3), s3 = mul_dir_i<DIR>(csub(c1, c3));
    c0 = cadd(s0, s2);
    c2 = csub(s0, s2);
    c1 = cadd(s1, s3);
    c3 = csub(s1, s3);
}

template <int DIR> FL_HD void radix8(double2 *v) {
    double2 a0 = cadd(v[0], v[4]), a1 = cadd(v[1], v[5]), a2 = cadd(v[2], v[6]), a3 = cadd(v[3], v[7]);
    double2 b0 = csub(v[0], v[4]), b1 = csub(v[1], v[5]), b2 = csub(v[2], v[6]), b3 = csub(v[3], v[7]);
    // b_n *= W8^n, W8 = exp(DIR * 2 pi i / 8)
    if (DIR < 0) {
        b1 = make_double2((b1.x + b1.y) * kInvSqrt2, (b1.y - b1.x) * kInvSqrt2);
        b2 = make_double2(b2.y, -b2.x);
        b3 = make_double2((b3.y - b3.x) * kInvSqrt2, (-b3.x - b3.y) * kInvSqrt2);
    } else {
        b1 = make_double2((b1.x - b1.y) * kInvSqrt2, (b1.x + b1.y) * kInvSqrt2);
        b2 = make_double2(-b2.y, b2.x);
        b3 = make_double2((-b3.x - b3.y) * kInvSqrt2, (b3.x - b3.y) * kInvSqrt2);
    }
    radix4<DIR>(a0, a1, a2, a3);   // even outputs
    radix4<DIR>(b0, b1, b2, b3);   // odd outputs
    v[0] = a0; v[2] = a1; v[4] = a2; v[6] = a3;
    v[1] = b0; v[3] = b1; v[5] = b2; v[7] = b3;
}

// a * W16^M, W16 = exp(DIR * 2 pi i / 16), for the exponents the radix-16 butterfly needs
constexpr double kCosPi8 = 0.92387953251128675612818318939678828682;
constexpr double kSinPi8 = 0.38268343236508977172845998403039886676;
template <int DIR, int M> FL_HD double2 mul_w16(double2 a) {
    // W16^M = (wr, DIR * wi) with (wr, wi) = (cos, sin)(2 pi M / 16)
    constexpr double wr = M == 1 ? kCosPi8 : M == 2 ? kInvSqrt2 : M == 3 ? kSinPi8 : M == 4 ? 0.0 : M == 6 ? -kInvSqrt2 : -kCosPi8;
    constexpr double wi = M == 1 ? kSinPi8 : M == 2 ? kInvSqrt2 : M == 3 ? kCosPi8 : M == 4 ? 1.0 : M == 6 ? kInvSqrt2 : -kSinPi8;
    static_assert(M == 1 || M == 2 || M == 3 || M == 4 || M == 6 || M == 9, "exponent not used by radix16");
    if (M == 4) return mul_dir_i<DIR>(a);
    if (M == 2) return DIR < 0 ? make_double2((a.x + a.y) * kInvSqrt2, (a.y - a.x) * kInvSqrt2)
                               : make_double2((a.x - a.y) * kInvSqrt2, (a.x + a.y) * kInvSqrt2);
    if (M == 6) return DIR < 0 ? make_double2((a.y - a.x) * kInvSqrt2, (-a.x - a.y) * kInvSqrt2)
                               : make_double2((-a.x - a.y) * kInvSqrt2, (a.x - a.y) * kInvSqrt2);
    const double si = DIR < 0 ? -wi : wi;
    return make_double2(a.x * wr - a.y * si, a.x * si + a.y * wr);
}

// 16-point butterfly, natural order in and out: n = 4 n1 + n0, k = k0 + 4 k1,
//   X[k0 + 4 k1] = sum_n0 W4^(n0 k1) [ W16^(n0 k0) sum_n1 W4^(n1 k0) x[4 n1 + n0] ]
template <int DIR> FL_HD void radix16(double2 *v) {
    radix4<DIR>(v[0], v[4], v[8], v[12]);      // slot n0 + 4 k0
    radix4<DIR>(v[1], v[5], v[9], v[13]);
    radix4<DIR>(v[2], v[6], v[10], v[14]);
    radix4<DIR>(v[3], v[7], v[11], v[15]);
    v[5] = mul_w16<DIR, 1>(v[5]);   v[9] = mul_w16<DIR, 2>(v[9]);    v[13] = mul_w16<DIR, 3>(v[13]);
    v[6] = mul_w16<DIR, 2>(v[6]);   v[10] = mul_w16<DIR, 4>(v[10]);  v[14] = mul_w16<DIR, 6>(v[14]);
    v[7] = mul_w16<DIR, 3>(v[7]);   v[11] = mul_w16<DIR, 6>(v[11]);  v[15] = mul_w16<DIR, 9>(v[15]);
    radix4<DIR>(v[0], v[1], v[2], v[3]);       // slot 4 k0 + k1 holds X[k0 + 4 k1]
    radix4<DIR>(v[4], v[5], v[6], v[7]);
    radix4<DIR>(v[8], v[9], v[10], v[11]);
    radix4<DIR>(v[12], v[13], v[14], v[15]);
    double2 t;                                   // 4 x 4 transpose of the slots -> natural order
    t = v[1]; v[1] = v[4]; v[4] = t;    t = v[2]; v[2] = v[8]; v[8] = t;     t = v[3]; v[3] = v[12]; v[12] = t;
    t = v[6]; v[6] = v[9]; v[9] = t;    t = v[7]; v[7] = v[13]; v[13] = t;   t = v[11]; v[11] = v[14]; v[14] = t;
}

// the small last pass: 8/R independent radix-R butterflies on contiguous groups of R
template <int DIR, int R> FL_HD void small_groups(double2 *v) {
    if (R == 8) radix8<DIR>(v);
    else if (R == 4) { radix4<DIR>(v[0], v[1], v[2], v[3]); radix4<DIR>(v[4], v[5], v[6], v[7]); }
    else { radix2<DIR>(v[0], v[1]); radix2<DIR>(v[2], v[3]); radix2<DIR>(v[4], v[5]); radix2<DIR>(v[6], v[7]); }
}

// ---- tile addressing ----------------------------------------------------------------------------

template <int C, bool SWZ> FL_HD int tile_index(int pos, int l) {
    return pos * C + (SWZ ? (l ^ (pos & (C - 1))) : l);
}

// ---- one pass of one butterfly --------------------------------------------------------------------
// t in [0, N/8): which group of 8 elements; fills pos[8] with the element positions of pass p.
template <int N> FL_HD void pass_positions(int p, int t, int *pos, int &n2) {
    if (p < Fact<N>::P || Fact<N>::RLAST == 8) {
        const int m = pass_stride<N>(p);
        const int b = t / m;
        n2 = t - b * m;
        const int base = b * 8 * m + n2;
        for (int e = 0; e < 8; ++e) pos[e] = base + e * m;
    } else {
        n2 = 0;
        for (int e = 0; e < 8; ++e) pos[e] = 8 * t + e;
    }
}

// forward (DIF) pass p on registers v: butterfly, then twiddle by W_N^(8^(p-1) * n2 * k1).
// tw[m * tws] = exp(-2 pi i m / N)   (tws lets a longer table serve a shorter transform)
template <int N> FL_HD void fwd_pass_regs(int p, int n2, double2 *v, const double2 *tw, int tws) {
    if (p < Fact<N>::P || Fact<N>::RLAST == 8) {
        radix8<-1>(v);
        if (pass_stride<N>(p) > 1) {
            const int step = ipow8(p - 1) * n2 * tws;
            for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmul(v[k1], tw[step * k1]);
        }
    } else {
        small_groups<-1, Fact<N>::RLAST>(v);
    }
}

// inverse (DIT) pass p: conjugate twiddle, then the conjugate butterfly. Passes run p = P..1.
template <int N> FL_HD void inv_pass_regs(int p, int n2, double2 *v, const double2 *tw, int tws) {
    if (p < Fact<N>::P || Fact<N>::RLAST == 8) {
        if (pass_stride<N>(p) > 1) {
            const int step = ipow8(p - 1) * n2 * tws;
            for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmulc(v[k1], tw[step * k1]);
        }
        radix8<+1>(v);
    } else {
        small_groups<+1, Fact<N>::RLAST>(v);
    }
}

}  // namespace flutas

// ---- real <-> half-complex along x (real-to-complex / complex-to-real transforms) ---
// A real line of nx = 2*N2 samples is packed as z[i] = x[2i] + i x[2i+1], transformed with the N2-point
// complex FFT above (result Z in permuted order), then turned into X[k] = sum_n x[n] e^{-2 pi i k n / nx}:
//     X[k]      = 1/2 [ (Z[k] + conj Z[N2-k]) - i W^k (Z[k] - conj Z[N2-k]) ],   W = e^{-2 pi i / nx}
// X[k], k = 0..N2-1, is stored where Z[k] was (position pos_of_freq(k)); the Nyquist value X[N2] goes to
// the extra row N2.  One work item handles the pair (q, N2-q), q in [0, N2/2].
namespace flutas {

template <int N2, int C, bool SWZ>
FL_HD void r2c_post_item(double2 *s, int q, int l, const double2 *tw /* tw[m] = e^{-2 pi i m / (2 N2)} */) {
    if (q == 0) {
        const double2 z = s[tile_index<C, SWZ>(0, l)];
        s[tile_index<C, SWZ>(0, l)] = make_double2(z.x + z.y, 0.0);
        s[tile_index<C, SWZ>(N2, l)] = make_double2(z.x - z.y, 0.0);
    } else if (2 * q == N2) {
        const int ia = tile_index<C, SWZ>(pos_of_freq<N2>(q), l);
        s[ia] = cconj(s[ia]);
    } else {
        const int ia = tile_index<C, SWZ>(pos_of_freq<N2>(q), l);
        const int ib = tile_index<C, SWZ>(pos_of_freq<N2>(N2 - q), l);
        const double2 zk = s[ia], zc = cconj(s[ib]);
        const double2 a = cadd(zk, zc), t = cmul(tw[q], csub(zk, zc));
        s[ia] = make_double2(0.5 * (a.x + t.y), 0.5 * (a.y - t.x));     // 1/2 (A - iT)
        s[ib] = make_double2(0.5 * (a.x - t.y), -0.5 * (a.y + t.x));    // 1/2 conj(A + iT)
    }
}

// inverse of the above, up to scale: builds Z' with  (unnormalised inverse FFT of Z')[i] = nx * (x[2i] + i x[2i+1])
//     Z'[k] = (X[k] + conj X[N2-k]) + i conj(W^k) (X[k] - conj X[N2-k])
template <int N2, int C, bool SWZ>
FL_HD void c2r_pre_item(double2 *s, int q, int l, const double2 *tw) {
    if (q == 0) {
        const double x0 = s[tile_index<C, SWZ>(0, l)].x, xn = s[tile_index<C, SWZ>(N2, l)].x;
        s[tile_index<C, SWZ>(0, l)] = make_double2(x0 + xn, x0 - xn);
    } else if (2 * q == N2) {
        const int ia = tile_index<C, SWZ>(pos_of_freq<N2>(q), l);
        const double2 x = s[ia];
        s[ia] = make_double2(2.0 * x.x, -2.0 * x.y);
    } else {
        const int ia = tile_index<C, SWZ>(pos_of_freq<N2>(q), l);
        const int ib = tile_index<C, SWZ>(pos_of_freq<N2>(N2 - q), l);
        const double2 xk = s[ia], xc = cconj(s[ib]);
        const double2 a = cadd(xk, xc), sv = cmulc(csub(xk, xc), tw[q]);
        s[ia] = make_double2(a.x - sv.y, a.y + sv.x);                   // A' + iS
        s[ib] = make_double2(a.x + sv.y, sv.x - a.y);                   // conj(A' - iS)
    }
}

}  // namespace flutas
