// kernels_x.cuh -- persistent, bulk-copy-fed transforms along x (sm_100a): rows a4 and a8 of the step.
//
//   fft_x_r2c_tma_kernel   real lines  -> half-spectrum rows (kx = 0..nx/2 in NATURAL order)
//   fft_x_c2r_tma_kernel   half-spectrum rows -> real lines, scaled by 1/(nx ny [nz])
//
// A tile is 8 consecutive x-lines: contiguous in memory on both sides (the spectrum row pitch is nx/2 + 8
// complex), so one elected thread moves it with a single linear cp.async.bulk (UBLKCP) into a landing buffer
// while the other warps still work on the previous tile.  A line of nx reals is transformed as an N2 = nx/2
// point complex FFT of z[i] = x[2i] + i x[2i+1] plus the usual split (fft_core.cuh).
//
// Shared-memory traffic is what bounds these kernels (every element crosses shared memory once per pass), so:
//  * pass 1 of the forward transform reads the landing buffer in its natural [line][pos] layout with threads
//    running along the line (conflict free), and every later exchange uses the interleaved layout
//    [pos][8 lines] of fft_core.cuh with threads running across the 8 lines;
//  * the slot of line l inside a 128-byte row is l ^ key(pos).  key = pos & 7 serves exchanges whose other side
//    runs along the line with consecutive positions; key = pos / (N2/8) (the digit that becomes kx mod 8)
//    serves the split, which runs along consecutive kx.  Changing key only permutes a row among the 8 threads
//    that own it, so a __syncwarp is enough when one pass re-keys its own rows;
//  * the split writes / reads the global spectrum directly in natural kx order (ascending q and descending
//    N2 - q are both coalesced), so no separate output staging pass exists;
//  * twiddles of the two twiddled passes are loop invariant per thread and live in registers.
//
// KIND = X_SPLIT: the same kernels for NON-PERIODIC x (kernels_r2r.cuh explains the algorithm and the "split column"
// layout): the cosine / sine expansion is the real transform of the re-ordered line, so the forward kernel gathers
// z[i] = (v[2i], v[2i+1]) out of the landing buffer (even samples forwards, odd samples backwards, sign flipped for the
// sine expansion) and multiplies the split by w_k = e^{-i pi k / (2 nx)}; the inverse kernel undoes the twiddle inside
// the inverse split and scatters its natural-order output back to the even / odd samples of the line.
#pragma once
#include "kernels_r2r.cuh"
#include "kernels_tma.cuh"

namespace flutas {

enum { KEY_LOW = 0, KEY_TOP = 1 };
enum { X_PERIODIC = 0, X_SPLIT = 1 };
template <int N, int KEY> __device__ __forceinline__ int xslot(int pos, int l) {
    return pos * 8 + (l ^ (KEY == KEY_LOW ? (pos & 7) : (pos / (N / 8))));
}

template <int N2> struct XGeom {
    static_assert(N2 >= 64, "the persistent x kernels need nx >= 128");
    static constexpr int P = Fact<N2>::P;
    static constexpr int B = N2 / 8;              // butterflies per line and pass = stride of pass 1
    static constexpr int PITCH = N2 + 8;          // complex elements per spectrum row
    static constexpr bool TW2 = PassGeom<N2, 2>::HAS_TW;
};

// twiddles of pass 1 (role "along the line", n2 = t) and pass 2 (role "across lines")
template <int N2> __device__ __forceinline__ void load_twiddle_regs(const double2 *__restrict__ tw, int ta, int tb,
                                                                     double2 *twr1, double2 *twr2) {
#pragma unroll
    for (int k1 = 1; k1 < 8; ++k1) twr1[k1 - 1] = tw[2 * ta * k1];
    if (XGeom<N2>::TW2) {
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) twr2[k1 - 1] = tw[2 * 8 * PassGeom<N2, 2>::n2(tb) * k1];
    }
}

// one pass "across lines" on the interleaved tile; key_in / key_out name the row keys on both sides
template <int N2, int PI, int DIR, int KEY_IN, int KEY_OUT>
__device__ __forceinline__ void xpass_b(double2 *X, int lb, int tb, const double2 *twr) {
    using G = PassGeom<N2, PI>;
    const int base = G::base(tb);
    double2 v[8];
#pragma unroll
    for (int e = 0; e < 8; ++e) v[e] = X[xslot<N2, KEY_IN>(base + e * G::M, lb)];
    butterfly_pass<N2, PI, DIR>(v, twr);
    if (KEY_IN != KEY_OUT) __syncwarp();
#pragma unroll
    for (int e = 0; e < 8; ++e) X[xslot<N2, KEY_OUT>(base + e * G::M, lb)] = v[e];
}

// ------------------------------------------------------------------------------------------------
// a4: real-to-complex along x
// ------------------------------------------------------------------------------------------------
template <int N2, int KIND = X_PERIODIC>
__global__ void __launch_bounds__(N2, N2 <= 256 ? 2 : 1)
fft_x_r2c_tma_kernel(const double *__restrict__ rhs, double2 *__restrict__ spec, const double2 *__restrict__ tw, int ntiles,
                     SpecRows sr, const double2 *__restrict__ wq = nullptr, int neg_odd = 0) {
    using XG = XGeom<N2>;
    constexpr int P = XG::P, B = XG::B, PITCH = XG::PITCH;
    static_assert(P <= 3, "nx <= 1024");
    constexpr uint32_t TILE_BYTES = 8u * N2 * 16u;
    extern __shared__ unsigned char smem_raw[];
    double2 *land = reinterpret_cast<double2 *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    double2 *X = land + 8 * N2;
    __shared__ uint64_t full;

    const int tid = threadIdx.x;
    const int la = tid / B, ta = tid % B;     // role a: threads run along the line
    const int lb = tid % 8, tb = tid / 8;     // role b: threads run across the 8 lines
    if (tid == 0) {
        mbar_init(&full, 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();
    double2 twr1[7], twr2[7];
    load_twiddle_regs<N2>(tw, ta, tb, twr1, twr2);

    auto issue_load = [&](int tile) {
        mbar_arrive_expect_tx(&full, TILE_BYTES);
        bulk_load(land, rhs + (long long)tile * 8 * 2 * N2, TILE_BYTES, &full);
    };
    if (tid == 0 && (int)blockIdx.x < ntiles) issue_load(blockIdx.x);

    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        mbar_wait(&full, it & 1);
        {   // pass 1 straight from the landing buffer (natural layout), written interleaved
            double2 v[8];
            if (KIND == X_PERIODIC) {
                const double2 *lp = land + la * N2 + ta;
#pragma unroll
                for (int e = 0; e < 8; ++e) v[e] = lp[e * B];
            } else {   // z[i] of the re-ordered line: (x[4i], x[4i+2]) in the first half, (x[2N-4i-1], x[2N-4i-3]) after it
                const double *L = reinterpret_cast<const double *>(land) + la * 2 * N2;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int i = ta + e * B;
                    if (e < 4) v[e] = make_double2(L[4 * i], L[4 * i + 2]);
                    else {
                        const double a = L[4 * N2 - 4 * i - 1], b = L[4 * N2 - 4 * i - 3];
                        v[e] = neg_odd ? make_double2(-a, -b) : make_double2(a, b);
                    }
                }
            }
            butterfly_pass<N2, 1, -1>(v, twr1);
#pragma unroll
            for (int e = 0; e < 8; ++e) X[xslot<N2, KEY_LOW>(ta + e * B, la)] = v[e];
        }
        __syncthreads();                       // landing buffer consumed: refill it while the tile is transformed
        if (tid == 0) {
            const int nxt = tile + gridDim.x;
            if (nxt < ntiles) issue_load(nxt);
        }
        if (P == 3) {
            xpass_b<N2, 2, -1, KEY_LOW, KEY_LOW>(X, lb, tb, twr2);
            __syncthreads();
            xpass_b<N2, 3, -1, KEY_LOW, KEY_TOP>(X, lb, tb, nullptr);
        } else {
            xpass_b<N2, 2, -1, KEY_LOW, KEY_TOP>(X, lb, tb, twr2);
        }
        __syncthreads();
        {   // split: Z -> X[q], X[N2 - q], written to the global row in natural kx order
            double2 *dst = spec + spec_row_offset(sr, (long long)tile * 8, PITCH) + la * PITCH;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int q = ta + r * B;                    // 0 .. N2/2 - 1
                if (q == 0) {
                    const double2 z = X[xslot<N2, KEY_TOP>(0, la)];
                    if (KIND == X_PERIODIC) {
                        dst[0] = make_double2(z.x + z.y, 0.0);
                        dst[N2] = make_double2(z.x - z.y, 0.0);
                    } else {
                        dst[0] = make_double2(2.0 * (z.x + z.y), kSqrt2 * (z.x - z.y));    // (X[0], X[nx/2])
                    }
                } else {
                    const double2 zk = X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(q), la)];
                    const double2 zc = cconj(X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(N2 - q), la)]);
                    const double2 a = cadd(zk, zc), t = cmul(__ldg(tw + q), csub(zk, zc));
                    const double2 va = make_double2(0.5 * (a.x + t.y), 0.5 * (a.y - t.x));          // 1/2 (A - iT)
                    const double2 vb = make_double2(0.5 * (a.x - t.y), -0.5 * (a.y + t.x));         // 1/2 conj(A + iT)
                    if (KIND == X_PERIODIC) {
                        dst[q] = va;
                        dst[N2 - q] = vb;
                    } else {                                                                        // 2 conj(w_k V[k])
                        const double2 ya = cmul(__ldg(wq + q), va), yb = cmul(__ldg(wq + N2 - q), vb);
                        dst[q] = make_double2(2.0 * ya.x, -2.0 * ya.y);
                        dst[N2 - q] = make_double2(2.0 * yb.x, -2.0 * yb.y);
                    }
                }
            }
            if (ta == 0) {
                const double2 vh = cconj(X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(N2 / 2), la)]);
                if (KIND == X_PERIODIC) dst[N2 / 2] = vh;
                else {
                    const double2 y = cmul(__ldg(wq + N2 / 2), vh);
                    dst[N2 / 2] = make_double2(2.0 * y.x, -2.0 * y.y);
                }
            }
        }
        __syncthreads();                       // X is free for the next tile
    }
}

// ------------------------------------------------------------------------------------------------
// a8: complex-to-real along x, scaled; writes p^(n+1)
// ------------------------------------------------------------------------------------------------
template <int N2, int KIND = X_PERIODIC>
__global__ void __launch_bounds__(N2, N2 <= 256 ? 2 : 1)
fft_x_c2r_tma_kernel(const double2 *__restrict__ spec, double *__restrict__ out, const double2 *__restrict__ tw,
                     double scale, int ntiles, SpecRows sr, const double2 *__restrict__ wq = nullptr, int neg_odd = 0) {
    using XG = XGeom<N2>;
    constexpr int P = XG::P, B = XG::B, PITCH = XG::PITCH;
    static_assert(P <= 3, "nx <= 1024");
    constexpr uint32_t TILE_BYTES = 8u * PITCH * 16u;
    extern __shared__ unsigned char smem_raw[];
    double2 *land = reinterpret_cast<double2 *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    double2 *X = land + 8 * PITCH;
    __shared__ uint64_t full;

    const int tid = threadIdx.x;
    const int la = tid / B, ta = tid % B;
    const int lb = tid % 8, tb = tid / 8;
    if (tid == 0) {
        mbar_init(&full, 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();
    double2 twr1[7], twr2[7];
    load_twiddle_regs<N2>(tw, ta, tb, twr1, twr2);

    auto issue_load = [&](int tile) {
        mbar_arrive_expect_tx(&full, TILE_BYTES);
        bulk_load(land, spec + spec_row_offset(sr, (long long)tile * 8, PITCH), TILE_BYTES, &full);
    };
    if (tid == 0 && (int)blockIdx.x < ntiles) issue_load(blockIdx.x);

    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        mbar_wait(&full, it & 1);
        {   // inverse split: X[q], X[N2 - q] -> Z'[q], Z'[N2 - q] at their transform positions
            const double2 *src = land + la * PITCH;
#pragma unroll
            for (int r = 0; r < 4; ++r) {
                const int q = ta + r * B;
                if (q == 0) {
                    const double x0 = KIND == X_PERIODIC ? src[0].x : 0.5 * src[0].x;                      // V[0]
                    const double xn = KIND == X_PERIODIC ? src[N2].x : src[0].y * (0.5 * kSqrt2);        // V[nx/2]
                    X[xslot<N2, KEY_TOP>(0, la)] = make_double2(x0 + xn, x0 - xn);
                } else {
                    double2 xk = src[q], xc = src[N2 - q];
                    if (KIND == X_SPLIT) {                                           // V[k] = conj(w_k) conj(column k) / 2
                        xk = cmulc(make_double2(0.5 * xk.x, -0.5 * xk.y), __ldg(wq + q));
                        xc = cmulc(make_double2(0.5 * xc.x, -0.5 * xc.y), __ldg(wq + N2 - q));
                    }
                    xc = cconj(xc);
                    const double2 a = cadd(xk, xc), sv = cmulc(csub(xk, xc), __ldg(tw + q));
                    X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(q), la)] = make_double2(a.x - sv.y, a.y + sv.x);        // A' + iS
                    X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(N2 - q), la)] = make_double2(a.x + sv.y, sv.x - a.y);   // conj(A' - iS)
                }
            }
            if (ta == 0) {
                double2 x = src[N2 / 2];
                if (KIND == X_SPLIT) x = cmulc(make_double2(0.5 * x.x, -0.5 * x.y), __ldg(wq + N2 / 2));
                X[xslot<N2, KEY_TOP>(pos_of_freq<N2>(N2 / 2), la)] = make_double2(2.0 * x.x, -2.0 * x.y);
            }
        }
        __syncthreads();                       // landing buffer consumed
        if (tid == 0) {
            const int nxt = tile + gridDim.x;
            if (nxt < ntiles) issue_load(nxt);
        }
        if (P == 3) {
            xpass_b<N2, 3, +1, KEY_TOP, KEY_LOW>(X, lb, tb, nullptr);
            __syncthreads();
            xpass_b<N2, 2, +1, KEY_LOW, KEY_LOW>(X, lb, tb, twr2);
        } else {
            xpass_b<N2, 2, +1, KEY_TOP, KEY_LOW>(X, lb, tb, twr2);
        }
        __syncthreads();
        {   // pass 1 along the line; its natural-order output goes straight to global memory
            double2 v[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) v[e] = X[xslot<N2, KEY_LOW>(ta + e * B, la)];
            butterfly_pass<N2, 1, +1>(v, twr1);
            if (KIND == X_PERIODIC) {
                double2 *dst = reinterpret_cast<double2 *>(out) + ((long long)tile * 8 + la) * N2 + ta;
#pragma unroll
                for (int e = 0; e < 8; ++e) dst[e * B] = cscale(v[e], scale);
            } else {   // z[i] = (v[2i], v[2i+1]) goes back to the even samples (forwards) and the odd samples (backwards):
                       // re-assembled as whole lines in X (free once every thread holds its operands), then stored coalesced
                __syncthreads();
                double *L = reinterpret_cast<double *>(X) + la * 2 * N2;
                const double so = neg_odd ? -scale : scale;
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int i = ta + e * B;
                    if (e < 4) { L[4 * i] = v[e].x * scale; L[4 * i + 2] = v[e].y * scale; }
                    else { L[4 * N2 - 4 * i - 1] = v[e].x * so; L[4 * N2 - 4 * i - 3] = v[e].y * so; }
                }
                __syncthreads();
                double2 *dst = reinterpret_cast<double2 *>(out) + (long long)tile * 8 * N2;
#pragma unroll
                for (int e = 0; e < 8; ++e) dst[tid + e * N2] = X[tid + e * N2];
            }
        }
        __syncthreads();                       // X is free for the next tile
    }
}

}  // namespace flutas
