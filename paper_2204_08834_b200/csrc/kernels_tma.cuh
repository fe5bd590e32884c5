// kernels_tma.cuh -- persistent, TMA-fed transform kernels (sm_100a).
//
//   fft_tma_kernel   a5 / a7 / a6p   complex FFT along y or z on tiles of C kx-columns x N positions.
//
// The half-spectrum is described to the TMA unit as a rank-3 tensor of doubles
//   dim0 = 2 * (nx/2 + 1)  (re, im interleaved; only the VALID columns),  dim1 = ny,  dim2 = nz
// with row pitch 2 * (nx/2 + 8) doubles.  A tile is the box {2C, rows, 1} (y pass) or {2C, 1, rows}
// (z pass), rows <= 256 per box, which lands in shared memory as [position][C columns] -- exactly the
// interleaved-lines layout of fft_core.cuh -- with out-of-range columns zero-filled on load and
// skipped on store (the last kx tile holds only the Nyquist column).
//
// Each CTA is persistent and walks tiles blockIdx.x, blockIdx.x + gridDim.x, ...; thread 0 keeps the
// load of the next tile and the store of the previous one in flight while all threads transform the
// current buffer in place (P passes, one __syncthreads between passes).
#pragma once
#include "fft_core.cuh"
#include "kernels.cuh"
#include "tma.cuh"

#include <type_traits>
#include <utility>

namespace flutas {

// compile-time loop: f(integral_constant<int, FIRST>) ... f(integral_constant<int, LAST>)
template <int FIRST, int LAST, typename F> __device__ __forceinline__ void static_for(F &&f) {
    if constexpr (FIRST <= LAST) {
        f(std::integral_constant<int, FIRST>{});
        static_for<FIRST + 1, LAST>(std::forward<F>(f));
    }
}

struct TmaFftArgs {
    int n_tiles_x;   // tiles along kx
    int n_outer;     // lines' outer index count: nz for the y pass, ny for the z pass (or the planes of one chunk)
    int outer0;      // first outer index of this launch
    int line_dim;    // tensor dimension the transform runs along: 1 (y) or 2 (z)
    int nxh;         // valid kx columns
    const double2 *tw;                            // e^{-2 pi i m / N}
    const double *lam_x, *lam_outer, *lam_pos;    // SOLVE: eigenvalues in storage (permuted) order
    const double2 *wq;                            // MODE_R2R_*: see Tma1Args
    int reorder, neg;
    const PeerScatter *sc;                        // MODE_*_SCAT: see Tma1Args
};

// reciprocal of a normal, non-zero double (either sign): hardware seed + two Newton steps, <= ~1 ulp
__device__ __forceinline__ double rcp_normal(double x) {
    double r;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(r) : "d"(x));
    r = fma(fma(-x, r, 1.0), r, r);
    r = fma(fma(-x, r, 1.0), r, r);
    return r;
}

template <int N, int C, int MODE, int NT, int NBUF>
__global__ void __launch_bounds__(NT, 1) fft_tma_kernel(const __grid_constant__ CUtensorMap tmap, TmaFftArgs a) {
    extern __shared__ unsigned char smem_raw[];
    constexpr int P = Fact<N>::P;
    constexpr int ROWS = N < 256 ? N : 256, NBOX = N / ROWS;
    constexpr int TILE_ELEMS = N * C;
    constexpr uint32_t TILE_BYTES = TILE_ELEMS * 16u;
    // 128-byte aligned start inside the dynamic allocation (pointer arithmetic keeps the shared address space)
    double2 *bufs = reinterpret_cast<double2 *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    __shared__ uint64_t full[NBUF];

    const int tid = threadIdx.x;
    const int l = tid % C;
    const int ntiles = a.n_tiles_x * a.n_outer;
    if (tid == 0) {
#pragma unroll
        for (int b = 0; b < NBUF; ++b) mbar_init(&full[b], 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    auto issue_load = [&](int tile, int b) {
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
        mbar_arrive_expect_tx(&full[b], TILE_BYTES);
#pragma unroll
        for (int c = 0; c < NBOX; ++c) {
            double2 *dst = bufs + b * TILE_ELEMS + c * ROWS * C;
            if (a.line_dim == 1) tma_load_3d(dst, &tmap, &full[b], tx * 2 * C, c * ROWS, outer);
            else tma_load_3d(dst, &tmap, &full[b], tx * 2 * C, outer, c * ROWS);
        }
    };
    auto issue_store = [&](int tile, int b) {
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
#pragma unroll
        for (int c = 0; c < NBOX; ++c) {
            const double2 *src = bufs + b * TILE_ELEMS + c * ROWS * C;
            if (a.line_dim == 1) tma_store_3d(&tmap, src, tx * 2 * C, c * ROWS, outer);
            else tma_store_3d(&tmap, src, tx * 2 * C, outer, c * ROWS);
        }
        bulk_commit();
    };

    if (tid == 0) {
#pragma unroll
        for (int q = 0; q < NBUF - 1; ++q) {
            const int tile = blockIdx.x + q * gridDim.x;
            if (tile < ntiles) issue_load(tile, q);
        }
    }

    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int b = it % NBUF;
        if (tid == 0) {
            const int nxt = tile + (NBUF - 1) * gridDim.x;
            if (nxt < ntiles) {
                bulk_wait_read<0>();   // the store that last read the target buffer has drained it
                issue_load(nxt, (it + NBUF - 1) % NBUF);
            }
        }
        mbar_wait(&full[b], (it / NBUF) & 1);
        double2 *s = bufs + b * TILE_ELEMS;

        if (MODE == MODE_FWD || MODE == MODE_INV) {
#pragma unroll
            for (int pp = 0; pp < P; ++pp) {
                const int p = (MODE == MODE_FWD) ? pp + 1 : P - pp;
                for (int t = tid / C; t < N / 8; t += NT / C) {
                    int pos[8], n2;
                    double2 v[8];
                    pass_positions<N>(p, t, pos, n2);
#pragma unroll
                    for (int e = 0; e < 8; ++e) v[e] = s[pos[e] * C + l];
                    if (MODE == MODE_FWD) fwd_pass_regs<N>(p, n2, v, a.tw, 1);
                    else inv_pass_regs<N>(p, n2, v, a.tw, 1);
#pragma unroll
                    for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
                }
                if (pp + 1 < P) __syncthreads();
            }
        } else {
            const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
            const int kx = tx * C + l;
            const double lam_xy = a.lam_x[kx < a.nxh ? kx : 0] + a.lam_outer[outer];
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
                    const double inv = (den == 0.0) ? 0.0 : rcp_normal(den);   // (0,0,0) mode dropped: zero-mean gauge
                    v[e] = cscale(v[e], inv);
                }
                inv_pass_regs<N>(P, n2, v, a.tw, 1);
#pragma unroll
                for (int e = 0; e < 8; ++e) s[pos[e] * C + l] = v[e];
            }
#pragma unroll
            for (int p = P - 1; p >= 1; --p) {
                __syncthreads();
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
            }
        }
        fence_proxy_async();
        __syncthreads();
        if (tid == 0) issue_store(tile, b);
    }
    if (tid == 0) bulk_wait_all<0>();
}


// ------------------------------------------------------------------------------------------------
// fft_tma1_kernel: the same transform for the case "one butterfly per thread" (NT == N*C/8), which
// covers every performance-relevant size.  Differences from fft_tma_kernel, all aimed at the SM-internal
// traffic that bounds the generic kernel (shared memory moves 32 B per element per pass):
//   * everything a thread needs per pass -- element offsets and the 7 twiddles of the first NCACHE
//     passes -- is loop-invariant across tiles and lives in registers: no twiddle loads, no index math;
//   * the last pass stores its registers straight to global memory (coalesced 128-byte rows), so a tile
//     crosses shared memory P times instead of P+2 and the buffer is free as soon as it has been read;
//   * TMA only prefetches: thread 0 issues the load of the next tile into the other buffer.
// ------------------------------------------------------------------------------------------------
struct Tma1Args {
    double2 *data;           // the half-spectrum (for the direct stores of the last pass)
    long long row_stride;    // elements between positions r and r+1 of a line
    long long outer_stride;  // elements between outer indices
    int n_tiles_x, n_outer, outer0, line_dim, nxh;   // outer indices outer0 .. outer0 + n_outer - 1
    const double2 *tw;
    const double *lam_x, *lam_outer, *lam_pos;
    // MODE_R2R_FWD / MODE_R2R_INV (non-periodic directions, kernels_r2r.cuh): the real-linear expansion applied to the
    // real and the imaginary part of every column separately
    const double2 *wq;       // e^{-i pi k / (2N)}, k = 0 .. N/2 (cosine / sine expansion); nullptr = half-complex (w = 1)
    int reorder;             // 1: rows enter as v[n] = z[2n], v[N-1-n] = z[2n+1] (cosine / sine), 0: as they are
    int neg;                 // 1: the odd rows change sign (sine expansion)
    const PeerScatter *sc;   // MODE_FWD_SCAT / MODE_SOLVE_SCAT: where the last pass stores (device memory, plan-owned)
};

template <int N, int P_IDX> struct PassGeom {     // geometry of pass P_IDX (1-based) for one thread
    static constexpr bool RADIX8 = (P_IDX < Fact<N>::P) || (Fact<N>::RLAST == 8);
    static constexpr int M = RADIX8 ? (P_IDX < Fact<N>::P ? N / ipow8(P_IDX) : 1) : 1;   // element stride
    static constexpr bool HAS_TW = RADIX8 && M > 1;
    __device__ static __forceinline__ int base(int t) { return RADIX8 ? (t / M) * 8 * M + (t % M) : 8 * t; }
    __device__ static __forceinline__ int n2(int t) { return RADIX8 ? t % M : 0; }
};

template <int N, int P_IDX, int DIR>
__device__ __forceinline__ void butterfly_pass(double2 *v, const double2 *twr) {
    using G = PassGeom<N, P_IDX>;
    if (G::RADIX8) {
        if (DIR < 0) {
            radix8<-1>(v);
            if (G::HAS_TW) {
#pragma unroll
                for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmul(v[k1], twr[k1 - 1]);
            }
        } else {
            if (G::HAS_TW) {
#pragma unroll
                for (int k1 = 1; k1 < 8; ++k1) v[k1] = cmulc(v[k1], twr[k1 - 1]);
            }
            radix8<+1>(v);
        }
    } else {
        small_groups<DIR, Fact<N>::RLAST>(v);
    }
}

// MODE_R2R_FWD / MODE_R2R_INV: a complex FFT of the (re-ordered) rows gives F; the expansion of the real part and of
// the imaginary part, still packed as one complex number per column, is a butterfly between k and N-k:
//     P = w_k F[k],  Q = conj(w_k) F[N-k]:   out[k] = P + Q,   out[N-k] = i (P - Q)        (k = 1 .. N/2 - 1)
//     out[0] = 2 F[0],  out[N/2] = 2 Re(w_{N/2}) F[N/2]
// (w_k = e^{-i pi k / (2N)}: componentwise unnormalised DCT-II, out[k] = X_re[k] + i X_im[k]; sign flip of the odd rows on
// entry: DST-II read backwards; w = 1 and no re-ordering: twice the cosine and minus twice the sine coefficient of the
// periodic expansion, both with eigenvalue lam[k]).  out[k] is stored at the position the FFT leaves frequency k at,
// so the eigenvalue tables are permuted exactly as in the periodic case.  One more trip through shared memory than the
// plain transform (the last pass cannot store straight to global), no extra trip through HBM.
// Barrier between pass P_IDX and pass P_IDX + 1 (either direction).  The butterflies of pass p + 1 that touch one block
// of 8 M_p positions are run by exactly the threads that ran pass p on that block (M_p butterflies x C columns,
// consecutive thread ids), so only the first exchange is CTA-wide; the later ones synchronise M_p C threads: a named
// barrier for 64 and more, __syncwarp below.  Besides being cheaper, this lets the groups drift apart, so that some are
// in the FP64 part of a pass while others are in its shared-memory part.
template <int N, int C, int P_IDX> __device__ __forceinline__ void exchange_sync(int tid) {
    constexpr int GS = (P_IDX < Fact<N>::P ? N / ipow8(P_IDX) : 1) * C;      // threads per group
    if constexpr (P_IDX == 1 || GS * 8 >= N * C) __syncthreads();
    else if constexpr (GS <= 32) __syncwarp();
    else asm volatile("bar.sync %0, %1;" ::"r"(1 + tid / GS), "n"(GS) : "memory");
}

template <int N, int C, int MODE_T, int NT, int NCACHE>
__global__ void __launch_bounds__(NT, 1) fft_tma1_kernel(const __grid_constant__ CUtensorMap tmap, Tma1Args a) {
    static_assert(NT == N * C / 8 || (N * C / 8 < 32 && NT == 32), "one butterfly per thread");
    constexpr bool SCAT = MODE_T == MODE_FWD_SCAT || MODE_T == MODE_SOLVE_SCAT;
    constexpr int MODE = MODE_T == MODE_FWD_SCAT ? MODE_FWD : (MODE_T == MODE_SOLVE_SCAT ? MODE_SOLVE : MODE_T);
    extern __shared__ unsigned char smem_raw[];
    constexpr int P = Fact<N>::P;
    constexpr int ROWS = N < 256 ? N : 256, NBOX = N / ROWS;
    constexpr int TILE_ELEMS = N * C;
    constexpr uint32_t TILE_BYTES = TILE_ELEMS * 16u;
    double2 *bufs = reinterpret_cast<double2 *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    __shared__ uint64_t full[2];

    const int tid = threadIdx.x;
    const int l = tid % C, t = tid / C;
    const bool active = t < N / 8;           // only false for the tiny sizes padded to one warp
    const int ntiles = a.n_tiles_x * a.n_outer;
    __shared__ PeerScatter sc_s;             // the peers' arrays (distributed spectrum), copied once per CTA
    if constexpr (SCAT) {
        static_assert(sizeof(PeerScatter) % 8 == 0, "copied as 8-byte words");
        for (int i = tid; i < (int)(sizeof(PeerScatter) / 8); i += NT)
            reinterpret_cast<unsigned long long *>(&sc_s)[i] = reinterpret_cast<const unsigned long long *>(a.sc)[i];
    }
    if (tid == 0) {
        mbar_init(&full[0], 1);
        mbar_init(&full[1], 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    // loop-invariant per-thread state: twiddles of the first NCACHE passes
    double2 twr[NCACHE > 0 ? NCACHE * 7 : 1];
    if (NCACHE >= 1 && PassGeom<N, 1>::HAS_TW) {
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) twr[k1 - 1] = a.tw[(active ? PassGeom<N, 1>::n2(t) : 0) * k1];
    }
    if (NCACHE >= 2 && PassGeom<N, 2>::HAS_TW) {
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) twr[7 + k1 - 1] = a.tw[8 * (active ? PassGeom<N, 2>::n2(t) : 0) * k1];
    }
    if (NCACHE >= 3 && PassGeom<N, 3>::HAS_TW) {
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1) twr[14 + k1 - 1] = a.tw[64 * (active ? PassGeom<N, 3>::n2(t) : 0) * k1];
    }

    auto issue_load = [&](int tile, int b) {
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
        mbar_arrive_expect_tx(&full[b], TILE_BYTES);
#pragma unroll
        for (int c = 0; c < NBOX; ++c) {
            double2 *dst = bufs + b * TILE_ELEMS + c * ROWS * C;
            if (a.line_dim == 1) tma_load_3d(dst, &tmap, &full[b], tx * 2 * C, c * ROWS, outer);
            else tma_load_3d(dst, &tmap, &full[b], tx * 2 * C, outer, c * ROWS);
        }
    };

    // one pass through shared memory; TW: where this pass's twiddles come from
    auto smem_pass = [&](auto pidx, auto dir, double2 *s, double2 *v) {
        constexpr int PI = decltype(pidx)::value, DIR = decltype(dir)::value;
        using G = PassGeom<N, PI>;
        double2 *sp = s + G::base(t) * C + l;
#pragma unroll
        for (int e = 0; e < 8; ++e) v[e] = sp[e * G::M * C];
        if (PI <= NCACHE) {
            butterfly_pass<N, PI, DIR>(v, twr + 7 * (PI - 1));
        } else {
            double2 tl[7];
            if (G::HAS_TW) {
#pragma unroll
                for (int k1 = 1; k1 < 8; ++k1) tl[k1 - 1] = a.tw[ipow8(PI - 1) * G::n2(t) * k1];
            }
            butterfly_pass<N, PI, DIR>(v, tl);
        }
    };
    auto smem_store = [&](auto pidx, double2 *s, const double2 *v) {
        constexpr int PI = decltype(pidx)::value;
        using G = PassGeom<N, PI>;
        double2 *sp = s + G::base(t) * C + l;
#pragma unroll
        for (int e = 0; e < 8; ++e) sp[e * G::M * C] = v[e];
    };
    ScatterRegs sc;
    sc.load(&sc_s);
    int st_outer = 0, st_kx = 0;          // outer index and column of the tile being stored (SCAT)
    auto global_store = [&](auto pidx, double2 *gp, bool valid, const double2 *v) {
        constexpr int PI = decltype(pidx)::value;
        using G = PassGeom<N, PI>;
        if (valid) {
            if constexpr (SCAT) {
#pragma unroll
                for (int e = 0; e < 8; ++e) scatter_store(sc, G::base(t) + e * G::M, st_outer, st_kx, v[e]);
            } else {
                double2 *q = gp + (long long)G::base(t) * a.row_stride;
                const long long step = (long long)G::M * a.row_stride;
#pragma unroll
                for (int e = 0; e < 8; ++e) q[e * step] = v[e];
            }
        }
    };

    if (tid == 0 && (int)blockIdx.x < ntiles) issue_load(blockIdx.x, 0);

    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int b = it & 1;
        // every thread has finished reading the other buffer (end of the previous iteration): refill it
        __syncthreads();
        if (tid == 0) {
            const int nxt = tile + gridDim.x;
            if (nxt < ntiles) issue_load(nxt, b ^ 1);
        }
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
        const int kx = tx * C + l;
        const bool valid = active && kx < a.nxh;
        double2 *gp = a.data + (long long)outer * a.outer_stride + kx;
        st_outer = outer; st_kx = kx;
        double2 *s = bufs + b * TILE_ELEMS;
        mbar_wait(&full[b], (it >> 1) & 1);

        double2 v[8];
        if (MODE == MODE_FWD) {
            static_for<1, P>([&](auto pi) {
                constexpr int PI = decltype(pi)::value;
                if (active) smem_pass(pi, std::integral_constant<int, -1>{}, s, v);
                if (PI < P) {
                    if (active) smem_store(pi, s, v);
                    exchange_sync<N, C, PI>(tid);
                } else {
                    global_store(pi, gp, valid, v);
                }
            });
        } else if (MODE == MODE_INV) {
            static_for<1, P>([&](auto pr) {
                constexpr int PI = P + 1 - decltype(pr)::value;
                if (active) smem_pass(std::integral_constant<int, PI>{}, std::integral_constant<int, +1>{}, s, v);
                if (PI > 1) {
                    if (active) smem_store(std::integral_constant<int, PI>{}, s, v);
                    exchange_sync<N, C, (PI > 1 ? PI - 1 : 1)>(tid);
                } else {
                    global_store(std::integral_constant<int, PI>{}, gp, valid, v);
                }
            });
        } else if (MODE == MODE_R2R_FWD) {
            auto row_of = [&](int n) { return a.reorder ? (n < N / 2 ? 2 * n : 2 * N - 1 - 2 * n) : n; };
            {   // pass 1 reads the rows in the order of the expansion; it is not in place, so all reads come first
                using G = PassGeom<N, 1>;
                const int base = G::base(t);
                if (active) {
#pragma unroll
                    for (int e = 0; e < 8; ++e) {
                        const int n = base + e * G::M;
                        v[e] = s[row_of(n) * C + l];
                        if (a.neg && n >= N / 2) v[e] = make_double2(-v[e].x, -v[e].y);
                    }
                }
                __syncthreads();
                if (NCACHE >= 1) butterfly_pass<N, 1, -1>(v, twr);
                else {
                    double2 tl[7];
                    if (G::HAS_TW) {
#pragma unroll
                        for (int k1 = 1; k1 < 8; ++k1) tl[k1 - 1] = a.tw[(active ? G::n2(t) : 0) * k1];
                    }
                    butterfly_pass<N, 1, -1>(v, tl);
                }
                if (active) smem_store(std::integral_constant<int, 1>{}, s, v);
                __syncthreads();
            }
            static_for<2, P>([&](auto pi) {
                if (active) {
                    smem_pass(pi, std::integral_constant<int, -1>{}, s, v);
                    smem_store(pi, s, v);
                }
                __syncthreads();
            });
            if (valid) {   // the butterfly between k and N - k, straight to global memory
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int k = t + r * (N / 8);
                    if (k == 0) {
                        const double2 f0 = s[l], fh = s[pos_of_freq<N>(N / 2) * C + l];
                        const double wh = a.wq ? 2.0 * a.wq[N / 2].x : 2.0;
                        gp[0] = make_double2(2.0 * f0.x, 2.0 * f0.y);
                        gp[(long long)pos_of_freq<N>(N / 2) * a.row_stride] = make_double2(wh * fh.x, wh * fh.y);
                    } else {
                        const int pa = pos_of_freq<N>(k), pb = pos_of_freq<N>(N - k);
                        const double2 w = a.wq ? a.wq[k] : make_double2(1.0, 0.0);
                        const double2 pp = cmul(w, s[pa * C + l]), qq = cmulc(s[pb * C + l], w);
                        gp[(long long)pa * a.row_stride] = cadd(pp, qq);
                        const double2 d = csub(pp, qq);
                        gp[(long long)pb * a.row_stride] = make_double2(-d.y, d.x);
                    }
                }
            }
        } else if (MODE == MODE_R2R_INV) {
            if (active) {   // undo the butterfly in place (every pair belongs to one thread)
#pragma unroll
                for (int r = 0; r < 4; ++r) {
                    const int k = t + r * (N / 8);
                    if (k == 0) {
                        const int ph = pos_of_freq<N>(N / 2) * C + l;
                        const double wh = a.wq ? 0.5 / a.wq[N / 2].x : 0.5;
                        s[l] = make_double2(0.5 * s[l].x, 0.5 * s[l].y);
                        s[ph] = make_double2(wh * s[ph].x, wh * s[ph].y);
                    } else {
                        const int pa = pos_of_freq<N>(k) * C + l, pb = pos_of_freq<N>(N - k) * C + l;
                        const double2 w = a.wq ? a.wq[k] : make_double2(1.0, 0.0);
                        const double2 c = s[pa], sn = s[pb];
                        const double2 pp = make_double2(0.5 * (c.x + sn.y), 0.5 * (c.y - sn.x));   // (c - i s) / 2
                        const double2 qq = make_double2(0.5 * (c.x - sn.y), 0.5 * (c.y + sn.x));   // (c + i s) / 2
                        s[pa] = cmulc(pp, w);
                        s[pb] = cmul(w, qq);
                    }
                }
            }
            __syncthreads();
            static_for<1, P>([&](auto pr) {
                constexpr int PI = P + 1 - decltype(pr)::value;
                if (active) smem_pass(std::integral_constant<int, PI>{}, std::integral_constant<int, +1>{}, s, v);
                if (PI > 1) {
                    if (active) smem_store(std::integral_constant<int, PI>{}, s, v);
                    __syncthreads();
                }
            });
            if (valid) {   // the last pass leaves natural order: element n goes back to the row it came from
                using G = PassGeom<N, 1>;
                const int base = G::base(t);
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const int n = base + e * G::M;
                    const int row = a.reorder ? (n < N / 2 ? 2 * n : 2 * N - 1 - 2 * n) : n;
                    const bool flip = a.neg && n >= N / 2;
                    gp[(long long)row * a.row_stride] = flip ? make_double2(-v[e].x, -v[e].y) : v[e];
                }
            }
        } else {
            const double lam_xy = a.lam_x[kx < a.nxh ? kx : 0] + a.lam_outer[outer];
            static_for<1, P>([&](auto pi) {
                constexpr int PI = decltype(pi)::value;
                if (active) smem_pass(pi, std::integral_constant<int, -1>{}, s, v);
                if (PI < P) {
                    if (active) smem_store(pi, s, v);
                    exchange_sync<N, C, PI>(tid);
                }
            });
            // v holds the last forward pass: divide by the eigenvalue sum, run the first inverse pass in registers
            {
                using G = PassGeom<N, P>;
                const int base = G::base(t);
#pragma unroll
                for (int e = 0; e < 8; ++e) {
                    const double den = lam_xy + a.lam_pos[active ? base + e * G::M : 0];
                    const double inv = (den == 0.0) ? 0.0 : rcp_normal(den);   // (0,0,0) mode dropped: zero-mean gauge
                    v[e] = cscale(v[e], inv);
                }
                if (P <= NCACHE) butterfly_pass<N, P, +1>(v, twr + 7 * (P - 1));
                else {
                    double2 tl[7];
                    if (G::HAS_TW) {
#pragma unroll
                        for (int k1 = 1; k1 < 8; ++k1) tl[k1 - 1] = a.tw[ipow8(P - 1) * G::n2(t) * k1];
                    }
                    butterfly_pass<N, P, +1>(v, tl);
                }
                if (P > 1) {
                    if (active) smem_store(std::integral_constant<int, P>{}, s, v);
                    exchange_sync<N, C, (P > 1 ? P - 1 : 1)>(tid);
                } else {
                    global_store(std::integral_constant<int, P>{}, gp, valid, v);
                }
            }
            static_for<2, P>([&](auto pr) {
                constexpr int PI = P + 1 - decltype(pr)::value;     // P-1 ... 1
                if (active) smem_pass(std::integral_constant<int, PI>{}, std::integral_constant<int, +1>{}, s, v);
                if (PI > 1) {
                    if (active) smem_store(std::integral_constant<int, PI>{}, s, v);
                    exchange_sync<N, C, (PI > 1 ? PI - 1 : 1)>(tid);
                } else {
                    global_store(std::integral_constant<int, PI>{}, gp, valid, v);
                }
            });
        }
    }
}

}  // namespace flutas
