// kernels_y16.cuh -- complex transform of length 1024 = 16 x 8 x 8 along a strided direction (rows a5 / a7 at
// ny = 1024), sm_100a.  Same tiles and the same TMA tensor map as fft_tma1_kernel (kernels_tma.cuh), but built for
// the case that kernel handles badly: at N = 1024 a tile of 8 kx columns is 128 KB, two of them do not fit in
// shared memory, and the 4-column fallback moves 64-byte rows through four passes (measured 3.5 TB/s).
//
// Here the tile lives in REGISTERS (512 threads x 16 elements) and shared memory only lands and exchanges:
//   L  128 KB  landing buffer of the TMA load; every thread takes its 16 operands out of it first thing, so it is
//              handed back to the TMA unit (load of the next tile) ~5 % into the tile: a 128 KB load needs > 3 us at
//              an SM's share of HBM bandwidth, about half of the tile's time
//   E   64 KB  exchange buffer: half a tile per round for the CTA-wide exchange, then 8 pairs of warps x 8 KB for
//              the pair-local one
//   T   16 KB  the twiddle table e^{-2 pi i m / 1024}
// Three passes (radix 16, 8, 8) instead of four, two exchanges, every shared-memory access a 128-byte row per
// quarter-warp (no conflicts, no swizzle), the last pass stores its registers straight to global memory.
//
// Forward (decimation in frequency), n = 64 n1 + n2, n2 = 8 a + c:
//   pass 1  x1[k1, n2]    = W1024^(n2 k1) sum_n1 W16^(n1 k1) x[64 n1 + n2]          role A: thread = n2, 16 n1
//   pass 2  x2[k1, k2, c] = W64^(c k2)    sum_a  W8^(a k2)  x1[k1, 8 a + c]          role B: thread = (k1 pair, c), 8 a each
//   pass 3  X[k1 + 16 k2 + 128 k3] = sum_c W8^(c k3) x2[k1, k2, c]                   role C: thread = (k1 pair, k2), 8 c each
// and the result is stored at position k1 * 64 + k2 * 8 + k3 (permuted order: y1024_freq_of_pos).  The inverse is the
// conjugate transpose, passes in reverse order, permuted input, natural output.
// Exchange A -> B crosses the whole CTA; B -> C stays inside the 64 threads that share a k1 pair (forward) -- and
// in the inverse the roles are laid out the other way round (C -> B crosses the CTA, B -> A stays inside the 64
// threads that share c); in both directions the pair-local exchange is the LAST one, so that the pairs drift apart
// only where nothing CTA-wide follows inside the tile.
#pragma once
#include "kernels_tma.cuh"

namespace flutas {

// storage position -> frequency of the 16 x 8 x 8 plan
__host__ __device__ inline int y1024_freq_of_pos(int pos) { return (pos >> 6) + 16 * ((pos >> 3) & 7) + 128 * (pos & 7); }

struct Y16Geom {
    static constexpr int N = 1024, C = 8, NT = 512;
    static constexpr int ROWS = 256, NBOX = N / ROWS;
    static constexpr uint32_t TILE_BYTES = N * C * 16u;
    static constexpr size_t SMEM = (size_t)TILE_BYTES + 64 * 1024 + N * 16 + 128;
};

__device__ __forceinline__ void pair_barrier(int pair) {   // the 64 threads of one pair of warps
    asm volatile("bar.sync %0, 64;" ::"r"(pair + 1) : "memory");
}

template <int MODE>
__global__ void __launch_bounds__(Y16Geom::NT, 1) fft_y1024_kernel(const __grid_constant__ CUtensorMap tmap, Tma1Args a) {
    using G = Y16Geom;
    static_assert(MODE == MODE_FWD || MODE == MODE_INV, "transform only");
    extern __shared__ unsigned char smem_raw[];
    double2 *L = reinterpret_cast<double2 *>(smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u));
    double2 *E = L + G::N * G::C;
    double2 *T = E + 4096;
    __shared__ uint64_t full;

    const int tid = threadIdx.x;
    const int l = tid & 7, t6 = tid >> 3;            // t6 in [0, 64)
    const int pair = tid >> 6, sub = t6 & 7;         // pair of warps, index inside it
    const int ntiles = a.n_tiles_x * a.n_outer;
    if (tid == 0) {
        mbar_init(&full, 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    for (int m = tid; m < G::N; m += G::NT) T[m] = a.tw[m];
    __syncthreads();

    auto issue_load = [&](int tile) {
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
        mbar_arrive_expect_tx(&full, G::TILE_BYTES);
#pragma unroll
        for (int c = 0; c < G::NBOX; ++c) {
            double2 *dst = L + c * G::ROWS * G::C;
            if (a.line_dim == 1) tma_load_3d(dst, &tmap, &full, tx * 2 * G::C, c * G::ROWS, outer);
            else tma_load_3d(dst, &tmap, &full, tx * 2 * G::C, outer, c * G::ROWS);
        }
    };
    if (tid == 0 && (int)blockIdx.x < ntiles) issue_load(blockIdx.x);

    double2 *Ep = E + pair * 512;                    // this pair's 8 KB of the exchange buffer
    int it = 0;
    for (int tile = blockIdx.x; tile < ntiles; tile += gridDim.x, ++it) {
        const int tx = tile % a.n_tiles_x, outer = a.outer0 + tile / a.n_tiles_x;
        const int kx = tx * G::C + l;
        const bool valid = kx < a.nxh;
        double2 *gp = a.data + (long long)outer * a.outer_stride + kx;
        double2 v[16];
        mbar_wait(&full, it & 1);

        if (MODE == MODE_FWD) {
            // ---- role A: n2 = t6; pass 1
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = L[(e * 64 + t6) * 8 + l];
            __syncthreads();                         // L is in registers: the next tile may land
            if (tid == 0) {
                const int nxt = tile + gridDim.x;
                if (nxt < ntiles) { fence_proxy_async(); issue_load(nxt); }
            }
            radix16<-1>(v);
#pragma unroll
            for (int k1 = 1; k1 < 16; ++k1) v[k1] = cmul(v[k1], T[t6 * k1]);
            // ---- CTA-wide exchange A -> B through E, two rounds of 32 n2 (a = n2 / 8 in [4h, 4h + 4)): the writers of
            //      a round put down all 16 k1, every thread picks up 2 k1 x 4 a.  Role B: k1 = 2 pair + r, c = sub
            double2 u[16];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (h == 1) __syncthreads();         // round 0 has been read
                if ((t6 >> 5) == h) {
#pragma unroll
                    for (int k1 = 0; k1 < 16; ++k1) E[(k1 * 32 + (t6 & 31)) * 8 + l] = v[k1];
                }
                __syncthreads();
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int aa = 0; aa < 4; ++aa) u[8 * r + 4 * h + aa] = E[((2 * pair + r) * 32 + 8 * aa + sub) * 8 + l];
            }
            __syncthreads();                         // E is free for the pair-local exchange
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = u[e];
            radix8<-1>(v);
            radix8<-1>(v + 8);
#pragma unroll
            for (int k2 = 1; k2 < 8; ++k2) {
                const double2 w = T[16 * sub * k2];
                v[k2] = cmul(v[k2], w);
                v[8 + k2] = cmul(v[8 + k2], w);
            }
            // ---- pair-local exchange B -> C, one k1 per round; role C: k2 = sub; v[8 r + c]
#pragma unroll
            for (int r = 0; r < 2; ++r) {
                if (r == 1) pair_barrier(pair);      // round 0 has been read
#pragma unroll
                for (int k2 = 0; k2 < 8; ++k2) Ep[(k2 * 8 + sub) * 8 + l] = v[8 * r + k2];
                pair_barrier(pair);
#pragma unroll
                for (int c = 0; c < 8; ++c) v[8 * r + c] = Ep[(sub * 8 + c) * 8 + l];
            }
            radix8<-1>(v);
            radix8<-1>(v + 8);
            if (valid) {
#pragma unroll
                for (int r = 0; r < 2; ++r)
#pragma unroll
                    for (int k3 = 0; k3 < 8; ++k3)
                        gp[(long long)((2 * pair + r) * 64 + sub * 8 + k3) * a.row_stride] = v[8 * r + k3];
            }
            // (the next write into E comes after three CTA-wide barriers of the next tile)
        } else {
            // ---- role C: (k1, k2 pair) = t6: rows 16 t6 + e, e = 8 q + k3; inverse pass 3
#pragma unroll
            for (int e = 0; e < 16; ++e) v[e] = L[(16 * t6 + e) * 8 + l];
            __syncthreads();                         // L is in registers: the next tile may land
            if (tid == 0) {
                const int nxt = tile + gridDim.x;
                if (nxt < ntiles) { fence_proxy_async(); issue_load(nxt); }
            }
            radix8<+1>(v);                           // -> c: v[8 q + c], k1 = t6 / 4, k2 = 2 (t6 % 4) + q
            radix8<+1>(v + 8);
            // ---- CTA-wide exchange C -> B through E, two rounds of 4 k2 (k2 in [4h, 4h + 4)): the writers of a round
            //      put down their 2 k2 x 8 c, every thread picks up 2 k1 x 4 k2.  Role B: c = pair, k1 = 2 sub + r
            {
                double2 u[16];
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    if (h == 1) __syncthreads();
                    if (((t6 & 3) >> 1) == h) {
#pragma unroll
                        for (int e = 0; e < 16; ++e)   // k2 - 4h = 2 (t6 & 1) + q
                            E[((t6 >> 2) * 32 + (2 * (t6 & 1) + (e >> 3)) * 8 + (e & 7)) * 8 + l] = v[e];
                    }
                    __syncthreads();
#pragma unroll
                    for (int r = 0; r < 2; ++r)
#pragma unroll
                        for (int kk = 0; kk < 4; ++kk) u[8 * r + 4 * h + kk] = E[((2 * sub + r) * 32 + kk * 8 + pair) * 8 + l];
                }
                __syncthreads();                     // E is free for the pair-local exchange
#pragma unroll
                for (int e = 0; e < 16; ++e) v[e] = u[e];
            }
#pragma unroll
            for (int k2 = 1; k2 < 8; ++k2) {
                const double2 w = T[16 * pair * k2];
                v[k2] = cmulc(v[k2], w);
                v[8 + k2] = cmulc(v[8 + k2], w);
            }
            radix8<+1>(v);                           // -> a
            radix8<+1>(v + 8);
            // ---- pair-local exchange B -> A in two rounds of 8 k1; role A: a = sub, n2 = 8 sub + pair; v[k1]
            double2 u[16];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                if (h == 1) pair_barrier(pair);
                if ((sub >> 2) == h) {               // this thread's two k1 belong to this round
#pragma unroll
                    for (int r = 0; r < 2; ++r)
#pragma unroll
                        for (int aa = 0; aa < 8; ++aa) Ep[(((2 * sub + r) & 7) * 8 + aa) * 8 + l] = v[8 * r + aa];
                }
                pair_barrier(pair);
#pragma unroll
                for (int q = 0; q < 8; ++q) u[8 * h + q] = Ep[(q * 8 + sub) * 8 + l];
            }
            const int n2 = 8 * sub + pair;
#pragma unroll
            for (int k1 = 1; k1 < 16; ++k1) u[k1] = cmulc(u[k1], T[n2 * k1]);
            radix16<+1>(u);
            if (valid) {
#pragma unroll
                for (int n1 = 0; n1 < 16; ++n1) gp[(long long)(n1 * 64 + n2) * a.row_stride] = u[n1];
            }
        }
    }
}

}  // namespace flutas
