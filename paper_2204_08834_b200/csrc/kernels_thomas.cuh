// kernels_thomas.cuh -- a6w in ONE pass over the half-spectrum: Gauss elimination along z per (kx, ky)
// ("step 5"; Neumann ends, R7) on tiles that live in shared memory (sm_100a).
//
//   a x_{k-1} + b_k x_k + a x_{k+1} = d_k,   a = 1/dz^2,  b_k = -2a + lam_xy (interior), -a + lam_xy (k = 0, nz-1)
//
// thomas_kernel (kernels.cuh) sweeps the spectrum twice through HBM (forward: read d, write d' and c'; backward:
// read both, write x: 5 passes of the half-spectrum).  Here a tile = 8 consecutive kx columns x all nz planes of one
// ky (nz x 128 bytes, the box {16 doubles, 1, rows} of the same rank-3 tensor map the periodic z transform uses)
// is fetched once by the TMA unit, solved in place in shared memory and written back once: 2 passes + the
// coefficient table below.
//
// The elimination is sequential in k, so the parallelism inside a tile is what the tile offers and no more:
// 8 columns x (re, im).  It is doubled by eliminating from BOTH ends towards the middle ("twisted" factorisation:
// still Gauss elimination without pivoting, rows 0..m-1 downwards and rows nz-1..m upwards, a 2x2 system where they
// meet, then back-substitution outwards): 32 chains = one warp per tile, every chain step one dependent FMA:
//     forward   g_j = d_row(j) * inv_j - c_j * g_{j-1}         c_j = a / (b_j - a c_{j-1}),  inv_j = c_j / a
//     middle    x_m = (h_m - c~_m g_{m-1}) / (1 - c~_m c_{m-1}),   x_{m-1} = g_{m-1} - c_{m-1} x_m
//     backward  x_j = g_j - c_j * x_{j+1}
// with row(j) = j for the chain from the bottom wall and nz-1-j for the chain from the top wall.  The matrix is
// symmetric under k -> nz-1-k, so both chains of a column use the SAME coefficients c_j: they depend on the grid
// only, not on the data, and are tabulated once per plan (thomas_table_kernel) in the order the solve reads them,
// [tile][j / 2][8 columns][j % 2] (a lane fetches two consecutive coefficients with one 16-byte load) with one more
// entry holding 1 / (1 - c~_m c_{m-1}); a tile's table is one contiguous block fetched by a linear bulk copy.
//
// CTA = NWARP (1 or 2) solving warps + one copy warp, persistent, one per SM.  Three data buffers and two table
// buffers rotate over the CTA's tile sequence n = 0, 1, 2, ... (data buffer n % 3, table buffer n % 2, solved by warp
// n % NWARP): while two tiles are being solved the third buffer drains its store and takes the load of tile n + 3,
// both issued by the copy warp when a solving warp reports its tile done (mbarrier).  A single warp runs this loop at
// ~30 cycles per chain step (about 3 cycles per instruction: there is nothing to switch to), so the kernel is bound
// by the two tiles that fit beside the one in flight, not by HBM: measured 2.1-2.2 ms at 1024 x 1024 x 512
// (4.3-4.6 TB/s of algorithmic bytes) against 3.75 ms for the two sweeps.
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

#include <type_traits>

namespace flutas {

struct ThomasGeom {
    static constexpr int C = 8;                     // kx columns per tile
    static constexpr int NBUF = 3, NTAB = 2, B = 8;   // data buffers, table buffers, chain steps per register batch
    __host__ __device__ static int nzh(int nz) { return nz - nz / 2; }            // steps of the longer chain
    // per tile: entries j = 0 .. nzh (c_0 .. c_{nzh-1}, then f), two consecutive j packed per column so that a lane
    // fetches c_j, c_{j+1} with one 16-byte load: [j / 2][column][j % 2].  cw = coefficient columns per tile: 8 when the
    // real and imaginary part of a column share their eigenvalue (periodic x), 16 = (column, component) when they are
    // two different modes along x (non-periodic x, kernels_r2r.cuh)
    __host__ __device__ static size_t tab_doubles(int nz, int cw = C) { return (size_t)((nzh(nz) + 2) / 2) * 2 * cw; }
    // rows per TMA box (<= 256): the column is cut into equal boxes, so a buffer is at most one row per box longer than nz
    __host__ __device__ static int box_rows(int nz) { const int nb = (nz + 255) / 256; return (nz + nb - 1) / nb; }
    // a buffer holds whole boxes: the last one may hang over the end of the column (zero-filled, never stored)
    __host__ __device__ static size_t data_bytes(int nz) {
        return (size_t)((nz + box_rows(nz) - 1) / box_rows(nz)) * box_rows(nz) * C * 16;
    }
    // a warp's table buffer, with room for the 2B rows the forward loop requests past the end
    __host__ __device__ static size_t tab_stride(int nz, int cw = C) { return ((tab_doubles(nz, cw) + 2 * B * cw) * 8 + 127) / 128 * 128; }
    __host__ __device__ static int tab_index(int j, int col, int cw = C) { return (j >> 1) * 2 * cw + col * 2 + (j & 1); }
    __host__ static size_t smem_bytes(int nz, int cw = C) {
        return NBUF * data_bytes(nz) + NTAB * tab_stride(nz, cw) + 128;
    }
};

// one thread per coefficient column of the tiled table; true divisions (this runs once per plan).
// lam_x2[2 kx + component]: eigenvalue along x of the real (0) / imaginary (1) part of column kx; cw = 8 uses component 0.
// end_coef: first / last diagonal = -end_coef a + lam: 1 Neumann (R7), 3 Dirichlet (p = 0 on the boundary face).
// has_null: the (0, 0) mode is singular (no Dirichlet direction) and gets benign coefficients (thomas_singular_kernel).
__global__ void thomas_table_kernel(double *__restrict__ tab, int n_tiles_x, int ny, int nz, int nxh, int cw,
                                    const double *__restrict__ lam_x2, const double *__restrict__ lam_y, double inv_dz2,
                                    double end_coef, int has_null) {
    using G = ThomasGeom;
    const long long c = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const long long ncol = (long long)n_tiles_x * ny * cw;
    if (c >= ncol) return;
    const int cc = (int)(c % cw);
    const int col = cw == G::C ? cc : cc >> 1, comp = cw == G::C ? 0 : cc & 1;
    const long long tile = c / cw;
    const int tx = (int)(tile % n_tiles_x), jy = (int)(tile / n_tiles_x);
    const int kx = tx * G::C + col;
    const int nzh = G::nzh(nz), m = nz / 2;
    double *t = tab + tile * G::tab_doubles(nz, cw);
    if (kx >= nxh || (has_null && kx == 0 && comp == 0 && jy == 0)) {   // padding columns and the singular mode: benign values
        for (int j = 0; j < nzh; ++j) t[G::tab_index(j, cc, cw)] = 0.0;
        t[G::tab_index(nzh, cc, cw)] = 1.0;
        return;
    }
    const double lam = lam_x2[2 * kx + comp] + lam_y[jy];
    const double a = inv_dz2, b_end = -end_coef * inv_dz2 + lam, b_in = -2.0 * inv_dz2 + lam;
    double cj = a / b_end, c_m1 = 0.0;                // c_m1 = c_{m-1}
    t[G::tab_index(0, cc, cw)] = cj;
    if (m == 1) c_m1 = cj;
    for (int j = 1; j < nzh; ++j) {
        cj = a / (b_in - a * cj);
        t[G::tab_index(j, cc, cw)] = cj;
        if (j == m - 1) c_m1 = cj;
    }
    t[G::tab_index(nzh, cc, cw)] = 1.0 / (1.0 - cj * c_m1);   // cj = c_{nzh-1} = c~_m
}

struct ThomasArgs {
    const double *tab;
    int n_tiles_x, ny, nz;
    double dz2;               // 1 / a
    int has_null;             // the (0, 0) mode is left to thomas_singular_kernel
    // SCAT (z-slab decomposition, kernels.cuh PeerScatter): the solved tile goes to the ranks that own its planes
    int n_peers, nzl, srows;  // ranks, planes per rank, rows per store box (divides nzl, <= 256)
    int row0, nxh;            // this rank's first row of ky in the peers' slab spectra; valid kx columns
    const PeerScatter *sc;    // row_stride = plane of a slab spectrum (for the two halo planes, written with plain stores)
};
struct ThomasPeerMaps { CUtensorMap m[kMaxRanks]; };   // the peers' slab spectra, box {16, 1, srows}

template <int NWARP, int CW, bool SCAT = false>
__global__ void __launch_bounds__(32 * (NWARP + 1), 1) thomas_tma_kernel(const __grid_constant__ CUtensorMap tmap, ThomasArgs a,
                                                                         const __grid_constant__ ThomasPeerMaps pm) {
    using G = ThomasGeom;
    static_assert(CW == 8 || CW == 16, "coefficient columns per tile");
    extern __shared__ unsigned char smem_raw[];
    __shared__ uint64_t full_d[G::NBUF], full_c[G::NTAB], done[G::NBUF];

    const int nz = a.nz, nzh = G::nzh(nz), m = nz / 2;
    const int rows = G::box_rows(nz), nbox = (nz + rows - 1) / rows;
    const uint32_t box_bytes = (uint32_t)rows * G::C * 16u;
    const uint32_t tab_bytes = (uint32_t)G::tab_doubles(nz, CW) * 8u;
    unsigned char *base = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
    const uint32_t buf_stride = (uint32_t)nbox * box_bytes;   // = G::data_bytes(nz)
    unsigned char *tab_base = base + G::NBUF * buf_stride;
    const uint32_t tab_stride = (uint32_t)G::tab_stride(nz, CW);

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int col = lane & 7, comp = (lane >> 3) & 1, top = lane >> 4;   // top = 1: the chain that starts at k = nz-1
    const int cc = CW == 8 ? col : col * 2 + comp;                       // this lane's coefficient column
    const long long ntiles = (long long)a.n_tiles_x * a.ny;
    const long long my_tiles = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
    auto tile_of = [&](long long n) { return (long long)blockIdx.x + n * gridDim.x; };

    if (threadIdx.x == 0) {
        for (int b = 0; b < G::NBUF; ++b) mbar_init(&full_d[b], 1);
        for (int w = 0; w < G::NTAB; ++w) mbar_init(&full_c[w], 1);
        for (int b = 0; b < G::NBUF; ++b) mbar_init(&done[b], 1);
        fence_barrier_init();
        fence_proxy_async();
    }
    __syncthreads();

    auto issue_data = [&](long long n) {       // one lane
        const long long tile = tile_of(n);
        const int tx = (int)(tile % a.n_tiles_x), jy = (int)(tile / a.n_tiles_x);
        const int b = (int)(n % G::NBUF);
        mbar_arrive_expect_tx(&full_d[b], (uint32_t)nbox * box_bytes);
        for (int c = 0; c < nbox; ++c)
            tma_load_3d(base + b * buf_stride + c * box_bytes, &tmap, &full_d[b], tx * 2 * G::C, jy, c * rows);
    };
    auto issue_table = [&](long long n) {
        const int w = (int)(n % G::NTAB);
        mbar_arrive_expect_tx(&full_c[w], tab_bytes);
        bulk_load(tab_base + w * tab_stride, a.tab + tile_of(n) * G::tab_doubles(nz, CW), tab_bytes, &full_c[w]);
    };
    auto issue_store = [&](long long n) {
        const long long tile = tile_of(n);
        const int tx = (int)(tile % a.n_tiles_x), jy = (int)(tile / a.n_tiles_x);
        const int b = (int)(n % G::NBUF);
        if constexpr (SCAT) {
            // rows r nzl .. (r + 1) nzl - 1 of the tile are planes 1 .. nzl of rank r's slab spectrum
            for (int r = 0; r < a.n_peers; ++r)
                for (int c = 0; c < a.nzl; c += a.srows)
                    tma_store_3d(&pm.m[r], base + b * buf_stride + (uint32_t)(r * a.nzl + c) * (G::C * 16u), tx * 2 * G::C,
                                 a.row0 + jy, 1 + c);
        } else {
            for (int c = 0; c < nbox; ++c)
                tma_store_3d(&tmap, base + b * buf_stride + c * box_bytes, tx * 2 * G::C, jy, c * rows);
        }
        bulk_commit();
    };
    // SCAT: the planes next to a slab boundary also go to the neighbour's halo planes (walls: no wrap-around); 8 columns
    // x 2 (P - 1) rows, plain stores by the lanes of the copy warp
    auto store_halos = [&](long long n) {
        const long long tile = tile_of(n);
        const int tx = (int)(tile % a.n_tiles_x), jy = (int)(tile / a.n_tiles_x);
        const int b = (int)(n % G::NBUF);
        const double2 *sd = reinterpret_cast<const double2 *>(base + b * buf_stride);
        const long long plane_s = a.sc->row_stride, row_off = (long long)(a.row0 + jy) * a.sc->outer_stride;
        for (int item = threadIdx.x & 31; item < 2 * (a.n_peers - 1) * G::C; item += 32) {
            const int c = item % G::C, e = item / G::C, r = e >> 1, up = e & 1;   // boundary between ranks r and r + 1
            const int kx = tx * G::C + c;
            if (kx >= a.nxh) continue;
            // up = 0: the last plane of rank r -> plane 0 (below) of rank r + 1; up = 1: the first plane of rank r + 1 -> plane nzl + 1 of rank r
            const int row = (r + 1) * a.nzl - 1 + up;
            double2 *dst = up ? a.sc->base[r] + (long long)(a.nzl + 1) * plane_s : a.sc->base[r + 1];
            dst[row_off + kx] = sd[row * G::C + c];
        }
    };

    if (threadIdx.x == 0) {
        for (int n = 0; n < G::NBUF; ++n)
            if (n < my_tiles) issue_data(n);
        for (int n = 0; n < G::NTAB; ++n)
            if (n < my_tiles) issue_table(n);
    }

    const int cnt = top ? nzh : m;                     // steps of this lane's chain
    const double dz2 = a.dz2;
    if (warp == NWARP) {
        // ---- the copy warp: as tiles are reported solved (in order), write them back, refill the table buffer at
        //      once and the data buffer as soon as the store has drained it.  The solving warps never wait for a drain.
        if (SCAT || lane == 0) {
            for (long long n = 0; n < my_tiles; ++n) {
                mbar_wait(&done[n % G::NBUF], (uint32_t)(n / G::NBUF) & 1);
                if constexpr (SCAT) {
                    store_halos(n);
                    __syncwarp();          // every lane has read its halo rows before the buffer can be refilled
                }
                if (lane == 0) {
                    issue_store(n);
                    if (n + G::NTAB < my_tiles) issue_table(n + G::NTAB);
                    if (n + G::NBUF < my_tiles) {
                        bulk_wait_read<0>();
                        issue_data(n + G::NBUF);
                    }
                }
                if constexpr (SCAT) __syncwarp();
            }
            if (lane == 0) bulk_wait_all<0>();
        }
        return;
    }
    for (long long n = warp; n < my_tiles; n += NWARP) {
        const int b = (int)(n % G::NBUF);
        const int tb = (int)(n % G::NTAB);
        const uint32_t it_c = (uint32_t)(n / G::NTAB), it_d = (uint32_t)(n / G::NBUF);
        double *s = reinterpret_cast<double *>(base + b * buf_stride) + col * 2 + comp;   // element (row, col): s[row * 16]
        const double *ctab = reinterpret_cast<const double *>(tab_base + tb * tab_stride);
        const double2 *ct2 = reinterpret_cast<const double2 *>(ctab) + cc;      // (c_2q, c_2q+1): ct2[q * CW]
        auto c_at = [&](int j) { return ctab[G::tab_index(j, cc, CW)]; };
        // the singular (0,0) mode is left as it is (thomas_singular_kernel): the whole column, or its real part only
        const bool nostore = a.has_null && tile_of(n) == 0 && col == 0 && (CW == 8 || comp == 0);
        if (lane == 0 && n + G::NTAB < my_tiles)       // the table that takes this buffer next: on its way to L2 meanwhile
            bulk_prefetch_l2(a.tab + tile_of(n + G::NTAB) * G::tab_doubles(nz, CW), tab_bytes);
        mbar_wait(&full_c[tb], it_c & 1);
        mbar_wait(&full_d[b], it_d & 1);
        auto row_of = [&](int j) { return top ? nz - 1 - j : j; };
        const int ds = top ? -16 : 16;                 // doubles from one row of this chain to the next

        // ---- forward elimination.  Full batches of B steps, software-pipelined two batches deep so that the chain --
        //      one dependent FMA per step -- is the only thing a step waits for: iteration bt requests the operands
        //      of batch bt+2, forms e_j = d_j inv_j of batch bt+1 and runs the chain of batch bt.  No predicates
        //      (requests run up to 2B rows past the chain's end: still inside the tile / the padded table when
        //      m >= 4B).  The remainder is predicated.
        double g = 0.0;
        const int nfull = m >= 4 * G::B ? m / G::B : 0;    // m <= cnt: the same trip count in every lane
        if (nfull > 0) {
            double *sp = s + row_of(0) * 16;
            const double2 *cp = ct2;
            double ec[G::B], cc[G::B], dn[G::B];
            double2 cn[G::B / 2];
#pragma unroll
            for (int q = 0; q < G::B / 2; ++q) {
                const double2 c2 = cp[q * CW];
                cc[2 * q] = c2.x; cc[2 * q + 1] = c2.y;
                ec[2 * q] = sp[(2 * q) * ds] * (c2.x * dz2);
                ec[2 * q + 1] = sp[(2 * q + 1) * ds] * (c2.y * dz2);
            }
#pragma unroll
            for (int e = 0; e < G::B; ++e) dn[e] = sp[(G::B + e) * ds];
#pragma unroll
            for (int q = 0; q < G::B / 2; ++q) cn[q] = cp[(G::B / 2 + q) * CW];
#pragma unroll 2
            for (int bt = 0; bt < nfull; ++bt) {
                double d2[G::B], gv[G::B];
                double2 c2[G::B / 2];
#pragma unroll
                for (int e = 0; e < G::B; ++e) d2[e] = sp[(2 * G::B + e) * ds];
#pragma unroll
                for (int q = 0; q < G::B / 2; ++q) c2[q] = cp[(G::B + q) * CW];
#pragma unroll
                for (int e = 0; e < G::B; ++e) {
                    g = fma(-cc[e], g, ec[e]);             // the only dependent operation of a step
                    gv[e] = g;
                    const double cnx = (e & 1) ? cn[e >> 1].y : cn[e >> 1].x;
                    cc[e] = cnx;
                    ec[e] = dn[e] * (cnx * dz2);
                }
                if (!nostore) {
#pragma unroll
                    for (int e = 0; e < G::B; ++e) sp[e * ds] = gv[e];
                }
#pragma unroll
                for (int e = 0; e < G::B; ++e) dn[e] = d2[e];
#pragma unroll
                for (int q = 0; q < G::B / 2; ++q) cn[q] = c2[q];
                sp += G::B * ds;
                cp += (G::B / 2) * CW;
            }
        }
        for (int j0 = nfull * G::B; j0 < nzh; j0 += G::B) {
            double d[G::B], c[G::B];
#pragma unroll
            for (int e = 0; e < G::B; ++e) {
                const bool ok = j0 + e < cnt;              // a masked step is the identity map: d = 0, c = -1
                d[e] = ok ? s[row_of(j0 + e) * 16] : 0.0;
                c[e] = ok ? c_at(j0 + e) : -1.0;
            }
#pragma unroll
            for (int e = 0; e < G::B; ++e) {
                g = fma(-c[e], g, d[e] * (c[e] * dz2));
                d[e] = g;
            }
            if (!nostore) {
#pragma unroll
                for (int e = 0; e < G::B; ++e)
                    if (j0 + e < cnt) s[row_of(j0 + e) * 16] = d[e];
            }
        }
        // ---- the 2 x 2 system where the two chains meet: g = g_{m-1} (bottom chain) or h_m (top chain)
        const double other = __shfl_xor_sync(0xffffffffu, g, 16);
        const double g_lo = top ? other : g, h_hi = top ? g : other;
        const double c_hi = c_at(nzh - 1), c_lo = c_at(m - 1), f = c_at(nzh);
        const double x_m = (h_hi - c_hi * g_lo) * f;
        double x = top ? x_m : fma(-c_lo, x_m, g_lo);      // x_{cnt-1} of this chain
        if (!nostore) s[row_of(cnt - 1) * 16] = x;
        // ---- back-substitution outwards: j = cnt-2 .. 0.  One step alone if that makes the next j odd (coefficient
        //      pairs are (c_2q, c_2q+1)), then full batches (operands requested one batch ahead; the last full batch
        //      requests nothing), then the predicated remainder
        int jb = cnt - 2;
        if (jb >= 0 && (jb & 1) == 0) {
            x = fma(-c_at(jb), x, s[row_of(jb) * 16]);
            if (!nostore) s[row_of(jb) * 16] = x;
            --jb;
        }
        const int nfull_b = m >= 4 * G::B ? (m - 2) / G::B : 0;   // every lane has at least m - 2 steps left
        if (nfull_b > 0) {
            double *sp = s + row_of(jb) * 16;
            const double2 *cp = ct2 + (jb >> 1) * CW;   // jb is odd: the pair (c_{jb-1}, c_jb)
            double dn[G::B];
            double2 cn[G::B / 2];
#pragma unroll
            for (int e = 0; e < G::B; ++e) dn[e] = sp[-e * ds];
#pragma unroll
            for (int q = 0; q < G::B / 2; ++q) cn[q] = cp[-q * CW];
            auto batch = [&](auto request_next) {
                double d[G::B];
                double2 c[G::B / 2];
#pragma unroll
                for (int e = 0; e < G::B; ++e) d[e] = dn[e];
#pragma unroll
                for (int q = 0; q < G::B / 2; ++q) c[q] = cn[q];
                if (decltype(request_next)::value) {
#pragma unroll
                    for (int e = 0; e < G::B; ++e) dn[e] = sp[-(G::B + e) * ds];
#pragma unroll
                    for (int q = 0; q < G::B / 2; ++q) cn[q] = cp[-(G::B / 2 + q) * CW];
                }
#pragma unroll
                for (int e = 0; e < G::B; ++e) {           // step e: j = jb - e, odd j first
                    x = fma(-((e & 1) ? c[e >> 1].x : c[e >> 1].y), x, d[e]);
                    d[e] = x;
                }
                if (!nostore) {
#pragma unroll
                    for (int e = 0; e < G::B; ++e) sp[-e * ds] = d[e];
                }
                sp -= G::B * ds;
                cp -= (G::B / 2) * CW;
            };
#pragma unroll 2
            for (int bt = 0; bt + 1 < nfull_b; ++bt) batch(std::true_type{});
            batch(std::false_type{});
        }
        for (int j0 = jb - nfull_b * G::B; j0 >= 0; j0 -= G::B) {
            double d[G::B], c[G::B];
#pragma unroll
            for (int e = 0; e < G::B; ++e) {
                const bool ok = j0 - e >= 0;
                d[e] = ok ? s[row_of(j0 - e) * 16] : 0.0;
                c[e] = ok ? c_at(j0 - e) : -1.0;
            }
#pragma unroll
            for (int e = 0; e < G::B; ++e) {
                x = fma(-c[e], x, d[e]);
                d[e] = x;
            }
            if (!nostore) {
#pragma unroll
                for (int e = 0; e < G::B; ++e)
                    if (j0 - e >= 0) s[row_of(j0 - e) * 16] = d[e];
            }
        }
        // ---- report the tile solved (the copy warp writes it back and refills the buffers)
        fence_proxy_async();
        __syncwarp();
        if (lane == 0) mbar_arrive(&done[b]);
    }
}

}  // namespace flutas
