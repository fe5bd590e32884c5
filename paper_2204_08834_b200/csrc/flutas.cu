// flutas.cu -- plan, launch sequence and C ABI of libflutas_b200.so (see include/flutas.h).
//
// build: nvcc -O3 -std=c++17 -gencode arch=compute_100a,code=sm_100a -lineinfo -Xcompiler -fPIC -shared -- see ../build.py
//        No --use_fast_math.  Host-side tables use IEEE divisions; on the device the face-density and eigenvalue
//        reciprocals are rcp.approx.ftz.f64 + two Newton steps (<= ~1 ulp; rcp_density, rcp_normal), everything else
//        is plain fp64 add / mul / fma.
#include "flutas.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <vector>

#include "kernels.cuh"
#include "momentum_launch.h"
#include "kernels_r2r.cuh"
#include "kernels_rhs.cuh"
#include "kernels_thomas.cuh"
#include "kernels_tma.cuh"
#include "kernels_vof.cuh"
#include "vof_launch.h"
#include "kernels_x.cuh"
#include "kernels_y16.cuh"

using namespace flutas;

// ------------------------------------------------------------------------------------ errors
static thread_local char g_err[512] = "";
static thread_local int g_err_code = FLUTAS_OK;

static int fail(int code, const char *fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
    g_err_code = code;
    return code;
}
#define CUDA_TRY(expr)                                                                         \
    do {                                                                                       \
        cudaError_t e_ = (expr);                                                               \
        if (e_ != cudaSuccess)                                                                 \
            return fail(e_ == cudaErrorMemoryAllocation ? FLUTAS_ERR_ALLOC : FLUTAS_ERR_CUDA,  \
                        "%s: %s", #expr, cudaGetErrorString(e_));                              \
    } while (0)

// the library's other translation units (vof_noalloc.cu) record their failures in the same thread-local slot (vof_launch.h)
int flutas::report_error(int code, const char *msg) { return fail(code, "%s", msg); }

extern "C" const char *flutas_last_error(void) { return g_err; }
extern "C" int flutas_last_error_code(void) { return g_err_code; }

// -------------------------------------------------------------------------------------- plan
enum KernelId { K_RHS = 0, K_FFTX, K_FFTY, K_Z, K_ZS, K_IFFTY, K_IFFTX, K_CORR, K_MAX };

static const int kMaxPendingSteps = 256;

struct flutas_plan {
    int nx, ny, nz, bc_z;        // bc_z: FLUTAS_BC_Z_PERIODIC (transform along z) or FLUTAS_BC_Z_WALL (elimination along z)
    int bc[3];                   // the conditions as given, per direction: FLUTAS_BC_PERIODIC / _NEUMANN / _DIRICHLET
    int xsplit;                  // x is not periodic: columns of the spectrum hold two real modes (kernels_r2r.cuh)
    int y_r2r;                   // y expansion: 0 complex FFT, 1 half-complex (periodic y under xsplit), 2 cosine, 3 sine
    int has_null;                // no Dirichlet direction: the (0,0,0) mode is singular, zero-mean gauge (R5)
    double end_coef_z;           // first / last diagonal of the elimination along z: -end_coef/dz^2 + lam (1 Neumann, 3 Dirichlet)
    double2 *wq_x, *wq_y;        // e^{-i pi k / (2n)}, k = 0 .. n/2, of the cosine / sine expansions
    double *lam_x2;              // eigenvalue along x per (column, component): 2 * pitch entries
    double lx, ly, lz, rho1, rho2;
    GridParams grid;
    int n2, nxh, pitch;          // nx/2, nx/2+1, padded row length of the half-spectrum (multiple of 8)
    long long npts, nspec;       // nx*ny*nz, plane*nz
    long long plane;             // complex elements from one plane of the half-spectrum to the next: pitch * (ny + pad rows)
    // device tables
    double2 *tw_x, *tw_y, *tw_z;
    double *lam_x, *lam_y, *lam_z;   // storage (permuted) order
    // device workspace
    double2 *spec;
    double *rhs, *up, *vp, *wp, *cp;
    double *sing_coef;           // wall: 1/(b_k - a c'_{k-1}) and c'_k of the singular (0,0) column, interleaved
    double *ttab;                // wall: elimination coefficients of the one-pass solve, [tile][j][8] (kernels_thomas.cuh)
    int thomas_warps;            // solving warps per CTA of the one-pass kernel (1 or 2)
    int thomas_variant;          // wall: 1 = one-pass shared-memory solve (nz <= 512), 0 = two sweeps through HBM
    size_t bytes;                // workspace bytes this plan needs (layout: plan_carve)
    void *ws_base;               // start of the workspace in use (plan-owned or the caller's), nullptr = none yet
    bool ws_owned;               // true: ws_base came from cudaMalloc here and is freed by the plan
    bool cp_owned;               // the c' array of the two-sweep option was allocated on demand (outside the workspace)
    // staging for the host entry point
    double *stage[6];
    // launch list
    int n_launch;
    int launch_ids[K_MAX];
    // tuning
    int y_cols, z_cols;          // tile width (columns of kx) of the strided passes: 8, or 4 for lines of >= 1024
    int rhs_kc;                  // planes one thread of the RHS kernel marches through
    int chunk;                   // planes per launch group of the step (0 = whole grid per kernel)
    int overlap;                 // chunked only: 1 = the three kernels of a group run on three internal streams (low, mid, high
                                 // priority; producer -> consumer), so groups overlap and tails are filled
    cudaStream_t lane[3];        // internal streams, created on first use
    cudaEvent_t ev_fork, *ev_dep;   // fork from the caller's stream; ev_dep[2 * chunk_index + {0, 1}]
    int n_dep;
    int y16;                     // ny = 1024: 1 = register-resident 16 x 8 x 8 kernel (kernels_y16.cuh), 0 = fft_tma1_kernel on 4 columns
    int num_sms;
    CUtensorMap map_y, map_z;    // boxes {2*y_cols, rows, 1} and {2*z_cols, 1, rows} over the half-spectrum
    // timing
    int timing;
    cudaEvent_t *events;         // kMaxPendingSteps * (n_launch + 1)
    int pending;
    // z-slab decomposition (flutas_slab_plan, flutas_slab.inl): a rank owns two plans of reduced geometry
    int role;                    // ROLE_FULL, ROLE_SLAB (nz = its planes + 2 halo planes: real-space kernels, x and y
                                 // transforms), ROLE_ZLOCAL (ny = its share of the ky rows: the z stage)
    int ny_full, row0;           // ROLE_ZLOCAL: rows of the whole spectrum and the first one this plan holds
    double2 *spec_ext;           // ROLE_SLAB / ROLE_ZLOCAL: the spectrum lives in the exchange buffer, not in the workspace
    PeerScatter *sc_dev;         // device copy of the store descriptor of the last forward y pass / of the z stage
    ThomasPeerMaps *tpm;         // ROLE_ZLOCAL, wall: tensor maps of the peers' slab spectra (host)
    int sc_nzl, sc_srows, sc_npeers;
    int mom_ty16;                // momentum kernel: tiles of 32 x 16 cells (one CTA per SM) instead of 32 x 8 (two)
};
enum { ROLE_FULL = 0, ROLE_SLAB = 1, ROLE_ZLOCAL = 2 };

static const char *kKernelNames[K_MAX] = {"splitting_rhs", "fft_x_r2c", "fft_y_fwd", "z_solve", "z_singular",
                                          "fft_y_inv", "fft_x_c2r", "correction"};

static bool is_pow2(int n) { return n > 0 && (n & (n - 1)) == 0; }

// storage position -> frequency for the run-time length n (same digit order as fft_core.cuh)
static int host_freq_of_pos(int n, int pos) {
    int lg = 0;
    while ((1 << lg) < n) ++lg;
    const int P = (lg + 2) / 3, rlast = 1 << (lg - 3 * (P - 1));
    int k = 0, w = 1, m = n;
    for (int p = 1; p <= P; ++p) {
        const int r = p < P ? 8 : rlast;
        m /= r;
        k += ((pos / m) % r) * w;
        w *= r;
    }
    return k;
}

static void host_twiddles(int n, std::vector<double2> &t) {
    t.resize(n);
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < n; ++m) {
        const long double a = -two_pi * (long double)m / (long double)n;
        t[m] = make_double2((double)cosl(a), (double)sinl(a));
    }
}
// eigenvalue of the periodic second difference, lambda(m) = -2 (1 - cos(2 pi m / n)) / d^2  (R6)
static double host_lambda(int m, int n, double d) {
    const long double two_pi = 6.283185307179586476925286766559005768L;
    return (double)(-2.0L * (1.0L - cosl(two_pi * (long double)m / (long double)n))) / (d * d);
}

// eigenvalue of mode index k of the cosine (Neumann) / sine (Dirichlet) expansion AS THE KERNELS INDEX IT: the cosine
// transform index k is mode k; the sine expansion is computed as a cosine transform of the sign-flipped line read
// backwards, so transform index k is sine mode n-1-k, frequency n-k:  lambda = -2 (1 - cos(pi f / n)) / d^2
static double host_lambda_r2r(int k, int n, double d, int bc) {
    const long double pi = 3.141592653589793238462643383279502884L;
    const int f = bc == FLUTAS_BC_NEUMANN ? k : n - k;
    return (double)(-2.0L * (1.0L - cosl(pi * (long double)f / (long double)n))) / (d * d);
}
static void host_wq(int n, std::vector<double2> &t) {
    t.resize(n / 2 + 1);
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int k = 0; k <= n / 2; ++k) {
        const long double a = -pi * (long double)k / (long double)(2 * n);
        t[k] = make_double2((double)cosl(a), (double)sinl(a));
    }
}

// eigenvalues along y in the storage order of the transform in use (the 16 x 8 x 8 kernel has its own digit order)
static int upload_lam_y(flutas_plan *pl) {
    std::vector<double> lam(pl->ny);
    const int nyf = pl->ny_full;                 // == ny except for the z-local plan of a slab decomposition (rows row0 ..)
    const double dy = pl->ly / nyf;
    for (int pos = 0; pos < pl->ny; ++pos) {
        const int k = pl->y16 ? y1024_freq_of_pos(pos) : host_freq_of_pos(nyf, pl->row0 + pos);
        lam[pos] = pl->bc[1] == FLUTAS_BC_PERIODIC ? host_lambda(k, nyf, dy) : host_lambda_r2r(k, nyf, dy, pl->bc[1]);
    }
    CUDA_TRY(cudaMemcpy(pl->lam_y, lam.data(), sizeof(double) * pl->ny, cudaMemcpyHostToDevice));
    return FLUTAS_OK;
}

// elimination coefficients of the one-pass wall solve (they depend on lam_x + lam_y in storage order)
static int thomas_cw(const flutas_plan *pl) { return pl->xsplit ? 16 : ThomasGeom::C; }
static int build_thomas_table(flutas_plan *pl) {
    const int n_tiles_x = (pl->nxh + ThomasGeom::C - 1) / ThomasGeom::C, cw = thomas_cw(pl);
    const long long ncol = (long long)n_tiles_x * pl->ny * cw;
    const double inv_dz = 1.0 / (pl->lz / pl->nz);
    thomas_table_kernel<<<(unsigned)((ncol + 127) / 128), 128>>>(pl->ttab, n_tiles_x, pl->ny, pl->nz, pl->nxh, cw, pl->lam_x2,
                                                               pl->lam_y, inv_dz * inv_dz, pl->end_coef_z, pl->has_null);
    CUDA_TRY(cudaGetLastError());
    CUDA_TRY(cudaDeviceSynchronize());
    return FLUTAS_OK;
}

template <typename T> static int upload(T **dst, const std::vector<T> &src, size_t *bytes) {
    CUDA_TRY(cudaMalloc((void **)dst, src.size() * sizeof(T)));
    CUDA_TRY(cudaMemcpy(*dst, src.data(), src.size() * sizeof(T), cudaMemcpyHostToDevice));
    *bytes += src.size() * sizeof(T);
    return FLUTAS_OK;
}

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link-time dependency on libcuda)
typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                  const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static int make_spectrum_map(flutas_plan *pl, CUtensorMap *map, int cols, int line_dim, int n, int box_rows = 0,
                             void *base = nullptr) {
    static EncodeTiledFn encode = nullptr;
    if (!encode) {
        void *fn = nullptr;
        cudaDriverEntryPointQueryResult q;
        CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
        if (!fn || q != cudaDriverEntryPointSuccess) return fail(FLUTAS_ERR_CUDA, "cuTensorMapEncodeTiled is not available");
        encode = (EncodeTiledFn)fn;
    }
    const cuuint32_t rows = (cuuint32_t)(box_rows ? box_rows : (n < 256 ? n : 256));
    const cuuint64_t gdim[3] = {(cuuint64_t)2 * pl->nxh, (cuuint64_t)pl->ny, (cuuint64_t)pl->nz};
    const cuuint64_t gstride[2] = {(cuuint64_t)pl->pitch * 16, (cuuint64_t)pl->plane * 16};
    const cuuint32_t box[3] = {(cuuint32_t)(2 * cols), line_dim == 1 ? rows : 1u, line_dim == 2 ? rows : 1u};
    const cuuint32_t estr[3] = {1, 1, 1};
    const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, base ? base : (void *)pl->spec, gdim, gstride, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                              cols >= 8 ? CU_TENSOR_MAP_L2_PROMOTION_L2_128B : CU_TENSOR_MAP_L2_PROMOTION_L2_64B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) return fail(FLUTAS_ERR_CUDA, "cuTensorMapEncodeTiled failed with code %d", (int)r);
    return FLUTAS_OK;
}

static int plan_make_maps(flutas_plan *pl) {
    if (pl->role != ROLE_ZLOCAL)
        if (int rc = make_spectrum_map(pl, &pl->map_y, pl->y16 ? Y16Geom::C : pl->y_cols, 1, pl->ny)) return rc;
    if (pl->role == ROLE_SLAB) return FLUTAS_OK;
    if (pl->bc_z == FLUTAS_BC_Z_PERIODIC) {
        if (int rc = make_spectrum_map(pl, &pl->map_z, pl->z_cols, 2, pl->nz)) return rc;
    } else if (pl->thomas_variant == 1) {
        if (int rc = make_spectrum_map(pl, &pl->map_z, ThomasGeom::C, 2, pl->nz, ThomasGeom::box_rows(pl->nz))) return rc;
    }
    return FLUTAS_OK;
}

// ---- sizes: everything that follows from (nx, ny, nz, bc_z) alone, no device needed
static bool sizes_supported(int nx, int ny, int nz, int bc_x, int bc_y, int bc_z) {
    const auto bc_ok = [](int b) { return b == FLUTAS_BC_PERIODIC || b == FLUTAS_BC_NEUMANN || b == FLUTAS_BC_DIRICHLET; };
    if (!bc_ok(bc_x) || !bc_ok(bc_y) || !bc_ok(bc_z)) return false;
    if (!is_pow2(nx) || nx < 8 || nx > 2048 || !is_pow2(ny) || ny < 8 || ny > 2048) return false;
    const bool xsplit = bc_x != FLUTAS_BC_PERIODIC;
    if (xsplit) {
        // cosine / sine expansion along x: staged kernels for nx = 16 .. 1024; the z stage must then be the one-pass
        // elimination with per-component coefficients (no transform along z; the column tile and its coefficient
        // table must fit in shared memory: nz <= 444)
        if (nx < 16 || nx > 1024) return false;
        if (bc_z == FLUTAS_BC_PERIODIC || nz < 2 || ThomasGeom::smem_bytes(nz, 16) > 227 * 1024) return false;   // nz <= 444
    }
    if ((xsplit || bc_y != FLUTAS_BC_PERIODIC) && ny > 1024) return false;   // the one-butterfly-per-thread y kernel
    if (bc_z != FLUTAS_BC_PERIODIC) return nz >= 2 && nz <= 4096;
    return is_pow2(nz) && nz >= 8 && nz <= 2048;
}

static size_t align_up(size_t x) { return (x + 1023) / 1024 * 1024; }

// Workspace layout, in this order, every part 1024-byte aligned:  spec | rhs | u' | v' | w' | wall: table or c'
struct WsLayout {
    size_t spec, rhs, up, vp, wp, zaux, total;
};
static WsLayout plan_layout(const flutas_plan *pl) {
    const size_t fb = sizeof(double) * (size_t)pl->npts, sb = sizeof(double2) * (size_t)pl->nspec;
    WsLayout w{};
    size_t o = 0;
    w.spec = o; if (pl->role == ROLE_FULL) o += align_up(sb);      // slab plans: the spectrum lives in the exchange buffer
    w.rhs = o; if (pl->role != ROLE_ZLOCAL) o += align_up(fb);
    w.up = o; if (pl->role != ROLE_ZLOCAL) o += align_up(fb);
    w.vp = o; if (pl->role != ROLE_ZLOCAL) o += align_up(fb);
    w.wp = o; if (pl->role != ROLE_ZLOCAL) o += align_up(fb);
    w.zaux = o;
    if (pl->bc_z == FLUTAS_BC_Z_WALL && pl->role != ROLE_SLAB) {
        if (ThomasGeom::smem_bytes(pl->nz, thomas_cw(pl)) <= 227 * 1024) {   // coefficient table of the one-pass solve
            const int n_tiles_x = (pl->nxh + ThomasGeom::C - 1) / ThomasGeom::C;
            o += align_up(sizeof(double) * ThomasGeom::tab_doubles(pl->nz, thomas_cw(pl)) * (size_t)n_tiles_x * pl->ny);
        } else {                                              // c' of the two sweeps
            o += align_up(sb / 2);
        }
    }
    w.total = o;
    return w;
}

static void plan_geometry(flutas_plan *pl) {
    const int nx = pl->nx, ny = pl->ny, nz = pl->nz;
    pl->n2 = nx / 2;
    pl->xsplit = pl->bc[0] != FLUTAS_BC_PERIODIC;
    pl->nxh = pl->xsplit ? nx / 2 : nx / 2 + 1;      // valid columns: nx/2 split columns, or kx = 0 .. nx/2
    pl->pitch = nx / 2 + 8;
    pl->npts = (long long)nx * ny * nz;
    // One unused row per plane, so that the stride of a line along z is an odd multiple of the row size instead of
    // (nx/2 + 8) * 16 bytes times a power of two.  Measured effect on the z stage: +3-5 % at 512^3, none at
    // 1024 x 1024 x 512 (the memory system's own address hashing already spreads such strides); kept because it is free.
    pl->plane = (long long)pl->pitch * (ny + 1);
    pl->nspec = pl->plane * nz;
    pl->bytes = plan_layout(pl).total;
}

// point the plan at a workspace (device memory of at least pl->bytes) and (re)build what lives in it or refers to it
static int plan_attach_workspace(flutas_plan *pl, void *base, bool owned) {
    const WsLayout w = plan_layout(pl);
    char *b = (char *)base;
    pl->ws_base = base;
    pl->ws_owned = owned;
    pl->spec = pl->role == ROLE_FULL ? (double2 *)(b + w.spec) : pl->spec_ext;
    pl->rhs = (double *)(b + w.rhs);
    pl->up = (double *)(b + w.up);
    pl->vp = (double *)(b + w.vp);
    pl->wp = (double *)(b + w.wp);
    if (!pl->cp_owned) pl->cp = nullptr;
    pl->ttab = nullptr;
    // padding columns / the pad row of the spectrum are read (never used) by the strided kernels: keep them finite
    CUDA_TRY(cudaMemset(pl->spec, 0, sizeof(double2) * (size_t)pl->nspec));
    if (pl->bc_z == FLUTAS_BC_Z_WALL && pl->role != ROLE_SLAB) {
        if (ThomasGeom::smem_bytes(pl->nz, thomas_cw(pl)) <= 227 * 1024) {
            pl->ttab = (double *)(b + w.zaux);
            if (int rc = build_thomas_table(pl)) return rc;
        } else if (!pl->cp_owned) {
            pl->cp = (double *)(b + w.zaux);
        }
    }
    return plan_make_maps(pl);
}

static void plan_detach_workspace(flutas_plan *pl) {
    if (pl->ws_owned && pl->ws_base) cudaFree(pl->ws_base);
    pl->ws_base = nullptr;
    pl->ws_owned = false;
    pl->spec = nullptr;
    pl->rhs = pl->up = pl->vp = pl->wp = pl->ttab = nullptr;
    if (!pl->cp_owned) pl->cp = nullptr;
}

static int plan_build(flutas_plan *pl, unsigned flags) {
    const int nx = pl->nx, ny = pl->ny, nz = pl->nz;
    const bool wall = pl->bc_z == FLUTAS_BC_Z_WALL && pl->role != ROLE_SLAB;   // a slab plan has no z stage
    const double dx = pl->lx / nx, dy = pl->ly / pl->ny_full, dz = pl->lz / nz;
    const bool same_rho = pl->rho1 == pl->rho2;    // (1 - rho0/rho_f) is then exactly 0 (flux_coef)
    pl->grid = GridParams{nx, ny, nz, pl->bc[2] == FLUTAS_BC_NEUMANN ? 1 : 0, 1.0 / dx, 1.0 / dy, 1.0 / dz, pl->rho1, pl->rho2,
                          pl->rho1 < pl->rho2 ? pl->rho1 : pl->rho2, 2.0, 1.0, same_rho ? 0.0 : 1.0,
                          pl->bc[0] == FLUTAS_BC_NEUMANN ? 1 : 0, pl->bc[1] == FLUTAS_BC_NEUMANN ? 1 : 0};
    plan_geometry(pl);
    pl->has_null = pl->bc[0] != FLUTAS_BC_DIRICHLET && pl->bc[1] != FLUTAS_BC_DIRICHLET && pl->bc[2] != FLUTAS_BC_DIRICHLET &&
                   pl->row0 == 0;                  // the (0, 0) column is on the rank that holds row 0
    pl->end_coef_z = pl->bc[2] == FLUTAS_BC_DIRICHLET ? 3.0 : 1.0;
    pl->y_r2r = pl->bc[1] == FLUTAS_BC_NEUMANN ? 2 : (pl->bc[1] == FLUTAS_BC_DIRICHLET ? 3 : (pl->xsplit ? 1 : 0));

    size_t tb = 0;   // table bytes (not part of the workspace)
    std::vector<double2> t;
    host_twiddles(nx, t);
    if (int rc = upload(&pl->tw_x, t, &tb)) return rc;
    host_twiddles(ny, t);
    if (int rc = upload(&pl->tw_y, t, &tb)) return rc;
    if (!wall && pl->role != ROLE_SLAB) {
        host_twiddles(nz, t);
        if (int rc = upload(&pl->tw_z, t, &tb)) return rc;
    }
    std::vector<double> lam(pl->pitch, 1.0);
    for (int k = 0; k <= pl->n2; ++k) lam[k] = host_lambda(k, nx, dx);   // x columns are stored in natural order
    if (int rc = upload(&pl->lam_x, lam, &tb)) return rc;
    {   // the same per (column, component).  Split columns (kernels_r2r.cuh): column k = (mode k, mode nx - k), column 0 = (0, nx/2)
        std::vector<double> lam2(2 * (size_t)pl->pitch, 1.0);
        for (int k = 0; k < pl->nxh; ++k) {
            if (!pl->xsplit) lam2[2 * k] = lam2[2 * k + 1] = lam[k];
            else {
                lam2[2 * k] = host_lambda_r2r(k, nx, dx, pl->bc[0]);
                lam2[2 * k + 1] = host_lambda_r2r(k == 0 ? nx / 2 : nx - k, nx, dx, pl->bc[0]);
            }
        }
        if (int rc = upload(&pl->lam_x2, lam2, &tb)) return rc;
    }
    if (pl->xsplit) {
        host_wq(nx, t);
        if (int rc = upload(&pl->wq_x, t, &tb)) return rc;
    }
    if (pl->y_r2r >= 2) {
        host_wq(ny, t);
        if (int rc = upload(&pl->wq_y, t, &tb)) return rc;
    }
    pl->y16 = (ny == Y16Geom::N && pl->y_r2r == 0 && pl->role == ROLE_FULL) ? 1 : 0;
    CUDA_TRY(cudaMalloc((void **)&pl->lam_y, sizeof(double) * ny));
    if (int rc = upload_lam_y(pl)) return rc;
    if (!wall && pl->role != ROLE_SLAB) {
        lam.assign(nz, 0.0);
        for (int pos = 0; pos < nz; ++pos) lam[pos] = host_lambda(host_freq_of_pos(nz, pos), nz, dz);
        if (int rc = upload(&pl->lam_z, lam, &tb)) return rc;
    }
    if (wall) {
        // the (0,0) column: lam = 0; the elimination coefficients do not depend on the data (same recurrence, same
        // IEEE divisions as a per-step evaluation would do)
        std::vector<double> sc(2 * (size_t)nz, 0.0);
        const double a = (1.0 / dz) * (1.0 / dz), b_end = -a, b_in = -2.0 * a;   // as GridParams::inv_dz squared (Neumann: singular)
        double inv = 1.0 / b_end, cpv = a * inv;
        sc[0] = inv; sc[1] = cpv;
        for (int k = 1; k <= nz - 2; ++k) {
            inv = 1.0 / (b_in - a * cpv);
            cpv = a * inv;
            sc[2 * k] = inv; sc[2 * k + 1] = cpv;
        }
        sc[2 * (size_t)nz - 1] = a;
        if (int rc = upload(&pl->sing_coef, sc, &tb)) return rc;
        pl->thomas_variant = ThomasGeom::smem_bytes(nz, thomas_cw(pl)) <= 227 * 1024 ? 1 : 0;
        pl->thomas_warps = 2;
    }

    int n = 0;
    pl->launch_ids[n++] = K_RHS;
    pl->launch_ids[n++] = K_FFTX;
    pl->launch_ids[n++] = K_FFTY;
    pl->launch_ids[n++] = K_Z;
    if (wall && pl->has_null) pl->launch_ids[n++] = K_ZS;
    pl->launch_ids[n++] = K_IFFTY;
    pl->launch_ids[n++] = K_IFFTX;
    pl->launch_ids[n++] = K_CORR;
    pl->n_launch = n;
    pl->y_cols = ny >= 1024 ? 4 : 8;
    pl->z_cols = nz >= 1024 ? 4 : 8;
    pl->rhs_kc = 32;
    pl->mom_ty16 = 1;
    int dev = 0;
    CUDA_TRY(cudaGetDevice(&dev));
    CUDA_TRY(cudaDeviceGetAttribute(&pl->num_sms, cudaDevAttrMultiProcessorCount, dev));
    if (flags & FLUTAS_PLAN_CALLER_WORKSPACE) return FLUTAS_OK;   // flutas_plan_set_workspace supplies it
    void *base = nullptr;
    CUDA_TRY(cudaMalloc(&base, pl->bytes));
    if (int rc = plan_attach_workspace(pl, base, true)) return rc;
    return FLUTAS_OK;
}

extern "C" flutas_plan *flutas_plan_create_ex(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y,
                                              int bc_z, double rho1, double rho2, unsigned flags) {
    for (int b : {bc_x, bc_y, bc_z})
        if (b != FLUTAS_BC_PERIODIC && b != FLUTAS_BC_NEUMANN && b != FLUTAS_BC_DIRICHLET) {
            fail(FLUTAS_ERR_INVALID_ARG, "boundary conditions must be FLUTAS_BC_PERIODIC, FLUTAS_BC_NEUMANN (wall) or FLUTAS_BC_DIRICHLET");
            return nullptr;
        }
    if (flags & ~(unsigned)FLUTAS_PLAN_CALLER_WORKSPACE) {
        fail(FLUTAS_ERR_INVALID_ARG, "unknown flag bits 0x%x", flags);
        return nullptr;
    }
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0) || !std::isfinite(lx + ly + lz)) {
        fail(FLUTAS_ERR_INVALID_ARG, "box lengths must be positive and finite");
        return nullptr;
    }
    if (!(rho1 >= 1e-100 && rho1 <= 1e100) || !(rho2 >= 1e-100 && rho2 <= 1e100)) {
        fail(FLUTAS_ERR_INVALID_ARG, "densities must lie in [1e-100, 1e100]");
        return nullptr;
    }
    if (!sizes_supported(nx, ny, nz, bc_x, bc_y, bc_z)) {
        fail(FLUTAS_ERR_UNSUPPORTED_SIZE,
             "unsupported grid %d x %d x %d with conditions (%d, %d, %d): nx, ny powers of two in [8,2048]; nz a power of two "
             "in [8,2048] (periodic z) or any value in [2,4096]; non-periodic y: ny <= 1024; non-periodic x: nx in [16,1024], "
             "ny <= 1024, z not periodic and nz <= 444", nx, ny, nz, bc_x, bc_y, bc_z);
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        fail(FLUTAS_ERR_CUDA, "no CUDA device available (there is no CPU fallback)");
        return nullptr;
    }
    flutas_plan *pl = new (std::nothrow) flutas_plan();
    if (!pl) {
        fail(FLUTAS_ERR_ALLOC, "host allocation failed");
        return nullptr;
    }
    memset(pl, 0, sizeof(*pl));
    pl->nx = nx; pl->ny = ny; pl->nz = nz;
    pl->ny_full = ny;
    pl->bc[0] = bc_x; pl->bc[1] = bc_y; pl->bc[2] = bc_z;
    pl->bc_z = bc_z == FLUTAS_BC_PERIODIC ? FLUTAS_BC_Z_PERIODIC : FLUTAS_BC_Z_WALL;
    pl->lx = lx; pl->ly = ly; pl->lz = lz; pl->rho1 = rho1; pl->rho2 = rho2;
    if (plan_build(pl, flags) != FLUTAS_OK) {
        flutas_plan_destroy(pl);   // keeps g_err of the failure
        return nullptr;
    }
    return pl;
}

extern "C" flutas_plan *flutas_plan_create(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                                           double rho1, double rho2) {
    return flutas_plan_create_ex(nx, ny, nz, lx, ly, lz, FLUTAS_BC_PERIODIC, FLUTAS_BC_PERIODIC, bc_z, rho1, rho2, 0u);
}

extern "C" size_t flutas_workspace_bytes(int nx, int ny, int nz, int bc_x, int bc_y, int bc_z) {
    if (!sizes_supported(nx, ny, nz, bc_x, bc_y, bc_z)) return 0;
    flutas_plan tmp;
    memset(&tmp, 0, sizeof(tmp));
    tmp.nx = nx; tmp.ny = ny; tmp.nz = nz;
    tmp.ny_full = ny;
    tmp.bc[0] = bc_x; tmp.bc[1] = bc_y; tmp.bc[2] = bc_z;
    tmp.bc_z = bc_z == FLUTAS_BC_PERIODIC ? FLUTAS_BC_Z_PERIODIC : FLUTAS_BC_Z_WALL;
    plan_geometry(&tmp);
    return tmp.bytes;
}

extern "C" int flutas_plan_set_workspace(flutas_plan *pl, void *dev_ptr, size_t bytes) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (dev_ptr) {
        if (((size_t)dev_ptr) & 255) return fail(FLUTAS_ERR_INVALID_ARG, "the workspace must be 256-byte aligned");
        if (bytes < pl->bytes)
            return fail(FLUTAS_ERR_INVALID_ARG, "the workspace is too small: %zu bytes given, %zu needed", bytes, pl->bytes);
    }
    CUDA_TRY(cudaDeviceSynchronize());
    plan_detach_workspace(pl);
    if (!dev_ptr) {
        void *base = nullptr;
        CUDA_TRY(cudaMalloc(&base, pl->bytes));
        return plan_attach_workspace(pl, base, true);
    }
    return plan_attach_workspace(pl, dev_ptr, false);
}

extern "C" void flutas_plan_destroy(flutas_plan *pl) {
    if (!pl) return;
    cudaDeviceSynchronize();
    cudaFree(pl->tw_x); cudaFree(pl->tw_y); cudaFree(pl->tw_z);
    cudaFree(pl->lam_x); cudaFree(pl->lam_y); cudaFree(pl->lam_z); cudaFree(pl->lam_x2);
    cudaFree(pl->wq_x); cudaFree(pl->wq_y);
    cudaFree(pl->sing_coef);
    cudaFree(pl->sc_dev);
    delete pl->tpm;
    if (pl->cp_owned) cudaFree(pl->cp);
    plan_detach_workspace(pl);
    for (int i = 0; i < 6; ++i) cudaFree(pl->stage[i]);
    for (int i = 0; i < 3; ++i) if (pl->lane[i]) cudaStreamDestroy(pl->lane[i]);
    if (pl->ev_fork) cudaEventDestroy(pl->ev_fork);
    if (pl->ev_dep) {
        for (int i = 0; i < pl->n_dep; ++i) cudaEventDestroy(pl->ev_dep[i]);
        delete[] pl->ev_dep;
    }
    if (pl->events) {
        for (int i = 0; i < kMaxPendingSteps * (pl->n_launch + 1); ++i) cudaEventDestroy(pl->events[i]);
        delete[] pl->events;
    }
    cudaGetLastError();
    delete pl;
}

static bool rhs_takes_ranges(const flutas_plan *pl);
static bool x_is_persistent(const flutas_plan *pl) { return pl->n2 >= 64 && pl->n2 <= 512; }   // nx = 128 .. 1024

extern "C" size_t flutas_plan_workspace_bytes(const flutas_plan *pl) { return pl ? pl->bytes : 0; }
extern "C" int flutas_plan_kernel_launches(const flutas_plan *pl) { return pl ? pl->n_launch : 0; }
extern "C" const char *flutas_plan_kernel_name(const flutas_plan *pl, int idx) {
    if (!pl || idx < 0 || idx >= pl->n_launch) return nullptr;
    return kKernelNames[pl->launch_ids[idx]];
}

extern "C" double flutas_plan_kernel_bytes(const flutas_plan *pl, int idx) {
    if (!pl || idx < 0 || idx >= pl->n_launch) return 0.0;
    const double f = 8.0 * (double)pl->npts;                    // one real field
    const double s = 16.0 * (double)pl->nxh * pl->ny * pl->nz;  // the half-spectrum (valid columns)
    switch (pl->launch_ids[idx]) {
        case K_RHS: return 6 * f + 4 * f;          // read u*,v*,w*,phi,p,p_old; write rhs,u',v',w'
        case K_FFTX: return f + s;                 // read rhs, write spectrum
        case K_FFTY: case K_IFFTY: return 2 * s;   // read + write spectrum
        case K_Z:
            if (pl->bc_z != FLUTAS_BC_Z_WALL) return 2 * s;
            if (pl->thomas_variant == 1)   // one pass + the coefficient table (one double per column and half the planes)
                return 2 * s + 8.0 * ThomasGeom::tab_doubles(pl->nz, thomas_cw(pl)) * ((pl->nxh + ThomasGeom::C - 1) / ThomasGeom::C) * pl->ny;
            return 4 * s + 2 * (s / 2);    // two sweeps + c'
        case K_ZS: return 2.0 * 16.0 * pl->nz;
        case K_IFFTX: return s + f;                // read spectrum, write p
        case K_CORR: return 4 * f + 3 * f;         // read p,u',v',w'; write u,v,w
    }
    return 0.0;
}

extern "C" const char *flutas_plan_kernel_symbol(const flutas_plan *pl, int idx) {
    if (!pl || idx < 0 || idx >= pl->n_launch) return nullptr;
    const bool wall = pl->bc_z == FLUTAS_BC_Z_WALL;
    switch (pl->launch_ids[idx]) {
        case K_RHS: return rhs_takes_ranges(pl) ? "splitting_rhs_kernel3" : "splitting_rhs_kernel2";
        case K_FFTX: return pl->xsplit ? (x_is_persistent(pl) ? "fft_x_r2c_tma_kernel" : "fft_x_r2r_fwd_kernel") : pl->nx == 8 ? "fft_x8_r2c_kernel" : (x_is_persistent(pl) ? "fft_x_r2c_tma_kernel" : "fft_x_r2c_kernel");
        case K_IFFTX: return pl->xsplit ? (x_is_persistent(pl) ? "fft_x_c2r_tma_kernel" : "fft_x_r2r_inv_kernel") : pl->nx == 8 ? "fft_x8_c2r_kernel" : (x_is_persistent(pl) ? "fft_x_c2r_tma_kernel" : "fft_x_c2r_kernel");
        case K_FFTY: case K_IFFTY:
            return pl->y16 ? "fft_y1024_kernel" : (pl->ny * pl->y_cols / 8 <= 512 ? "fft_tma1_kernel" : "fft_tma_kernel");
        case K_Z:
            if (wall) return pl->thomas_variant == 1 ? "thomas_tma_kernel" : "thomas_kernel";
            return pl->nz * pl->z_cols / 8 <= 512 ? "fft_tma1_kernel" : "fft_tma_kernel";
        case K_ZS: return "thomas_singular_kernel";
        case K_CORR: return "correction_kernel";
    }
    return nullptr;
}

extern "C" int flutas_plan_set_option(flutas_plan *pl, const char *name, int value) {
    if (!pl || !name) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan or option name");
    if (!strcmp(name, "thomas") && pl->bc_z == FLUTAS_BC_Z_WALL && !(value == 0 && pl->xsplit) &&
        (value == 0 || (value == 1 && ThomasGeom::smem_bytes(pl->nz, thomas_cw(pl)) <= 227 * 1024))) {
        if (value == 0 && !pl->cp) {   // the two-sweep kernel keeps c' in half a spectrum of its own
            CUDA_TRY(cudaMalloc((void **)&pl->cp, sizeof(double) * (size_t)pl->nspec));
            pl->cp_owned = true;
        }
        pl->thomas_variant = value;
        return pl->ws_base ? plan_make_maps(pl) : FLUTAS_OK;
    }
    if (!strcmp(name, "y16") && (value == 0 || (value == 1 && pl->ny == Y16Geom::N && pl->y_r2r == 0))) {
        CUDA_TRY(cudaDeviceSynchronize());
        pl->y16 = value;                        // the storage order along y changes with the kernel
        if (int rc = upload_lam_y(pl)) return rc;
        if (pl->ttab) if (int rc = build_thomas_table(pl)) return rc;
        return pl->ws_base ? plan_make_maps(pl) : FLUTAS_OK;
    }
    if (!strcmp(name, "thomas_warps") && (value == 1 || value == 2)) { pl->thomas_warps = value; return FLUTAS_OK; }
    if (!strcmp(name, "mom_ty16") && (value == 0 || value == 1)) { pl->mom_ty16 = value; return FLUTAS_OK; }
    if (!strcmp(name, "chunk") && value >= 0) { pl->chunk = value; return FLUTAS_OK; }
    if (!strcmp(name, "overlap") && (value == 0 || value == 1)) { pl->overlap = value; return FLUTAS_OK; }
    return fail(FLUTAS_ERR_INVALID_ARG, "unknown option or value: %s = %d", name, value);
}

// ---------------------------------------------------------------------------- launch helpers
template <typename K> static cudaError_t set_smem(K kernel, size_t bytes) {
    if (bytes <= 48 * 1024) return cudaSuccess;
    return cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

constexpr int clamp_nt(int n) { return n < 32 ? 32 : (n > 256 ? 256 : n); }

// ---- persistent TMA-fed strided passes
constexpr int tma_nt(int n, int c) { return n * c / 8 < 32 ? 32 : (n * c / 8 > 512 ? 512 : n * c / 8); }
constexpr int tma_nbuf(int n, int c) { return 2 * n * c * 16 + 4096 <= 227 * 1024 ? 2 : 1; }

template <int N, int C, int MODE>
static cudaError_t launch_tma_nc(const CUtensorMap &map, const TmaFftArgs &a, const Tma1Args &a1, int num_sms,
                                 cudaStream_t st) {
    const long long ntiles = (long long)a.n_tiles_x * a.n_outer;
    if constexpr (N * C / 8 <= 512) {
        {
            // one butterfly per thread: register-cached twiddles, direct stores, TMA prefetch only
            constexpr int NT = N * C / 8 < 32 ? 32 : N * C / 8;
            constexpr int P = Fact<N>::P, NCACHE = P - 1 < 2 ? P - 1 : 2;
            const size_t smem = (size_t)2 * N * C * 16 + 128;
            auto kern = fft_tma1_kernel<N, C, MODE, NT, NCACHE>;
            cudaError_t e = set_smem(kern, smem);
            if (e != cudaSuccess) return e;
            int per_sm = 0;
            e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem);
            if (e != cudaSuccess) return e;
            if (per_sm < 1) return cudaErrorLaunchOutOfResources;
            long long grid = (long long)num_sms * per_sm;
            if (grid > ntiles) grid = ntiles;
            kern<<<(unsigned)grid, NT, smem, st>>>(map, a1);
            return cudaGetLastError();
        }
    }
    // lines of 2048 (1024 butterflies per tile): the generic kernel, several butterflies per thread (complex transforms only)
    if constexpr (MODE == MODE_R2R_FWD || MODE == MODE_R2R_INV || MODE == MODE_FWD_SCAT || MODE == MODE_SOLVE_SCAT)
        return cudaErrorInvalidValue;
    else {
    constexpr int NT = tma_nt(N, C), NBUF = tma_nbuf(N, C);
    const size_t smem = (size_t)NBUF * N * C * 16 + 128;
    auto kern = fft_tma_kernel<N, C, MODE, NT, NBUF>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, NT, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    long long grid = (long long)num_sms * per_sm;
    if (grid > ntiles) grid = ntiles;
    kern<<<(unsigned)grid, NT, smem, st>>>(map, a);
    return cudaGetLastError();
    }
}
template <int N, int MODE>
static cudaError_t launch_tma_n(int cols, const CUtensorMap &map, TmaFftArgs a, Tma1Args a1, cudaStream_t st,
                                int num_sms) {
    a.n_tiles_x = a1.n_tiles_x = (a.nxh + cols - 1) / cols;
    if (cols == 4) return launch_tma_nc<N, 4, MODE>(map, a, a1, num_sms, st);
    if constexpr (N >= 2048) return cudaErrorInvalidValue;
    else return launch_tma_nc<N, 8, MODE>(map, a, a1, num_sms, st);
}
template <int MODE>
static cudaError_t launch_tma(int n, int cols, const CUtensorMap &map, TmaFftArgs a, long long row_stride,
                              long long outer_stride, double2 *data, cudaStream_t st, int num_sms,
                              int outer0, int n_outer) {
    a.outer0 = outer0; a.n_outer = n_outer;
    Tma1Args a1{};
    a1.outer0 = outer0;
    a1.data = data; a1.row_stride = row_stride; a1.outer_stride = outer_stride;
    a1.n_outer = a.n_outer; a1.line_dim = a.line_dim; a1.nxh = a.nxh; a1.tw = a.tw;
    a1.lam_x = a.lam_x; a1.lam_outer = a.lam_outer; a1.lam_pos = a.lam_pos;
    a1.wq = a.wq; a1.reorder = a.reorder; a1.neg = a.neg; a1.sc = a.sc;
    switch (n) {
        case 8: return launch_tma_n<8, MODE>(cols, map, a, a1, st, num_sms);
        case 16: return launch_tma_n<16, MODE>(cols, map, a, a1, st, num_sms);
        case 32: return launch_tma_n<32, MODE>(cols, map, a, a1, st, num_sms);
        case 64: return launch_tma_n<64, MODE>(cols, map, a, a1, st, num_sms);
        case 128: return launch_tma_n<128, MODE>(cols, map, a, a1, st, num_sms);
        case 256: return launch_tma_n<256, MODE>(cols, map, a, a1, st, num_sms);
        case 512: return launch_tma_n<512, MODE>(cols, map, a, a1, st, num_sms);
        case 1024: return launch_tma_n<1024, MODE>(cols, map, a, a1, st, num_sms);
        case 2048: return launch_tma_n<2048, MODE>(4, map, a, a1, st, num_sms);
    }
    return cudaErrorInvalidValue;
}

template <int N2> static cudaError_t launch_r2c_n(const flutas_plan *pl, const double *rhs, cudaStream_t st, long long tile0, long long ntiles) {
    constexpr int NT = clamp_nt(N2);
    const size_t smem = sizeof(double2) * (size_t)(N2 + 1) * 8;
    auto kern = fft_x_r2c_kernel<N2, NT>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)ntiles, NT, smem, st>>>(rhs + tile0 * 8 * 2 * N2, pl->spec, pl->tw_x, SpecRows{pl->ny, pl->plane, tile0 * 8});
    return cudaGetLastError();
}
template <int N2> static cudaError_t launch_c2r_n(const flutas_plan *pl, double *out, double scale, cudaStream_t st, long long tile0, long long ntiles) {
    constexpr int NT = clamp_nt(N2);
    const size_t smem = sizeof(double2) * (size_t)(N2 + 1) * 8;
    auto kern = fft_x_c2r_kernel<N2, NT>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)ntiles, NT, smem, st>>>(pl->spec, out + tile0 * 8 * 2 * N2, pl->tw_x, scale, SpecRows{pl->ny, pl->plane, tile0 * 8});
    return cudaGetLastError();
}
// cosine / sine expansion along x (non-periodic x; staged kernels, nx = 16 .. 1024)
template <int N2> static cudaError_t launch_r2r_fwd_n(const flutas_plan *pl, const double *rhs, cudaStream_t st, long long tile0, long long ntiles) {
    constexpr int NT = clamp_nt(N2);
    const size_t smem = sizeof(double2) * (size_t)N2 * 16;
    auto kern = fft_x_r2r_fwd_kernel<N2, NT>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)ntiles, NT, smem, st>>>(rhs + tile0 * 8 * 2 * N2, pl->spec, pl->tw_x, pl->wq_x, pl->bc[0] == FLUTAS_BC_DIRICHLET ? 1 : 0,
                                             SpecRows{pl->ny, pl->plane, tile0 * 8});
    return cudaGetLastError();
}
template <int N2> static cudaError_t launch_r2r_inv_n(const flutas_plan *pl, double *out, double scale, cudaStream_t st, long long tile0, long long ntiles) {
    constexpr int NT = clamp_nt(N2);
    const size_t smem = sizeof(double2) * (size_t)N2 * 16;
    auto kern = fft_x_r2r_inv_kernel<N2, NT>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    kern<<<(unsigned)ntiles, NT, smem, st>>>(pl->spec, out + tile0 * 8 * 2 * N2, pl->tw_x, pl->wq_x, pl->bc[0] == FLUTAS_BC_DIRICHLET ? 1 : 0, scale,
                                             SpecRows{pl->ny, pl->plane, tile0 * 8});
    return cudaGetLastError();
}
// persistent bulk-copy-fed x kernels (nx = 128 .. 1024)
template <int N2, int KIND> static cudaError_t launch_r2c_tma_n(const flutas_plan *pl, const double *rhs, cudaStream_t st, long long tile0, long long ntiles) {
    const size_t smem = (size_t)2 * 8 * N2 * 16 + 128;
    auto kern = fft_x_r2c_tma_kernel<N2, KIND>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, N2, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    long long grid = (long long)pl->num_sms * per_sm;
    if (grid > ntiles) grid = ntiles;
    kern<<<(unsigned)grid, N2, smem, st>>>(rhs + tile0 * 8 * 2 * N2, pl->spec, pl->tw_x, (int)ntiles, SpecRows{pl->ny, pl->plane, tile0 * 8},
                                           pl->wq_x, pl->bc[0] == FLUTAS_BC_DIRICHLET ? 1 : 0);
    return cudaGetLastError();
}
template <int N2, int KIND> static cudaError_t launch_c2r_tma_n(const flutas_plan *pl, double *out, double scale, cudaStream_t st, long long tile0, long long ntiles) {
    const size_t smem = (size_t)8 * (N2 + 8) * 16 + (size_t)8 * N2 * 16 + 128;
    auto kern = fft_x_c2r_tma_kernel<N2, KIND>;
    cudaError_t e = set_smem(kern, smem);
    if (e != cudaSuccess) return e;
    int per_sm = 0;
    e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, N2, smem);
    if (e != cudaSuccess) return e;
    if (per_sm < 1) return cudaErrorLaunchOutOfResources;
    long long grid = (long long)pl->num_sms * per_sm;
    if (grid > ntiles) grid = ntiles;
    kern<<<(unsigned)grid, N2, smem, st>>>(pl->spec, out + tile0 * 8 * 2 * N2, pl->tw_x, scale, (int)ntiles, SpecRows{pl->ny, pl->plane, tile0 * 8},
                                           pl->wq_x, pl->bc[0] == FLUTAS_BC_DIRICHLET ? 1 : 0);
    return cudaGetLastError();
}
#define FOR_EACH_N2_TMA(X) X(64) X(128) X(256) X(512)
#define FOR_EACH_N2(X) X(8) X(16) X(32) X(64) X(128) X(256) X(512) X(1024)
// planes k0 .. k1 - 1 (a tile is 8 consecutive x-lines; ny is a multiple of 8)
static cudaError_t launch_r2c(const flutas_plan *pl, const double *rhs, cudaStream_t st, int k0, int k1) {
    const long long tile0 = (long long)k0 * pl->ny / 8, ntiles = (long long)(k1 - k0) * pl->ny / 8;
    if (pl->xsplit && x_is_persistent(pl))
        switch (pl->n2) {
#define X(n) case n: return launch_r2c_tma_n<n, X_SPLIT>(pl, rhs, st, tile0, ntiles);
            FOR_EACH_N2_TMA(X)
#undef X
        }
    if (pl->xsplit)
        switch (pl->n2) {
#define X(n) case n: return launch_r2r_fwd_n<n>(pl, rhs, st, tile0, ntiles);
            X(8) X(16) X(32)
#undef X
        }
    if (pl->nx == 8) {   // the degenerate length: one thread per line
        const long long nlines = ntiles * 8;
        fft_x8_r2c_kernel<<<(unsigned)((nlines + 127) / 128), 128, 0, st>>>(rhs + tile0 * 64, pl->spec, nlines, SpecRows{pl->ny, pl->plane, tile0 * 8});
        return cudaGetLastError();
    }
    if (x_is_persistent(pl))
        switch (pl->n2) {
#define X(n) case n: return launch_r2c_tma_n<n, X_PERIODIC>(pl, rhs, st, tile0, ntiles);
            FOR_EACH_N2_TMA(X)
#undef X
        }
    switch (pl->n2) {
#define X(n) case n: return launch_r2c_n<n>(pl, rhs, st, tile0, ntiles);
        FOR_EACH_N2(X)
#undef X
    }
    return cudaErrorInvalidValue;
}
static cudaError_t launch_c2r(const flutas_plan *pl, double *out, double scale, cudaStream_t st, int k0, int k1) {
    const long long tile0 = (long long)k0 * pl->ny / 8, ntiles = (long long)(k1 - k0) * pl->ny / 8;
    if (pl->xsplit && x_is_persistent(pl))
        switch (pl->n2) {
#define X(n) case n: return launch_c2r_tma_n<n, X_SPLIT>(pl, out, scale, st, tile0, ntiles);
            FOR_EACH_N2_TMA(X)
#undef X
        }
    if (pl->xsplit)
        switch (pl->n2) {
#define X(n) case n: return launch_r2r_inv_n<n>(pl, out, scale, st, tile0, ntiles);
            X(8) X(16) X(32)
#undef X
        }
    if (pl->nx == 8) {
        const long long nlines = ntiles * 8;
        fft_x8_c2r_kernel<<<(unsigned)((nlines + 127) / 128), 128, 0, st>>>(pl->spec, out + tile0 * 64, scale, nlines, SpecRows{pl->ny, pl->plane, tile0 * 8});
        return cudaGetLastError();
    }
    if (x_is_persistent(pl))
        switch (pl->n2) {
#define X(n) case n: return launch_c2r_tma_n<n, X_PERIODIC>(pl, out, scale, st, tile0, ntiles);
            FOR_EACH_N2_TMA(X)
#undef X
        }
    switch (pl->n2) {
#define X(n) case n: return launch_c2r_n<n>(pl, out, scale, st, tile0, ntiles);
        FOR_EACH_N2(X)
#undef X
    }
    return cudaErrorInvalidValue;
}

// -------------------------------------------------------------------------- the launch sequence
struct StepTimer {
    flutas_plan *pl;
    cudaStream_t st;
    cudaEvent_t *ev;
    int n;
    StepTimer(flutas_plan *p, cudaStream_t s) : pl(p), st(s), ev(nullptr), n(0) {
        if (p->timing && p->events) {
            if (p->pending == kMaxPendingSteps) p->pending = 0;   // drop the oldest batch
            ev = p->events + (size_t)p->pending * (p->n_launch + 1);
        }
    }
    void mark() { if (ev) cudaEventRecord(ev[n++], st); }
    void done() { if (ev) pl->pending++; }
};

static int check_launch(cudaError_t e, const char *what) {
    if (e != cudaSuccess) return fail(FLUTAS_ERR_CUDA, "launch of %s failed: %s", what, cudaGetErrorString(e));
    return FLUTAS_OK;
}

// planes k0 .. k1 - 1 of rhs, u', v', w' (the bulk-copy-fed form takes any range; the register form the whole grid)
static bool rhs_takes_ranges(const flutas_plan *pl) {
    return pl->nx % Rhs3Geom::X == 0 && pl->ny % Rhs3Geom::TY == 0;
}
// g: the grid as the kernel is to see it (a slab plan passes its own nz / wall; everyone else pl->grid); up, vp, wp: where
// the half-corrected velocity goes
static int enqueue_rhs_g(flutas_plan *pl, GridParams g, const double *u, const double *v, const double *w, const double *phi,
                         const double *p, const double *po, double dt, double dt_ratio, double *rhs, double *up, double *vp,
                         double *wp, cudaStream_t st, int k0, int k1) {
    g.c_pn = 1.0 + dt_ratio;    // p_hat = (1 + r) p^n - r p^(n-1)
    g.c_po = dt_ratio;
    const int nk = k1 - k0;
    const int kc = pl->rhs_kc < nk ? pl->rhs_kc : nk;
    if (rhs_takes_ranges(pl)) {
        // bulk-copy-fed form: tile = 128 x 8 cells, three plane slabs in shared memory
        const dim3 b3(Rhs3Geom::NTX, Rhs3Geom::TY), g3(pl->nx / Rhs3Geom::X, pl->ny / Rhs3Geom::TY, (nk + kc - 1) / kc);
        auto k3 = g.wall ? splitting_rhs_kernel3<true> : splitting_rhs_kernel3<false>;
        if (set_smem(k3, Rhs3Geom::SMEM) != cudaSuccess) return check_launch(cudaGetLastError(), "splitting_rhs attr");
        k3<<<g3, b3, Rhs3Geom::SMEM, st>>>(g, dt, kc, k0, k1, u, v, w, phi, p, po, rhs, up, vp, wp);
        return check_launch(cudaGetLastError(), "splitting_rhs");
    }
    // small grids (nx < 128 or ny < 8 rows per tile): the register-marching form.
    // block = (bx threads x 2 points) x ty rows; nx/2 and ny are powers of two, so the grid divides evenly
    if (k0 != 0 || k1 != pl->nz) return fail(FLUTAS_ERR_INVALID_ARG, "this form of the RHS kernel takes the whole grid");
    const int bx = pl->nx / 2 < 64 ? pl->nx / 2 : 64;
    int ty = 256 / bx;
    if (ty > pl->ny) ty = pl->ny;
    dim3 block(bx, ty), grid(pl->nx / 2 / bx, pl->ny / ty, (nk + kc - 1) / kc);
    if (g.wall)
        splitting_rhs_kernel2<true><<<grid, block, 0, st>>>(g, dt, kc, u, v, w, phi, p, po, rhs, up, vp, wp);
    else
        splitting_rhs_kernel2<false><<<grid, block, 0, st>>>(g, dt, kc, u, v, w, phi, p, po, rhs, up, vp, wp);
    return check_launch(cudaGetLastError(), "splitting_rhs");
}
static int enqueue_rhs(flutas_plan *pl, const double *u, const double *v, const double *w, const double *phi,
                       const double *p, const double *po, double dt, double dt_ratio, double *rhs, cudaStream_t st,
                       int k0, int k1) {
    return enqueue_rhs_g(pl, pl->grid, u, v, w, phi, p, po, dt, dt_ratio, rhs, pl->up, pl->vp, pl->wp, st, k0, k1);
}

// transform along y (MODE_FWD or MODE_INV) of planes k0 .. k1 - 1 of the half-spectrum
template <int MODE> static int enqueue_y(flutas_plan *pl, cudaStream_t st, int k0, int k1) {
    const char *what = MODE == MODE_FWD ? "fft_y_fwd" : "fft_y_inv";
    const long long row_stride = pl->pitch, outer_stride = pl->plane;
    if (pl->y16) {
        Tma1Args a1{};
        a1.data = pl->spec; a1.row_stride = row_stride; a1.outer_stride = outer_stride;
        a1.n_tiles_x = (pl->nxh + Y16Geom::C - 1) / Y16Geom::C;
        a1.n_outer = k1 - k0; a1.outer0 = k0; a1.line_dim = 1; a1.nxh = pl->nxh; a1.tw = pl->tw_y;
        auto kern = fft_y1024_kernel<MODE>;
        if (set_smem(kern, Y16Geom::SMEM) != cudaSuccess) return check_launch(cudaGetLastError(), what);
        long long grid = pl->num_sms;
        if (grid > (long long)a1.n_tiles_x * a1.n_outer) grid = (long long)a1.n_tiles_x * a1.n_outer;
        kern<<<(unsigned)grid, Y16Geom::NT, Y16Geom::SMEM, st>>>(pl->map_y, a1);
        return check_launch(cudaGetLastError(), what);
    }
    TmaFftArgs ty{};
    ty.line_dim = 1;
    ty.nxh = pl->nxh;
    ty.tw = pl->tw_y;
    if (pl->y_r2r) {   // real-linear expansion of both components of every column (kernels_r2r.cuh, kernels_tma.cuh)
        ty.wq = pl->y_r2r >= 2 ? pl->wq_y : nullptr;
        ty.reorder = pl->y_r2r >= 2 ? 1 : 0;
        ty.neg = pl->y_r2r == 3 ? 1 : 0;
        constexpr int RMODE = MODE == MODE_FWD ? MODE_R2R_FWD : MODE_R2R_INV;
        return check_launch(launch_tma<RMODE>(pl->ny, pl->y_cols, pl->map_y, ty, row_stride, outer_stride, pl->spec,
                                              st, pl->num_sms, k0, k1 - k0), what);
    }
    if (MODE == MODE_FWD && pl->sc_dev) {   // slab decomposition: the last pass stores into the peers' z-local spectra
        ty.sc = pl->sc_dev;
        return check_launch(launch_tma<MODE_FWD_SCAT>(pl->ny, pl->y_cols, pl->map_y, ty, row_stride, outer_stride, pl->spec,
                                                      st, pl->num_sms, k0, k1 - k0), what);
    }
    return check_launch(launch_tma<MODE>(pl->ny, pl->y_cols, pl->map_y, ty, row_stride, outer_stride, pl->spec,
                                         st, pl->num_sms, k0, k1 - k0), what);
}

// the z stage on the whole half-spectrum (every line along z crosses all planes); timer marks between kernels
static int enqueue_z(flutas_plan *pl, cudaStream_t st, StepTimer *tm) {
    const bool wall = pl->bc_z == FLUTAS_BC_Z_WALL;
    if (!wall) {
        const long long row_stride = pl->plane, outer_stride = pl->pitch;
        TmaFftArgs tz{};
        tz.line_dim = 2;
        tz.nxh = pl->nxh;
        tz.tw = pl->tw_z;
        tz.lam_x = pl->lam_x;
        tz.lam_outer = pl->lam_y;
        tz.lam_pos = pl->lam_z;
        if (pl->sc_dev) {   // slab decomposition: the last inverse pass stores into the peers' slab spectra
            tz.sc = pl->sc_dev;
            if (int rc = check_launch(launch_tma<MODE_SOLVE_SCAT>(pl->nz, pl->z_cols, pl->map_z, tz, row_stride, outer_stride,
                                                                  pl->spec, st, pl->num_sms, 0, pl->ny), "z_solve")) return rc;
        } else if (int rc = check_launch(launch_tma<MODE_SOLVE>(pl->nz, pl->z_cols, pl->map_z, tz, row_stride, outer_stride, pl->spec,
                                                                st, pl->num_sms, 0, pl->ny), "z_solve")) return rc;
        if (tm) tm->mark();
    } else {
        const long long ncol = (long long)pl->pitch * pl->ny;
        const double inv_dz2 = pl->grid.inv_dz * pl->grid.inv_dz;
        if (pl->thomas_variant == 1) {
            ThomasArgs ta{};
            ta.tab = pl->ttab;
            ta.n_tiles_x = (pl->nxh + ThomasGeom::C - 1) / ThomasGeom::C;
            ta.ny = pl->ny;
            ta.nz = pl->nz;
            ta.dz2 = 1.0 / inv_dz2;
            ta.has_null = pl->has_null;
            const size_t smem_t = ThomasGeom::smem_bytes(pl->nz, thomas_cw(pl));
            static const ThomasPeerMaps no_peers{};
            if (pl->sc_dev) {   // slab decomposition: the solved tile goes to the ranks that own its planes
                ta.n_peers = pl->sc_npeers; ta.nzl = pl->sc_nzl; ta.srows = pl->sc_srows;
                ta.row0 = pl->row0; ta.nxh = pl->nxh; ta.sc = pl->sc_dev;
            }
            auto kern = pl->sc_dev ? (pl->thomas_warps == 2 ? thomas_tma_kernel<2, 8, true> : thomas_tma_kernel<1, 8, true>)
                      : pl->xsplit ? (pl->thomas_warps == 2 ? thomas_tma_kernel<2, 16> : thomas_tma_kernel<1, 16>)
                                   : (pl->thomas_warps == 2 ? thomas_tma_kernel<2, 8> : thomas_tma_kernel<1, 8>);
            if (set_smem(kern, smem_t) != cudaSuccess) return check_launch(cudaGetLastError(), "z_solve attr");
            long long grid = pl->num_sms;
            if (grid > (long long)ta.n_tiles_x * ta.ny) grid = (long long)ta.n_tiles_x * ta.ny;
            kern<<<(unsigned)grid, 32 * (pl->thomas_warps + 1), smem_t, st>>>(pl->map_z, ta, pl->sc_dev ? *pl->tpm : no_peers);
        } else {
            thomas_kernel<<<(unsigned)((ncol + 127) / 128), 128, 0, st>>>(pl->spec, pl->cp, pl->pitch, pl->ny, pl->nz, pl->nxh,
                                                                        pl->lam_x, pl->lam_y, inv_dz2, pl->plane, pl->end_coef_z, pl->has_null);
        }
        if (int rc = check_launch(cudaGetLastError(), "z_solve (thomas)")) return rc;
        if (tm) tm->mark();
        if (!pl->has_null) return FLUTAS_OK;   // a Dirichlet direction: no singular mode
        const size_t smem = sizeof(double) * (4 * (size_t)pl->nz + 2);
        // nz <= 4096 (checked at plan creation): at most 128 KB
        if (set_smem(thomas_singular_kernel, smem) != cudaSuccess) return check_launch(cudaGetLastError(), "z_singular attr");
        thomas_singular_kernel<<<1, 256, smem, st>>>(pl->spec, pl->plane, pl->nz, pl->sing_coef, pl->xsplit, pl->sc_dev);
        if (int rc = check_launch(cudaGetLastError(), "z_singular")) return rc;
        if (tm) tm->mark();
    }
    return FLUTAS_OK;
}

// planes k0 .. k1 - 1 of u, v, w (reads p^(n+1) of planes k0 .. k1, wrapped)
static int enqueue_correction_g(flutas_plan *pl, const GridParams &g, double dt, const double *pn, double *u, double *v, double *w,
                                cudaStream_t st, int k0, int k1) {
    if (k1 <= k0) return FLUTAS_OK;
    const long long plane = (long long)pl->nx * pl->ny, q0 = k0 * plane, q1 = k1 * plane;
    const unsigned nb = (unsigned)(((q1 - q0) / 2 + 255) / 256);   // two points per thread
    correction_kernel<<<nb, 256, 0, st>>>(g, dt, q0, q1, pn, pl->up, pl->vp, pl->wp, u, v, w);
    return check_launch(cudaGetLastError(), "correction");
}
static int enqueue_correction(flutas_plan *pl, double dt, const double *pn, double *u, double *v, double *w,
                              cudaStream_t st, int k0, int k1) {
    return enqueue_correction_g(pl, pl->grid, dt, pn, u, v, w, st, k0, k1);
}

static double norm_scale(const flutas_plan *pl) {
    const double n = (double)pl->nx * (double)pl->ny * (pl->bc_z == FLUTAS_BC_Z_WALL ? 1.0 : (double)pl->nz);
    return 1.0 / n;
}

static int check_fields(const flutas_plan *pl, const void *const *ptrs, int n) {
    const size_t fb = sizeof(double) * (size_t)pl->npts;
    for (int a = 0; a < n; ++a) {
        if (!ptrs[a]) return fail(FLUTAS_ERR_INVALID_ARG, "NULL field pointer (argument %d)", a);
        if (((size_t)ptrs[a]) & 15) return fail(FLUTAS_ERR_ALIAS, "field pointer %d is not 16-byte aligned", a);
    }
    for (int a = 0; a < n; ++a)
        for (int b = a + 1; b < n; ++b) {
            const char *x = (const char *)ptrs[a], *y = (const char *)ptrs[b];
            if (x < y + fb && y < x + fb) return fail(FLUTAS_ERR_ALIAS, "field arguments %d and %d overlap", a, b);
        }
    return FLUTAS_OK;
}

// internal streams (non-blocking, priorities low / mid / high) and dependency events of the chunked launch order
static int ensure_lanes(flutas_plan *pl, int nchunk) {
    if (!pl->lane[0]) {
        int lo = 0, hi = 0;
        CUDA_TRY(cudaDeviceGetStreamPriorityRange(&lo, &hi));   // lo = least urgent (numerically largest)
        const int mid = (lo + hi) / 2;
        const int prio[3] = {lo, mid, hi};
        for (int i = 0; i < 3; ++i) CUDA_TRY(cudaStreamCreateWithPriority(&pl->lane[i], cudaStreamNonBlocking, prio[i]));
        CUDA_TRY(cudaEventCreateWithFlags(&pl->ev_fork, cudaEventDisableTiming));
    }
    if (pl->n_dep < 2 * nchunk) {
        cudaEvent_t *ev = new (std::nothrow) cudaEvent_t[2 * nchunk];
        if (!ev) return fail(FLUTAS_ERR_ALLOC, "host allocation failed");
        for (int i = 0; i < pl->n_dep; ++i) ev[i] = pl->ev_dep[i];
        for (int i = pl->n_dep; i < 2 * nchunk; ++i) CUDA_TRY(cudaEventCreateWithFlags(&ev[i], cudaEventDisableTiming));
        delete[] pl->ev_dep;
        pl->ev_dep = ev;
        pl->n_dep = 2 * nchunk;
    }
    return FLUTAS_OK;
}

// Dirichlet pressure conditions are for flutas_poisson_solve only: the step needs the boundary-normal velocity on both
// boundary faces of such a direction, and a line of n cells stores n faces (include/flutas.h)
static int check_step_bc(const flutas_plan *pl) {
    for (int d = 0; d < 3; ++d)
        if (pl->bc[d] == FLUTAS_BC_DIRICHLET)
            return fail(FLUTAS_ERR_INVALID_ARG, "the projection step takes periodic or wall (Neumann) directions only; "
                                                "a Dirichlet plan serves flutas_poisson_solve");
    return FLUTAS_OK;
}

// p_out may be p (in place) or p_old (ping-pong) exactly, or a seventh field; anything else must not overlap
static int check_step_fields(const flutas_plan *pl, const double *u, const double *v, const double *w, const double *phi,
                             const double *p, const double *p_old, const double *p_out) {
    const void *ptrs[7] = {u, v, w, phi, p, p_old, p_out};
    const int n = (p_out == p || p_out == p_old) ? 6 : 7;
    return check_fields(pl, ptrs, n);
}

extern "C" int flutas_projection_step_ex(flutas_plan *pl, double *u, double *v, double *w, const double *phi,
                                         const double *p, const double *p_old, double *p_out, double dt,
                                         double dt_ratio, void *stream) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(FLUTAS_ERR_INVALID_ARG, "dt must be positive and finite");
    if (!(dt_ratio > 0.0) || !std::isfinite(dt_ratio)) return fail(FLUTAS_ERR_INVALID_ARG, "dt_ratio must be positive and finite");
    if (int rc = check_step_fields(pl, u, v, w, phi, p, p_old, p_out)) return rc;
    if (int rc = check_step_bc(pl)) return rc;
    if (!pl->ws_base) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no workspace (flutas_plan_set_workspace)");
    cudaStream_t st = (cudaStream_t)stream;
    StepTimer tm(pl, st);
    const int nz = pl->nz;
    // planes per launch group: 0 = every kernel covers the whole grid.  With a chunk of a few planes the kernels of one
    // group run back to back on the same planes, so rhs, the x-transformed spectrum and p^(n+1) are still in L2
    // when their consumer asks for them ("plane-chunked launch order").
    const int chunk = (pl->chunk > 0 && pl->chunk < nz && rhs_takes_ranges(pl)) ? pl->chunk : nz;
    const int nchunk = (nz + chunk - 1) / chunk;
    const bool lanes = chunk != nz && pl->overlap;
    cudaStream_t s_lo = st, s_mid = st, s_hi = st;
    if (lanes) {
        if (int rc = ensure_lanes(pl, nchunk)) return rc;
        s_lo = pl->lane[0]; s_mid = pl->lane[1]; s_hi = pl->lane[2];
        CUDA_TRY(cudaEventRecord(pl->ev_fork, st));
        CUDA_TRY(cudaStreamWaitEvent(s_lo, pl->ev_fork, 0));
    }
    tm.mark();
    for (int c = 0, k0 = 0; k0 < nz; k0 += chunk, ++c) {
        const int k1 = k0 + chunk < nz ? k0 + chunk : nz;
        if (int rc = enqueue_rhs(pl, u, v, w, phi, p, p_old, dt, dt_ratio, pl->rhs, s_lo, k0, k1)) return rc;
        if (chunk == nz) tm.mark();
        if (lanes) { CUDA_TRY(cudaEventRecord(pl->ev_dep[2 * c], s_lo)); CUDA_TRY(cudaStreamWaitEvent(s_mid, pl->ev_dep[2 * c], 0)); }
        if (int rc = check_launch(launch_r2c(pl, pl->rhs, s_mid, k0, k1), "fft_x_r2c")) return rc;
        if (chunk == nz) tm.mark();
        if (lanes) { CUDA_TRY(cudaEventRecord(pl->ev_dep[2 * c + 1], s_mid)); CUDA_TRY(cudaStreamWaitEvent(s_hi, pl->ev_dep[2 * c + 1], 0)); }
        if (int rc = enqueue_y<MODE_FWD>(pl, s_hi, k0, k1)) return rc;
    }
    if (lanes) {   // the last transform along y depends on every launch of the three lanes
        CUDA_TRY(cudaEventRecord(pl->ev_fork, s_hi));
        CUDA_TRY(cudaStreamWaitEvent(st, pl->ev_fork, 0));
    }
    if (chunk != nz) { tm.mark(); tm.mark(); }   // chunked: the group's time is booked on its first kernel
    tm.mark();
    if (int rc = enqueue_z(pl, st, &tm)) return rc;
    if (lanes) {
        CUDA_TRY(cudaEventRecord(pl->ev_fork, st));
        CUDA_TRY(cudaStreamWaitEvent(s_lo, pl->ev_fork, 0));
    }
    // p, p_old and phi are dead after the RHS kernel: p^(n+1) may go straight into either of them
    int corrected = 0;   // planes 0 .. corrected - 1 of u, v, w are final
    for (int c = 0, k0 = 0; k0 < nz; k0 += chunk, ++c) {
        const int k1 = k0 + chunk < nz ? k0 + chunk : nz;
        if (int rc = enqueue_y<MODE_INV>(pl, s_lo, k0, k1)) return rc;
        if (chunk == nz) tm.mark();
        if (lanes) { CUDA_TRY(cudaEventRecord(pl->ev_dep[2 * c], s_lo)); CUDA_TRY(cudaStreamWaitEvent(s_mid, pl->ev_dep[2 * c], 0)); }
        if (int rc = check_launch(launch_c2r(pl, p_out, norm_scale(pl), s_mid, k0, k1), "fft_x_c2r")) return rc;
        if (chunk == nz) tm.mark();
        if (lanes) { CUDA_TRY(cudaEventRecord(pl->ev_dep[2 * c + 1], s_mid)); CUDA_TRY(cudaStreamWaitEvent(s_hi, pl->ev_dep[2 * c + 1], 0)); }
        // plane k needs p^(n+1) of plane k + 1: the last plane of a chunk waits for the next chunk
        const int upto = k1 == nz ? nz : k1 - 1;
        if (int rc = enqueue_correction(pl, dt, p_out, u, v, w, s_hi, corrected, upto)) return rc;
        corrected = upto;
    }
    if (lanes) {
        CUDA_TRY(cudaEventRecord(pl->ev_fork, s_hi));
        CUDA_TRY(cudaStreamWaitEvent(st, pl->ev_fork, 0));
    }
    if (chunk != nz) { tm.mark(); tm.mark(); }
    tm.mark();
    tm.done();
    return FLUTAS_OK;
}

// ---- momentum prediction fused with the splitting right-hand side (kernels_momentum.cuh), and the whole update
static int enqueue_momentum(flutas_plan *pl, const double *u, const double *v, const double *w, const double *phi,
                            const double *kappa, const double *p, const double *po, const double *const *m_old,
                            double *const *m_new, const double *prm /* mu1 mu2 sigma gx gy gz */, double dt, double dt_ratio,
                            double *us, double *vs, double *ws, double *rhs, cudaStream_t st) {
    GridParams g = pl->grid;
    g.c_pn = 1.0 + dt_ratio;
    g.c_po = dt_ratio;
    MomentumParams mp{prm[0], prm[1], prm[2], prm[3], prm[4], prm[5], 1.0 + 0.5 * dt_ratio, 0.5 * dt_ratio, kappa ? 1 : 0, p ? 1 : 0};
    return check_launch(launch_momentum_rhs(g, mp, dt, pl->mom_ty16 != 0, u, v, w, phi, kappa, p, po, m_old, m_new, rhs, us, vs, ws, st), "momentum_rhs");
}

static int check_momentum_args(const flutas_plan *pl, double mu1, double mu2, double sigma, double gx, double gy, double gz,
                               double dt, double dt_ratio) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (pl->bc[0] != FLUTAS_BC_PERIODIC || pl->bc[1] != FLUTAS_BC_PERIODIC || pl->bc[2] != FLUTAS_BC_PERIODIC ||
        pl->nx % kMomTileX != 0 || pl->ny % kMomTileYMin != 0)
        return fail(FLUTAS_ERR_UNSUPPORTED_SIZE, "the momentum prediction takes triply periodic plans with nx a multiple of 32");
    // dt_ratio = 0: the start-up step (f1 = 1, f2 = 0: explicit Euler; p_hat = p^n), R29
    if (!(dt > 0.0) || !std::isfinite(dt) || !(dt_ratio >= 0.0) || !std::isfinite(dt_ratio))
        return fail(FLUTAS_ERR_INVALID_ARG, "dt must be positive, dt_ratio non-negative, both finite");
    if (!(mu1 >= 0.0) || !(mu2 >= 0.0) || !std::isfinite(mu1 + mu2 + sigma + gx + gy + gz))
        return fail(FLUTAS_ERR_INVALID_ARG, "viscosities must be non-negative; sigma and g finite");
    if (!pl->ws_base) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no workspace (flutas_plan_set_workspace)");
    return FLUTAS_OK;
}

extern "C" int flutas_momentum_rhs(flutas_plan *pl, const double *u, const double *v, const double *w, const double *phi,
                                   const double *kappa, const double *p, const double *p_old, const double *m_old_u,
                                   const double *m_old_v, const double *m_old_w, double *m_new_u, double *m_new_v,
                                   double *m_new_w, double mu1, double mu2, double sigma, double gx, double gy, double gz,
                                   double dt, double dt_ratio, double *us_out, double *vs_out, double *ws_out,
                                   double *rhs_out, void *stream) {
    if (int rc = check_momentum_args(pl, mu1, mu2, sigma, gx, gy, gz, dt, dt_ratio)) return rc;
    if ((p == nullptr) != (p_old == nullptr)) return fail(FLUTAS_ERR_INVALID_ARG, "p and p_old must both be given or both be NULL");
    const void *ptrs[17] = {u, v, w, phi, m_old_u, m_old_v, m_old_w, m_new_u, m_new_v, m_new_w, us_out, vs_out, ws_out, rhs_out, kappa, p, p_old};
    int n = 14;
    if (kappa) ptrs[n++] = kappa;
    if (p) { ptrs[n++] = p; ptrs[n++] = p_old; }
    if (int rc = check_fields(pl, ptrs, n)) return rc;
    const double *mo[3] = {m_old_u, m_old_v, m_old_w};
    double *mn[3] = {m_new_u, m_new_v, m_new_w};
    const double prm[6] = {mu1, mu2, sigma, gx, gy, gz};
    return enqueue_momentum(pl, u, v, w, phi, kappa, p, p_old, mo, mn, prm, dt, dt_ratio, us_out, vs_out, ws_out, rhs_out,
                            (cudaStream_t)stream);
}

extern "C" int flutas_time_step(flutas_plan *pl, double *u, double *v, double *w, const double *phi, const double *kappa,
                                const double *p, const double *p_old, double *p_out, const double *m_old_u,
                                const double *m_old_v, const double *m_old_w, double *m_new_u, double *m_new_v,
                                double *m_new_w, double mu1, double mu2, double sigma, double gx, double gy, double gz,
                                double dt, double dt_ratio, void *stream) {
    if (int rc = check_momentum_args(pl, mu1, mu2, sigma, gx, gy, gz, dt, dt_ratio)) return rc;
    const void *ptrs[14] = {u, v, w, phi, p, p_old, m_old_u, m_old_v, m_old_w, m_new_u, m_new_v, m_new_w, kappa, p_out};
    int n = 12;
    if (kappa) ptrs[n++] = kappa;
    if (p_out != p && p_out != p_old) ptrs[n++] = p_out;
    if (!p_out) return fail(FLUTAS_ERR_INVALID_ARG, "NULL field pointer (p_out)");
    if (int rc = check_fields(pl, ptrs, n)) return rc;
    cudaStream_t st = (cudaStream_t)stream;
    StepTimer tm(pl, st);
    const double *mo[3] = {m_old_u, m_old_v, m_old_w};
    double *mn[3] = {m_new_u, m_new_v, m_new_w};
    const double prm[6] = {mu1, mu2, sigma, gx, gy, gz};
    tm.mark();
    if (int rc = enqueue_momentum(pl, u, v, w, phi, kappa, p, p_old, mo, mn, prm, dt, dt_ratio, pl->up, pl->vp, pl->wp, pl->rhs, st)) return rc;
    tm.mark();
    if (int rc = check_launch(launch_r2c(pl, pl->rhs, st, 0, pl->nz), "fft_x_r2c")) return rc;
    tm.mark();
    if (int rc = enqueue_y<MODE_FWD>(pl, st, 0, pl->nz)) return rc;
    tm.mark();
    if (int rc = enqueue_z(pl, st, &tm)) return rc;
    if (int rc = enqueue_y<MODE_INV>(pl, st, 0, pl->nz)) return rc;
    tm.mark();
    if (int rc = check_launch(launch_c2r(pl, p_out, norm_scale(pl), st, 0, pl->nz), "fft_x_c2r")) return rc;
    tm.mark();
    if (int rc = enqueue_correction(pl, dt, p_out, u, v, w, st, 0, pl->nz)) return rc;
    tm.mark();
    tm.done();
    return FLUTAS_OK;
}

// ---- MTHINC volume-of-fluid step (kernels_vof.cuh): three sweeps (flux, update) and the divergence correction
extern "C" int flutas_vof_step(flutas_plan *pl, const double *phi, const double *u, const double *v, const double *w,
                               double *phi_out, double beta, double dt, void *stream) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (pl->bc[0] != FLUTAS_BC_PERIODIC || pl->bc[1] != FLUTAS_BC_PERIODIC || pl->bc[2] != FLUTAS_BC_PERIODIC)
        return fail(FLUTAS_ERR_UNSUPPORTED_SIZE, "the volume-of-fluid step takes triply periodic plans");
    if (!(beta > 0.0) || !std::isfinite(beta) || !(dt > 0.0) || !std::isfinite(dt))
        return fail(FLUTAS_ERR_INVALID_ARG, "beta and dt must be positive and finite");
    const void *ptrs[5] = {phi, u, v, w, phi_out};
    if (int rc = check_fields(pl, ptrs, phi_out == phi ? 4 : 5)) return rc;
    if (!pl->ws_base) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no workspace (flutas_plan_set_workspace)");
    cudaStream_t st = (cudaStream_t)stream;
    const GridParams g = pl->grid;
    const unsigned nb = (unsigned)((pl->npts + 255) / 256), nbf = (unsigned)((pl->npts + VofTile::CELLS - 1) / VofTile::CELLS);
    double *flux = pl->rhs, *px = pl->up, *py = pl->vp, *pz = pl->wp;
    vof_flux_kernel<0><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, phi, u, flux);
    vof_update_kernel<0><<<nb, 256, 0, st>>>(g, dt, phi, u, flux, px);
    vof_flux_kernel<1><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, px, v, flux);
    vof_update_kernel<1><<<nb, 256, 0, st>>>(g, dt, px, v, flux, py);
    vof_flux_kernel<2><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, py, w, flux);
    vof_update_kernel<2><<<nb, 256, 0, st>>>(g, dt, py, w, flux, pz);
    vof_final_kernel<<<nb, 256, 0, st>>>(g, dt, px, py, pz, u, v, w, phi_out);
    return check_launch(cudaGetLastError(), "vof_step");
}

// The launch sequence of flutas_vof_step on caller-given intermediate fields, for vof_noalloc.cu (vof_launch.h): the VoF
// kernels read only the sizes and spacings of g.
cudaError_t flutas::launch_vof_step(const GridParams &g, double beta, double dt, const double *phi, const double *u, const double *v,
                                    const double *w, double *flux, double *px, double *py, double *pz, double *phi_out,
                                    cudaStream_t st) {
    const long long npts = (long long)g.nx * g.ny * g.nz;
    const unsigned nb = (unsigned)((npts + 255) / 256), nbf = (unsigned)((npts + VofTile::CELLS - 1) / VofTile::CELLS);
    vof_flux_kernel<0><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, phi, u, flux);
    vof_update_kernel<0><<<nb, 256, 0, st>>>(g, dt, phi, u, flux, px);
    vof_flux_kernel<1><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, px, v, flux);
    vof_update_kernel<1><<<nb, 256, 0, st>>>(g, dt, px, v, flux, py);
    vof_flux_kernel<2><<<nbf, VofTile::NT, 0, st>>>(g, beta, dt, py, w, flux);
    vof_update_kernel<2><<<nb, 256, 0, st>>>(g, dt, py, w, flux, pz);
    vof_final_kernel<<<nb, 256, 0, st>>>(g, dt, px, py, pz, u, v, w, phi_out);
    return cudaGetLastError();
}

extern "C" int flutas_projection_step(flutas_plan *pl, double *u, double *v, double *w, const double *phi, double *p,
                                      const double *p_old, double dt, void *stream) {
    return flutas_projection_step_ex(pl, u, v, w, phi, p, p_old, p, dt, 1.0, stream);
}

extern "C" int flutas_splitting_rhs_ex(flutas_plan *pl, const double *u, const double *v, const double *w,
                                       const double *phi, const double *p, const double *p_old, double dt,
                                       double dt_ratio, double *rhs_out, void *stream) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(FLUTAS_ERR_INVALID_ARG, "dt must be positive and finite");
    if (!(dt_ratio > 0.0) || !std::isfinite(dt_ratio)) return fail(FLUTAS_ERR_INVALID_ARG, "dt_ratio must be positive and finite");
    const void *ptrs[7] = {u, v, w, phi, p, p_old, rhs_out};
    if (int rc = check_fields(pl, ptrs, 7)) return rc;
    if (int rc = check_step_bc(pl)) return rc;
    if (!pl->ws_base) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no workspace (flutas_plan_set_workspace)");
    return enqueue_rhs(pl, u, v, w, phi, p, p_old, dt, dt_ratio, rhs_out, (cudaStream_t)stream, 0, pl->nz);
}

extern "C" int flutas_splitting_rhs(flutas_plan *pl, const double *u, const double *v, const double *w, const double *phi,
                                    const double *p, const double *p_old, double dt, double *rhs_out, void *stream) {
    return flutas_splitting_rhs_ex(pl, u, v, w, phi, p, p_old, dt, 1.0, rhs_out, stream);
}

extern "C" int flutas_poisson_solve(flutas_plan *pl, const double *rhs, double *p_out, void *stream) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    const void *ptrs[2] = {rhs, p_out};
    if (rhs == p_out) { if (int rc = check_fields(pl, ptrs, 1)) return rc; }
    else if (int rc = check_fields(pl, ptrs, 2)) return rc;
    if (!pl->ws_base) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no workspace (flutas_plan_set_workspace)");
    cudaStream_t st = (cudaStream_t)stream;
    if (int rc = check_launch(launch_r2c(pl, rhs, st, 0, pl->nz), "fft_x_r2c")) return rc;
    if (int rc = enqueue_y<MODE_FWD>(pl, st, 0, pl->nz)) return rc;
    if (int rc = enqueue_z(pl, st, nullptr)) return rc;
    if (int rc = enqueue_y<MODE_INV>(pl, st, 0, pl->nz)) return rc;
    return check_launch(launch_c2r(pl, p_out, norm_scale(pl), st, 0, pl->nz), "fft_x_c2r");
}

extern "C" int flutas_projection_step_host(flutas_plan *pl, double *u, double *v, double *w, const double *phi, double *p,
                                           const double *p_old, double dt, void *stream) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    const void *src[6] = {u, v, w, phi, p, p_old};
    for (int i = 0; i < 6; ++i)
        if (!src[i]) return fail(FLUTAS_ERR_INVALID_ARG, "NULL host pointer (argument %d)", i);
    const size_t fb = sizeof(double) * (size_t)pl->npts;
    for (int i = 0; i < 6; ++i)
        if (!pl->stage[i]) CUDA_TRY(cudaMalloc((void **)&pl->stage[i], fb));
    cudaStream_t st = (cudaStream_t)stream;
    for (int i = 0; i < 6; ++i) CUDA_TRY(cudaMemcpyAsync(pl->stage[i], src[i], fb, cudaMemcpyHostToDevice, st));
    if (int rc = flutas_projection_step(pl, pl->stage[0], pl->stage[1], pl->stage[2], pl->stage[3], pl->stage[4],
                                        pl->stage[5], dt, stream))
        return rc;
    double *dst[4] = {u, v, w, p};
    const int from[4] = {0, 1, 2, 4};
    for (int i = 0; i < 4; ++i) CUDA_TRY(cudaMemcpyAsync(dst[i], pl->stage[from[i]], fb, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(cudaStreamSynchronize(st));
    return FLUTAS_OK;
}

// -------------------------------------------------------------------------------------- timing
extern "C" int flutas_plan_set_timing(flutas_plan *pl, int enabled) {
    if (!pl) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (enabled && !pl->events) {
        const int n = kMaxPendingSteps * (pl->n_launch + 1);
        pl->events = new (std::nothrow) cudaEvent_t[n];
        if (!pl->events) return fail(FLUTAS_ERR_ALLOC, "host allocation failed");
        for (int i = 0; i < n; ++i) CUDA_TRY(cudaEventCreate(&pl->events[i]));
    }
    pl->timing = enabled ? 1 : 0;
    pl->pending = 0;
    return FLUTAS_OK;
}

extern "C" int flutas_plan_read_timing(flutas_plan *pl, float *ms_out, int n_out, int *steps_out) {
    if (!pl || !ms_out || n_out < pl->n_launch) return fail(FLUTAS_ERR_INVALID_ARG, "bad arguments to read_timing");
    for (int i = 0; i < n_out; ++i) ms_out[i] = 0.0f;
    const int steps = pl->pending;
    for (int s = 0; s < steps; ++s) {
        cudaEvent_t *ev = pl->events + (size_t)s * (pl->n_launch + 1);
        CUDA_TRY(cudaEventSynchronize(ev[pl->n_launch]));
        for (int i = 0; i < pl->n_launch; ++i) {
            float ms = 0.0f;
            CUDA_TRY(cudaEventElapsedTime(&ms, ev[i], ev[i + 1]));
            ms_out[i] += ms;
        }
    }
    if (steps_out) *steps_out = steps;
    pl->pending = 0;
    return FLUTAS_OK;
}

// -------------------------------------------------------------------------------------- z-slab decomposition (NEXT-3)
#include "flutas_slab.inl"
