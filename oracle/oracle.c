/*
 * oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT.  See oracle.h for the contract, the
 * passages of the paper each function follows, and who may load this library.
 *
 * Deliberately plain: every discrete operator is written out index by index, the
 * Fourier expansions are naive O(n^2) sums against a table of roots of unity, the
 * tridiagonal systems are solved by the textbook Thomas recurrences.  Nothing here is
 * blocked, fused or reordered beyond "which thread gets which independent line".
 *
 * build: gcc -O3 -fopenmp -fPIC -shared (no -ffast-math, no -march flags) -- see build.py
 */
#include "oracle.h"

#include <math.h>
#include <omp.h>
#include <stdlib.h>
#include <string.h>

/* ------------------------------------------------------------------ helpers */

typedef struct {
    int nx, ny, nz, wall;
    int bcx, bcy, bcz;   /* ORACLE_BC_PERIODIC / _NEUMANN / _DIRICHLET per direction; wall = (bcz == NEUMANN) */
    double dx, dy, dz;
    double rho1, rho2, rho0, dt;
    double r;   /* dt^(n+1) / dt^n, the time-step ratio of the pressure extrapolation; 1 = constant dt */
} grid_t;

static int grid_init(grid_t *g, int nx, int ny, int nz, double lx, double ly, double lz,
                     int bc_z, double rho1, double rho2, double dt) {
    if (nx < 1 || ny < 1 || nz < 1) return 1;
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0)) return 1;
    if (bc_z != ORACLE_BC_Z_PERIODIC && bc_z != ORACLE_BC_Z_WALL) return 1;
    if (bc_z == ORACLE_BC_Z_WALL && nz < 2) return 1;
    g->nx = nx; g->ny = ny; g->nz = nz; g->wall = (bc_z == ORACLE_BC_Z_WALL);
    g->bcx = ORACLE_BC_PERIODIC; g->bcy = ORACLE_BC_PERIODIC; g->bcz = bc_z;
    g->dx = lx / nx; g->dy = ly / ny; g->dz = lz / nz;         /* uniform spacing */
    g->rho1 = rho1; g->rho2 = rho2;
    g->rho0 = rho1 < rho2 ? rho1 : rho2;                        /* rho0 = min density, PAPER.md:161 (R3) */
    g->dt = dt;
    g->r = 1.0;
    return 0;
}

/* the same with boundary conditions along x and y as well; Dirichlet along z is allowed here (Poisson problem only) */
static int grid_init_bc(grid_t *g, int nx, int ny, int nz, double lx, double ly, double lz,
                        int bc_x, int bc_y, int bc_z, double rho1, double rho2, double dt) {
    if (bc_x < 0 || bc_x > 2 || bc_y < 0 || bc_y > 2 || bc_z < 0 || bc_z > 2) return 1;
    if (grid_init(g, nx, ny, nz, lx, ly, lz, bc_z == ORACLE_BC_DIRICHLET ? ORACLE_BC_NEUMANN : bc_z, rho1, rho2, dt)) return 1;
    if ((bc_x != ORACLE_BC_PERIODIC && nx < 2) || (bc_y != ORACLE_BC_PERIODIC && ny < 2)) return 1;
    g->bcx = bc_x; g->bcy = bc_y; g->bcz = bc_z;
    g->wall = (bc_z == ORACLE_BC_NEUMANN);
    return 0;
}

static inline size_t at(const grid_t *g, int i, int j, int k) {
    return (size_t)i + (size_t)g->nx * ((size_t)j + (size_t)g->ny * (size_t)k);
}
static inline int wrap(int i, int n) { return i < 0 ? i + n : (i >= n ? i - n : i); }

static void set_threads(int nthreads) {
    if (nthreads > 0) omp_set_num_threads(nthreads);
    else omp_set_num_threads(omp_get_num_procs());
}
int oracle_threads(int nthreads) { return nthreads > 0 ? nthreads : omp_get_num_procs(); }

/* cell density, eq. (2): rho = rho1*phi + rho2*(1-phi) (phi = 1 is phase 1, R11) */
static inline double rho_c(const grid_t *g, const double *phi, int i, int j, int k) {
    double f = phi[at(g, i, j, k)];
    return g->rho1 * f + g->rho2 * (1.0 - f);
}
/* time-extrapolated pressure: p_hat = (1 + r) p^n - r p^(n-1), r = dt^(n+1)/dt^n;
 * constant dt (r = 1, R4) gives p_hat = 2 p^n - p^(n-1) */
static inline double p_hat(const grid_t *g, const double *p, const double *p_old, int i, int j, int k) {
    size_t q = at(g, i, j, k);
    return (1.0 + g->r) * p[q] - g->r * p_old[q];
}

/* gradient of a centred field f on the east / north / top face of cell (i,j,k) */
/* On the LAST face of a non-periodic direction (the boundary face): Neumann -> the normal gradient is 0 (a wall,
 * PAPER.md:161, R8); Dirichlet -> f = 0 ON the face, i.e. ghost value -f_last (cell-centred reflection), so the
 * gradient is (-f_last - f_last)/d. */
static inline double grad_x(const grid_t *g, const double *f, int i, int j, int k) {
    if (g->bcx != ORACLE_BC_PERIODIC && i == g->nx - 1)
        return g->bcx == ORACLE_BC_NEUMANN ? 0.0 : (-f[at(g, i, j, k)] - f[at(g, i, j, k)]) / g->dx;
    return (f[at(g, wrap(i + 1, g->nx), j, k)] - f[at(g, i, j, k)]) / g->dx;
}
static inline double grad_y(const grid_t *g, const double *f, int i, int j, int k) {
    if (g->bcy != ORACLE_BC_PERIODIC && j == g->ny - 1)
        return g->bcy == ORACLE_BC_NEUMANN ? 0.0 : (-f[at(g, i, j, k)] - f[at(g, i, j, k)]) / g->dy;
    return (f[at(g, i, wrap(j + 1, g->ny), k)] - f[at(g, i, j, k)]) / g->dy;
}
static inline double grad_z(const grid_t *g, const double *f, int i, int j, int k) {
    if (g->wall && k == g->nz - 1) return 0.0;    /* top wall face: normal gradient is 0 (R8) */
    if (g->bcz == ORACLE_BC_DIRICHLET && k == g->nz - 1) return (-f[at(g, i, j, k)] - f[at(g, i, j, k)]) / g->dz;
    return (f[at(g, i, j, wrap(k + 1, g->nz))] - f[at(g, i, j, k)]) / g->dz;
}
/* gradient on the FIRST boundary face of a non-periodic direction (west / south / bottom of cell 0; not a stored
 * face): Neumann 0, Dirichlet (f_0 - (-f_0))/d */
static inline double grad_first_face(int bc, double f0, double d) {
    return bc == ORACLE_BC_NEUMANN ? 0.0 : (f0 + f0) / d;
}

/* the same three gradients for p_hat */
static inline double gph_x(const grid_t *g, const double *p, const double *po, int i, int j, int k) {
    if (g->bcx == ORACLE_BC_NEUMANN && i == g->nx - 1) return 0.0;      /* east wall face */
    return (p_hat(g, p, po, wrap(i + 1, g->nx), j, k) - p_hat(g, p, po, i, j, k)) / g->dx;
}
static inline double gph_y(const grid_t *g, const double *p, const double *po, int i, int j, int k) {
    if (g->bcy == ORACLE_BC_NEUMANN && j == g->ny - 1) return 0.0;      /* north wall face */
    return (p_hat(g, p, po, i, wrap(j + 1, g->ny), k) - p_hat(g, p, po, i, j, k)) / g->dy;
}
static inline double gph_z(const grid_t *g, const double *p, const double *po, int i, int j, int k) {
    if (g->wall && k == g->nz - 1) return 0.0;
    return (p_hat(g, p, po, i, j, wrap(k + 1, g->nz)) - p_hat(g, p, po, i, j, k)) / g->dz;
}

/* face densities: arithmetic mean of the two adjacent cells (R2) */
static inline double rho_fx(const grid_t *g, const double *phi, int i, int j, int k) {
    if (g->bcx == ORACLE_BC_NEUMANN && i == g->nx - 1) return rho_c(g, phi, i, j, k);   /* wall face: as rho_fz below */
    return 0.5 * (rho_c(g, phi, i, j, k) + rho_c(g, phi, wrap(i + 1, g->nx), j, k));
}
static inline double rho_fy(const grid_t *g, const double *phi, int i, int j, int k) {
    if (g->bcy == ORACLE_BC_NEUMANN && j == g->ny - 1) return rho_c(g, phi, i, j, k);
    return 0.5 * (rho_c(g, phi, i, j, k) + rho_c(g, phi, i, wrap(j + 1, g->ny), k));
}
static inline double rho_fz(const grid_t *g, const double *phi, int i, int j, int k) {
    /* at the top wall face the value is never used with a non-zero gradient; use the cell value */
    if (g->wall && k == g->nz - 1) return rho_c(g, phi, i, j, k);
    return 0.5 * (rho_c(g, phi, i, j, k) + rho_c(g, phi, i, j, wrap(k + 1, g->nz)));
}

/* splitting flux F = (1 - rho0/rho_f) grad p_hat on the three faces of cell (i,j,k) */
static inline double flux_x(const grid_t *g, const double *phi, const double *p, const double *po, int i, int j, int k) {
    return (1.0 - g->rho0 / rho_fx(g, phi, i, j, k)) * gph_x(g, p, po, i, j, k);
}
static inline double flux_y(const grid_t *g, const double *phi, const double *p, const double *po, int i, int j, int k) {
    return (1.0 - g->rho0 / rho_fy(g, phi, i, j, k)) * gph_y(g, p, po, i, j, k);
}
static inline double flux_z(const grid_t *g, const double *phi, const double *p, const double *po, int i, int j, int k) {
    return (1.0 - g->rho0 / rho_fz(g, phi, i, j, k)) * gph_z(g, p, po, i, j, k);
}

/* divergence of a face field at cell (i,j,k); the bottom wall face (k = -1) is 0 and not stored */
static inline double div_at(const grid_t *g, const double *a, const double *b, const double *c, int i, int j, int k) {
    /* the first wall face of a walled direction (west / south / bottom) carries 0 and is not stored */
    double am = (g->bcx == ORACLE_BC_NEUMANN && i == 0) ? 0.0 : a[at(g, wrap(i - 1, g->nx), j, k)];
    double bm = (g->bcy == ORACLE_BC_NEUMANN && j == 0) ? 0.0 : b[at(g, i, wrap(j - 1, g->ny), k)];
    double cm = (g->wall && k == 0) ? 0.0 : c[at(g, i, j, wrap(k - 1, g->nz))];
    size_t q = at(g, i, j, k);
    return (a[q] - am) / g->dx + (b[q] - bm) / g->dy + (c[q] - cm) / g->dz;
}

/* ------------------------------------------------------- discrete operators */

int oracle_divergence(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                      const double *u, const double *v, const double *w, double *div_out, int nthreads) {
    return oracle_divergence_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, u, v, w, div_out, nthreads);
}

/* walls (Neumann) along x / y as along z: the first wall face carries 0 and is not stored */
int oracle_divergence_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                         const double *u, const double *v, const double *w, double *div_out, int nthreads) {
    grid_t g;
    if (bc_x == ORACLE_BC_DIRICHLET || bc_y == ORACLE_BC_DIRICHLET || bc_z == ORACLE_BC_DIRICHLET) return 1;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, 1.0, 1.0, 1.0)) return 1;
    set_threads(nthreads);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) div_out[at(&g, i, j, k)] = div_at(&g, u, v, w, i, j, k);
    return 0;
}

/* L p = div(grad p): (Gx p[i] - Gx p[i-1])/dx + ... with the wall faces carrying 0 */
int oracle_laplacian(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                     const double *p, double *lap_out, int nthreads) {
    return oracle_laplacian_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, p, lap_out, nthreads);
}

int oracle_laplacian_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                        const double *p, double *lap_out, int nthreads) {
    grid_t g;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, 1.0, 1.0, 1.0)) return 1;
    set_threads(nthreads);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                double gxp = grad_x(&g, p, i, j, k), gyp = grad_y(&g, p, i, j, k), gzp = grad_z(&g, p, i, j, k);
                double gxm = (g.bcx != ORACLE_BC_PERIODIC && i == 0) ? grad_first_face(g.bcx, p[at(&g, i, j, k)], g.dx)
                                                                      : grad_x(&g, p, wrap(i - 1, nx), j, k);
                double gym = (g.bcy != ORACLE_BC_PERIODIC && j == 0) ? grad_first_face(g.bcy, p[at(&g, i, j, k)], g.dy)
                                                                      : grad_y(&g, p, i, wrap(j - 1, ny), k);
                double gzm = (g.bcz != ORACLE_BC_PERIODIC && k == 0) ? grad_first_face(g.bcz, p[at(&g, i, j, k)], g.dz)
                                                                      : grad_z(&g, p, i, j, wrap(k - 1, nz));
                lap_out[at(&g, i, j, k)] = (gxp - gxm) / g.dx + (gyp - gym) / g.dy + (gzp - gzm) / g.dz;
            }
    return 0;
}

/* ------------------------------------------------------------ splitting RHS */

int oracle_rhs_vdt(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                   double rho1, double rho2, double dt, double dt_ratio,
                   const double *u, const double *v, const double *w, const double *phi,
                   const double *p, const double *p_old, double *rhs_out, int nthreads) {
    return oracle_rhs_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, rho1, rho2, dt, dt_ratio,
                         u, v, w, phi, p, p_old, rhs_out, nthreads);
}

int oracle_rhs_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                  double rho1, double rho2, double dt, double dt_ratio,
                  const double *u, const double *v, const double *w, const double *phi,
                  const double *p, const double *p_old, double *rhs_out, int nthreads) {
    grid_t g;
    if (bc_x == ORACLE_BC_DIRICHLET || bc_y == ORACLE_BC_DIRICHLET || bc_z == ORACLE_BC_DIRICHLET) return 1;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, rho1, rho2, dt)) return 1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(dt > 0.0) || !(dt_ratio >= 0.0)) return 1;
    g.r = dt_ratio;
    set_threads(nthreads);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                /* rho0/dt * div(u*)   -- eq. (17) */
                double d_u = div_at(&g, u, v, w, i, j, k);
                /* div[(1 - rho0/rho) grad p_hat]  -- splitting term of eq. (16) moved to the RHS (R1) */
                double fxp = flux_x(&g, phi, p, p_old, i, j, k);
                double fxm = (g.bcx == ORACLE_BC_NEUMANN && i == 0) ? 0.0 : flux_x(&g, phi, p, p_old, wrap(i - 1, nx), j, k);
                double fyp = flux_y(&g, phi, p, p_old, i, j, k);
                double fym = (g.bcy == ORACLE_BC_NEUMANN && j == 0) ? 0.0 : flux_y(&g, phi, p, p_old, i, wrap(j - 1, ny), k);
                double fzp = flux_z(&g, phi, p, p_old, i, j, k);
                double fzm = (g.wall && k == 0) ? 0.0 : flux_z(&g, phi, p, p_old, i, j, wrap(k - 1, nz));
                double d_f = (fxp - fxm) / g.dx + (fyp - fym) / g.dy + (fzp - fzm) / g.dz;
                rhs_out[at(&g, i, j, k)] = g.rho0 / g.dt * d_u + d_f;
            }
    return 0;
}

int oracle_rhs(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
               double rho1, double rho2, double dt,
               const double *u, const double *v, const double *w, const double *phi,
               const double *p, const double *p_old, double *rhs_out, int nthreads) {
    return oracle_rhs_vdt(nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, dt, 1.0, u, v, w, phi, p, p_old, rhs_out, nthreads);
}

/* ------------------------------------------------------------- naive DFT */

/* table of roots of unity e^{sign*2*pi*i*m/n}, m = 0..n-1, evaluated in long double */
static int root_table(int n, int sign, double **tr, double **ti) {
    *tr = (double *)malloc(sizeof(double) * (size_t)n);
    *ti = (double *)malloc(sizeof(double) * (size_t)n);
    if (!*tr || !*ti) { free(*tr); free(*ti); return 1; }
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < n; ++m) {
        long double a = two_pi * (long double)m / (long double)n;
        (*tr)[m] = (double)cosl(a);
        (*ti)[m] = (double)((long double)sign * sinl(a));
    }
    return 0;
}

#define LINE_BATCH 128  /* independent lines handed to one thread at a time; not a blocking of the sum */

int oracle_dft_axis(long n_outer, int n, long n_inner, int sign,
                    const double *in_re, const double *in_im,
                    double *out_re, double *out_im, int nthreads) {
    if (n_outer < 1 || n < 1 || n_inner < 1 || (sign != 1 && sign != -1)) return 1;
    double *tr, *ti;
    if (root_table(n, sign, &tr, &ti)) return 2;
    set_threads(nthreads);
    long n_batch = (n_inner + LINE_BATCH - 1) / LINE_BATCH;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (long o = 0; o < n_outer; ++o)
        for (long b = 0; b < n_batch; ++b) {
            long q0 = b * LINE_BATCH;
            int len = (int)((n_inner - q0) < LINE_BATCH ? (n_inner - q0) : LINE_BATCH);
            double acc_re[LINE_BATCH], acc_im[LINE_BATCH];
            for (int k = 0; k < n; ++k) {            /* output index */
                for (int q = 0; q < len; ++q) { acc_re[q] = 0.0; acc_im[q] = 0.0; }
                int m = 0;                           /* m = (k*j) mod n, kept exactly in integers */
                for (int j = 0; j < n; ++j) {        /* the O(n) sum, in increasing j */
                    double wr = tr[m], wi = ti[m];
                    const double *xr = in_re + ((size_t)o * n + j) * (size_t)n_inner + q0;
                    const double *xi = in_im + ((size_t)o * n + j) * (size_t)n_inner + q0;
                    for (int q = 0; q < len; ++q) {
                        acc_re[q] += wr * xr[q] - wi * xi[q];
                        acc_im[q] += wr * xi[q] + wi * xr[q];
                    }
                    m += k; if (m >= n) m -= n;
                }
                double *yr = out_re + ((size_t)o * n + k) * (size_t)n_inner + q0;
                double *yi = out_im + ((size_t)o * n + k) * (size_t)n_inner + q0;
                for (int q = 0; q < len; ++q) { yr[q] = acc_re[q]; yi[q] = acc_im[q]; }
            }
        }
    free(tr); free(ti);
    return 0;
}

/* ------------------------------------------- naive cosine / sine expansions (non-periodic directions)
 *
 * "Fourier-based expansions [that] depend on the boundary conditions": the eigenvectors of the
 * second-difference operator on n cell centres (i + 1/2) d with homogeneous conditions at both boundary FACES are
 *   Neumann   (ghost f_{-1} = f_0, f_n = f_{n-1}):    e_m[i] = cos(pi m (2i+1) / (2n)),      m = 0..n-1
 *   Dirichlet (ghost f_{-1} = -f_0, f_n = -f_{n-1}):  e_m[i] = sin(pi (m+1) (2i+1) / (2n)),  m = 0..n-1
 * with eigenvalues -2 (1 - cos(pi m / n)) / d^2 and -2 (1 - cos(pi (m+1) / n)) / d^2 (oracle_eigenvalues).
 * They are orthogonal: sum_i e_m[i]^2 = n for the constant / alternating vector (Neumann m = 0, Dirichlet m = n-1),
 * n/2 otherwise.  sign = -1 (analysis):  c_m = sum_i f[i] e_m[i] / |e_m|^2;   sign = +1 (synthesis):  f[i] = sum_m c_m e_m[i].
 * Both are plain O(n^2) sums; the argument of cos / sin is reduced exactly in integers (q mod 4n) and looked up in a
 * table evaluated in long double.  Real data, (n_outer, n, n_inner) C order like oracle_dft_axis. */
int oracle_r2r_axis(long n_outer, int n, long n_inner, int bc, int sign,
                    const double *in, double *out, int nthreads) {
    if (n_outer < 1 || n < 1 || n_inner < 1 || (sign != 1 && sign != -1)) return 1;
    if (bc != ORACLE_BC_NEUMANN && bc != ORACLE_BC_DIRICHLET) return 1;
    const int n4 = 4 * n;
    double *tab = (double *)malloc(sizeof(double) * (size_t)n4);   /* cos (Neumann) or sin (Dirichlet) of pi q / (2n) */
    if (!tab) return 2;
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int q = 0; q < n4; ++q) {
        long double a = pi * (long double)q / (long double)(2 * n);
        tab[q] = (double)(bc == ORACLE_BC_NEUMANN ? cosl(a) : sinl(a));
    }
    const int mode_shift = bc == ORACLE_BC_NEUMANN ? 0 : 1;        /* mode m has "frequency" m (Neumann) or m + 1 (Dirichlet) */
    const int long_mode = bc == ORACLE_BC_NEUMANN ? 0 : n - 1;     /* the one mode of squared norm n */
    set_threads(nthreads);
    long n_batch = (n_inner + LINE_BATCH - 1) / LINE_BATCH;
#pragma omp parallel for collapse(2) schedule(dynamic, 1)
    for (long o = 0; o < n_outer; ++o)
        for (long b = 0; b < n_batch; ++b) {
            long q0 = b * LINE_BATCH;
            int len = (int)((n_inner - q0) < LINE_BATCH ? (n_inner - q0) : LINE_BATCH);
            double acc[LINE_BATCH];
            for (int r = 0; r < n; ++r) {            /* output index: mode m (analysis) or cell i (synthesis) */
                for (int q = 0; q < len; ++q) acc[q] = 0.0;
                for (int t = 0; t < n; ++t) {        /* the O(n) sum, in increasing index */
                    int m = sign < 0 ? r : t, i = sign < 0 ? t : r;
                    int arg = (int)(((long)(m + mode_shift) * (long)(2 * i + 1)) % n4);
                    double e = tab[arg];
                    const double *x = in + ((size_t)o * n + t) * (size_t)n_inner + q0;
                    for (int q = 0; q < len; ++q) acc[q] += e * x[q];
                }
                double norm2 = (sign < 0) ? ((r == long_mode) ? (double)n : 0.5 * (double)n) : 1.0;
                double *y = out + ((size_t)o * n + r) * (size_t)n_inner + q0;
                for (int q = 0; q < len; ++q) y[q] = acc[q] / norm2;
            }
        }
    free(tab);
    return 0;
}

/* eigenvalues of the periodic second-difference operator (R6):
 * lambda[m] = -2 (1 - cos(2 pi m / n)) / d^2 */
static double *eigenvalues(int n, double d) {
    double *lam = (double *)malloc(sizeof(double) * (size_t)n);
    if (!lam) return NULL;
    const long double two_pi = 6.283185307179586476925286766559005768L;
    for (int m = 0; m < n; ++m)
        lam[m] = (double)(-2.0L * (1.0L - cosl(two_pi * (long double)m / (long double)n))) / (d * d);
    return lam;
}
/* ... and of the Neumann / Dirichlet second difference: -2 (1 - cos(pi m / n)) / d^2, -2 (1 - cos(pi (m+1) / n)) / d^2 */
static double *eigenvalues_bc(int n, double d, int bc) {
    if (bc == ORACLE_BC_PERIODIC) return eigenvalues(n, d);
    double *lam = (double *)malloc(sizeof(double) * (size_t)n);
    if (!lam) return NULL;
    const long double pi = 3.141592653589793238462643383279502884L;
    for (int m = 0; m < n; ++m) {
        int f = bc == ORACLE_BC_NEUMANN ? m : m + 1;
        lam[m] = (double)(-2.0L * (1.0L - cosl(pi * (long double)f / (long double)n))) / (d * d);
    }
    return lam;
}
int oracle_eigenvalues(int n, double d, int bc, double *lam_out) {
    if (n < 1 || !(d > 0.0) || bc < 0 || bc > 2) return 1;
    double *lam = eigenvalues_bc(n, d, bc);
    if (!lam) return 2;
    memcpy(lam_out, lam, sizeof(double) * (size_t)n);
    free(lam);
    return 0;
}

/* ------------------------------------------------------ tridiagonal in z */

/* textbook Thomas for one (kx,ky): a x_{k-1} + b_k x_k + c x_{k+1} = d_k, a = c = 1/dz^2,
 * b_k = -2/dz^2 + lam_xy inside, -1/dz^2 + lam_xy in the first/last row (Neumann, R7).
 * d is complex (dr, di), the coefficients are real.  stride = distance between k and k+1.
 * singular != 0 (the (0,0) column, lam_xy = 0): eliminate rows 0..nz-2, pin x_{nz-1} = 0,
 * back-substitute, then remove the mean over k (R5). cp, dpr, dpi: scratch of length nz.
 * end_coef: the diagonal of the first / last row is -end_coef/dz^2 + lam_xy: 1 for Neumann (ghost = interior, R7),
 * 3 for Dirichlet (ghost = -interior: p = 0 on the boundary face). */
static void thomas_column(int nz, double dz, double lam_xy, int singular, double end_coef,
                          double *dr, double *di, size_t stride,
                          double *cp, double *dpr, double *dpi) {
    const double a = 1.0 / (dz * dz), c = a;
    const double b_end = -end_coef / (dz * dz) + lam_xy, b_in = -2.0 / (dz * dz) + lam_xy;
    cp[0] = c / b_end;
    dpr[0] = dr[0] / b_end;
    dpi[0] = di[0] / b_end;
    int last = singular ? nz - 2 : nz - 1;           /* last row that is eliminated */
    for (int k = 1; k <= last; ++k) {
        double b = (k == nz - 1) ? b_end : b_in;
        double m = b - a * cp[k - 1];
        cp[k] = c / m;
        dpr[k] = (dr[k * stride] - a * dpr[k - 1]) / m;
        dpi[k] = (di[k * stride] - a * dpi[k - 1]) / m;
    }
    if (singular) { dr[(nz - 1) * stride] = 0.0; di[(nz - 1) * stride] = 0.0; }
    else { dr[(nz - 1) * stride] = dpr[nz - 1]; di[(nz - 1) * stride] = dpi[nz - 1]; }
    for (int k = nz - 2; k >= 0; --k) {
        dr[k * stride] = dpr[k] - cp[k] * dr[(k + 1) * stride];
        di[k * stride] = dpi[k] - cp[k] * di[(k + 1) * stride];
    }
    if (singular) {
        double mr = 0.0, mi = 0.0;
        for (int k = 0; k < nz; ++k) { mr += dr[k * stride]; mi += di[k * stride]; }
        mr /= nz; mi /= nz;
        for (int k = 0; k < nz; ++k) { dr[k * stride] -= mr; di[k * stride] -= mi; }
    }
}

/* --------------------------------------------------------- Poisson solve */

int oracle_poisson(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                   const double *rhs, double *p_out, double *imag_residue_out, int nthreads) {
    return oracle_poisson_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, rhs, p_out,
                             imag_residue_out, nthreads);
}

/* one expansion step along an axis of the (re, im) pair a -> b: complex DFT when periodic, the real cosine / sine
 * expansion applied to the real and imaginary parts when not */
static int expand_axis(long n_outer, int n, long n_inner, int bc, int sign,
                       const double *ar, const double *ai, double *br, double *bi, int nthreads) {
    if (bc == ORACLE_BC_PERIODIC) return oracle_dft_axis(n_outer, n, n_inner, sign, ar, ai, br, bi, nthreads);
    if (oracle_r2r_axis(n_outer, n, n_inner, bc, sign, ar, br, nthreads)) return 2;
    return oracle_r2r_axis(n_outer, n, n_inner, bc, sign, ai, bi, nthreads);
}

int oracle_poisson_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                      const double *rhs, double *p_out, double *imag_residue_out, int nthreads) {
    grid_t g;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, 1.0, 1.0, 1.0)) return 1;
    set_threads(nthreads);
    const size_t n = (size_t)nx * ny * nz;
    /* the operator has a null space (constants) unless some direction is Dirichlet */
    const int has_null = bc_x != ORACLE_BC_DIRICHLET && bc_y != ORACLE_BC_DIRICHLET && bc_z != ORACLE_BC_DIRICHLET;
    double *ar = (double *)malloc(sizeof(double) * n), *ai = (double *)calloc(n, sizeof(double));
    double *br = (double *)malloc(sizeof(double) * n), *bi = (double *)malloc(sizeof(double) * n);
    double *lamx = eigenvalues_bc(nx, g.dx, bc_x), *lamy = eigenvalues_bc(ny, g.dy, bc_y), *lamz = eigenvalues(nz, g.dz);
    int rc = 0;
    if (!ar || !ai || !br || !bi || !lamx || !lamy || !lamz) { rc = 2; goto done; }
    memcpy(ar, rhs, sizeof(double) * n);

    /* step 1: forward expansion along x;  a -> b */
    if (expand_axis((long)ny * nz, nx, 1, bc_x, -1, ar, ai, br, bi, nthreads)) { rc = 2; goto done; }
    /* step 3: forward expansion along y;  b -> a   (steps 2,4,6,8 are transposes: no-ops here) */
    if (expand_axis(nz, ny, nx, bc_y, -1, br, bi, ar, ai, nthreads)) { rc = 2; goto done; }

    if (bc_z == ORACLE_BC_PERIODIC) {
        /* periodic z: expand along z as well, divide by the eigenvalue sum, the null mode -> 0 */
        if (oracle_dft_axis(1, nz, (long)nx * ny, -1, ar, ai, br, bi, nthreads)) { rc = 2; goto done; }
#pragma omp parallel for collapse(2) schedule(static)
        for (int kz = 0; kz < nz; ++kz)
            for (int ky = 0; ky < ny; ++ky)
                for (int kx = 0; kx < nx; ++kx) {
                    size_t q = at(&g, kx, ky, kz);
                    if (has_null && kx == 0 && ky == 0 && kz == 0) { br[q] = 0.0; bi[q] = 0.0; }
                    else {
                        double lam = lamx[kx] + lamy[ky] + lamz[kz];
                        br[q] = br[q] / lam;
                        bi[q] = bi[q] / lam;
                    }
                }
        if (oracle_dft_axis(1, nz, (long)nx * ny, +1, br, bi, ar, ai, nthreads)) { rc = 2; goto done; }
    } else {
        /* step 5: Gauss elimination along z for every (kx,ky) */
        int fail = 0;
        const double end_coef = bc_z == ORACLE_BC_NEUMANN ? 1.0 : 3.0;
#pragma omp parallel
        {
            double *cp = (double *)malloc(sizeof(double) * (size_t)nz);
            double *dpr = (double *)malloc(sizeof(double) * (size_t)nz);
            double *dpi = (double *)malloc(sizeof(double) * (size_t)nz);
            if (!cp || !dpr || !dpi) {
#pragma omp atomic write
                fail = 1;
            } else {
#pragma omp for collapse(2) schedule(static)
                for (int ky = 0; ky < ny; ++ky)
                    for (int kx = 0; kx < nx; ++kx) {
                        size_t q = at(&g, kx, ky, 0);
                        thomas_column(nz, g.dz, lamx[kx] + lamy[ky], (has_null && kx == 0 && ky == 0), end_coef,
                                      ar + q, ai + q, (size_t)nx * ny, cp, dpr, dpi);
                    }
            }
            free(cp); free(dpr); free(dpi);
        }
        if (fail) { rc = 2; goto done; }
    }

    /* step 7: backward expansion along y;  a -> b */
    if (expand_axis(nz, ny, nx, bc_y, +1, ar, ai, br, bi, nthreads)) { rc = 2; goto done; }
    /* step 9: backward expansion along x;  b -> a */
    if (expand_axis((long)ny * nz, nx, 1, bc_x, +1, br, bi, ar, ai, nthreads)) { rc = 2; goto done; }

    {
        /* normalisation of the unnormalised forward/backward DFT pairs (R9; the cosine / sine expansions carry
         * their own 1/|e_m|^2); real part */
        double norm = 1.0;
        if (bc_x == ORACLE_BC_PERIODIC) norm *= (double)nx;
        if (bc_y == ORACLE_BC_PERIODIC) norm *= (double)ny;
        if (bc_z == ORACLE_BC_PERIODIC) norm *= (double)nz;
        double max_re = 0.0, max_im = 0.0;
#pragma omp parallel for reduction(max : max_re, max_im) schedule(static)
        for (size_t q = 0; q < n; ++q) {
            double re = ar[q] / norm, im = ai[q] / norm;
            p_out[q] = re;
            if (fabs(re) > max_re) max_re = fabs(re);
            if (fabs(im) > max_im) max_im = fabs(im);
        }
        if (imag_residue_out) *imag_residue_out = (max_re > 0.0) ? max_im / max_re : max_im;
    }
done:
    free(ar); free(ai); free(br); free(bi); free(lamx); free(lamy); free(lamz);
    return rc;
}

/* ------------------------------------------------------------- full step */

/* u = u* - dt [ (1/rho0) grad p_new + (1/rho_f - 1/rho0) grad p_hat ]  on every stored face;
 * at the top wall face both gradients are 0, so w keeps its entry value (R8). */
static void correct_velocity(const grid_t *g, double *u, double *v, double *w, const double *phi,
                             const double *p_new, const double *p, const double *p_old) {
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < g->nz; ++k)
        for (int j = 0; j < g->ny; ++j)
            for (int i = 0; i < g->nx; ++i) {
                size_t q = at(g, i, j, k);
                double rx = rho_fx(g, phi, i, j, k), ry = rho_fy(g, phi, i, j, k), rz = rho_fz(g, phi, i, j, k);
                u[q] = u[q] - g->dt * (grad_x(g, p_new, i, j, k) / g->rho0 +
                                       (1.0 / rx - 1.0 / g->rho0) * gph_x(g, p, p_old, i, j, k));
                v[q] = v[q] - g->dt * (grad_y(g, p_new, i, j, k) / g->rho0 +
                                       (1.0 / ry - 1.0 / g->rho0) * gph_y(g, p, p_old, i, j, k));
                w[q] = w[q] - g->dt * (grad_z(g, p_new, i, j, k) / g->rho0 +
                                       (1.0 / rz - 1.0 / g->rho0) * gph_z(g, p, p_old, i, j, k));
            }
}

int oracle_correction(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                      double rho1, double rho2, double dt,
                      double *u, double *v, double *w, const double *phi,
                      const double *p, const double *p_old, const double *p_new, int nthreads) {
    return oracle_correction_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, rho1, rho2, dt,
                                u, v, w, phi, p, p_old, p_new, nthreads);
}

int oracle_correction_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                         double rho1, double rho2, double dt,
                         double *u, double *v, double *w, const double *phi,
                         const double *p, const double *p_old, const double *p_new, int nthreads) {
    grid_t g;
    if (bc_x == ORACLE_BC_DIRICHLET || bc_y == ORACLE_BC_DIRICHLET || bc_z == ORACLE_BC_DIRICHLET) return 1;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, rho1, rho2, dt)) return 1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(dt > 0.0)) return 1;
    set_threads(nthreads);
    correct_velocity(&g, u, v, w, phi, p_new, p, p_old);
    return 0;
}

int oracle_projection_step_vdt(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                               double rho1, double rho2, double dt, double dt_ratio,
                               double *u, double *v, double *w, const double *phi,
                               double *p, const double *p_old, double *rhs_out, int nthreads) {
    return oracle_projection_step_bc(nx, ny, nz, lx, ly, lz, ORACLE_BC_PERIODIC, ORACLE_BC_PERIODIC, bc_z, rho1, rho2, dt,
                                     dt_ratio, u, v, w, phi, p, p_old, rhs_out, nthreads);
}

/* the step with walls (Neumann p, u_n = 0) along x and / or y as well: the closed cavity of PAPER.md:287 is
 * (NEUMANN, NEUMANN, NEUMANN).  Wall faces: the last stored face of a walled direction is the wall (0 on entry, passed
 * through), the first wall face is not stored. */
int oracle_projection_step_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                              double rho1, double rho2, double dt, double dt_ratio,
                              double *u, double *v, double *w, const double *phi,
                              double *p, const double *p_old, double *rhs_out, int nthreads) {
    grid_t g;
    if (bc_x == ORACLE_BC_DIRICHLET || bc_y == ORACLE_BC_DIRICHLET || bc_z == ORACLE_BC_DIRICHLET) return 1;
    if (grid_init_bc(&g, nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, rho1, rho2, dt)) return 1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(dt > 0.0) || !(dt_ratio >= 0.0)) return 1;
    g.r = dt_ratio;
    const size_t n = (size_t)nx * ny * nz;
    double *rhs = (double *)malloc(sizeof(double) * n), *p_new = (double *)malloc(sizeof(double) * n);
    int rc = 0;
    if (!rhs || !p_new) { rc = 2; goto done; }
    if ((rc = oracle_rhs_bc(nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, rho1, rho2, dt, dt_ratio, u, v, w, phi, p, p_old, rhs, nthreads))) goto done;
    if (rhs_out) memcpy(rhs_out, rhs, sizeof(double) * n);
    if ((rc = oracle_poisson_bc(nx, ny, nz, lx, ly, lz, bc_x, bc_y, bc_z, rhs, p_new, NULL, nthreads))) goto done;
    set_threads(nthreads);
    correct_velocity(&g, u, v, w, phi, p_new, p, p_old);
    memcpy(p, p_new, sizeof(double) * n);                       /* p <- p^(n+1), zero mean */
done:
    free(rhs); free(p_new);
    return rc;
}

int oracle_projection_step(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                           double rho1, double rho2, double dt,
                           double *u, double *v, double *w, const double *phi,
                           double *p, const double *p_old, double *rhs_out, int nthreads) {
    return oracle_projection_step_vdt(nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, dt, 1.0, u, v, w, phi, p, p_old,
                                      rhs_out, nthreads);
}

/* the paper's incremental grouping, eqs. (16)-(19), with the sign of R1 */
int oracle_projection_step_paper(int nx, int ny, int nz, double lx, double ly, double lz,
                                 int bc_z, double rho1, double rho2, double dt,
                                 double *u, double *v, double *w, const double *phi,
                                 double *p, const double *p_old, int nthreads) {
    grid_t g;
    if (grid_init(&g, nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, dt)) return 1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(dt > 0.0)) return 1;
    const size_t n = (size_t)nx * ny * nz;
    double *us = (double *)malloc(sizeof(double) * n), *vs = (double *)malloc(sizeof(double) * n);
    double *ws = (double *)malloc(sizeof(double) * n), *rhs = (double *)malloc(sizeof(double) * n);
    double *psi = (double *)malloc(sizeof(double) * n);
    int rc = 0;
    if (!us || !vs || !ws || !rhs || !psi) { rc = 2; goto done; }
    set_threads(nthreads);
    /* eq. (16): u*_paper = u** - dt/rho0 [ grad p^n - (1 - rho0/rho) grad p_hat ]  (input u is the paper's u**) */
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t q = at(&g, i, j, k);
                us[q] = u[q] - dt / g.rho0 * (grad_x(&g, p, i, j, k) - flux_x(&g, phi, p, p_old, i, j, k));
                vs[q] = v[q] - dt / g.rho0 * (grad_y(&g, p, i, j, k) - flux_y(&g, phi, p, p_old, i, j, k));
                ws[q] = w[q] - dt / g.rho0 * (grad_z(&g, p, i, j, k) - flux_z(&g, phi, p, p_old, i, j, k));
            }
    /* eq. (17): L psi = rho0/dt div u*_paper */
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) rhs[at(&g, i, j, k)] = g.rho0 / dt * div_at(&g, us, vs, ws, i, j, k);
    if ((rc = oracle_poisson(nx, ny, nz, lx, ly, lz, bc_z, rhs, psi, NULL, nthreads))) goto done;
    set_threads(nthreads);
    /* eq. (18): u = u*_paper - dt/rho0 grad psi */
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t q = at(&g, i, j, k);
                u[q] = us[q] - dt / g.rho0 * grad_x(&g, psi, i, j, k);
                v[q] = vs[q] - dt / g.rho0 * grad_y(&g, psi, i, j, k);
                w[q] = ws[q] - dt / g.rho0 * grad_z(&g, psi, i, j, k);
            }
    /* eq. (19): p = p^n + psi, then the zero-mean gauge (R5) */
    {
        double mean = 0.0;
        for (size_t q = 0; q < n; ++q) { p[q] = p[q] + psi[q]; mean += p[q]; }
        mean /= (double)n;
        for (size_t q = 0; q < n; ++q) p[q] -= mean;
    }
done:
    free(us); free(vs); free(ws); free(rhs); free(psi);
    return rc;
}

/* ------------------------------------------------- momentum prediction (eq. 15) */

/* SURVEY.md sec. 8(f) NEXT-5.  PAPER.md:148-151, eq. (15), and PAPER.md:161:
 *     (u** - u^n) / dt = f1 M(u^n) - f2 M(u^(n-1)) + (sigma kappa delta_Gamma + rho_hat g) / rho,
 *     f1 = 1 + dt_ratio / 2,  f2 = dt_ratio / 2  (the Adams-Bashforth coefficients of eq. (13)),
 *     M(u) = - div(u u) + (1/rho) div[ mu (grad u + grad u^T) ]   (eq. (5); "central schemes")
 * on the staggered grid, triply periodic, written out face by face:
 *   convection in divergence form with arithmetic two-point means of the transported and the transporting velocity;
 *   the stress tensor with mu = mu1 phi + mu2 (1 - phi) at cell centres (eq. 2) for the normal stresses and the mean of
 *   the four surrounding cells at cell edges for the shear stresses; 1/rho on the face with the face density of the
 *   projection (R2);
 *   surface tension as the continuum surface force sigma kappa grad(phi) with kappa a given cell-centred field
 *   (it comes from the VoF module) averaged to the face, and gravity with rho_hat = rho (no thermal
 *   expansion): readings R18-R20 of DESIGN.md.
 * In: u, v, w = u^n; mold_* = M(u^(n-1)).  Out: us, vs, ws = u**; mnew_* = M(u^n).  kappa may be NULL (sigma = 0). */
static inline double mu_c(double mu1, double mu2, const double *phi, size_t q) {
    return mu1 * phi[q] + mu2 * (1.0 - phi[q]);
}

int oracle_momentum_prediction(int nx, int ny, int nz, double lx, double ly, double lz,
                               double rho1, double rho2, double mu1, double mu2, double sigma,
                               double gx, double gy, double gz, double dt, double dt_ratio,
                               const double *u, const double *v, const double *w, const double *phi, const double *kappa,
                               const double *mold_u, const double *mold_v, const double *mold_w,
                               double *us, double *vs, double *ws,
                               double *mnew_u, double *mnew_v, double *mnew_w, int nthreads) {
    grid_t g;
    if (grid_init(&g, nx, ny, nz, lx, ly, lz, ORACLE_BC_Z_PERIODIC, rho1, rho2, dt)) return 1;
    if (!(rho1 > 0.0) || !(rho2 > 0.0) || !(mu1 >= 0.0) || !(mu2 >= 0.0) || !(dt > 0.0) || !(dt_ratio >= 0.0)) return 1;
    const double f1 = 1.0 + 0.5 * dt_ratio, f2 = 0.5 * dt_ratio;
    const double dx = g.dx, dy = g.dy, dz = g.dz;
    set_threads(nthreads);
#define AT(i, j, k) at(&g, wrap((i), nx), wrap((j), ny), wrap((k), nz))
#define MU(i, j, k) mu_c(mu1, mu2, phi, AT(i, j, k))
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                const size_t q = at(&g, i, j, k);
                /* ------------------------------------------------ x component, east face (i+1/2, j, k) */
                {
                    double ue = 0.5 * (u[AT(i, j, k)] + u[AT(i + 1, j, k)]), uw = 0.5 * (u[AT(i - 1, j, k)] + u[AT(i, j, k)]);
                    double un = 0.5 * (u[AT(i, j, k)] + u[AT(i, j + 1, k)]), us_ = 0.5 * (u[AT(i, j - 1, k)] + u[AT(i, j, k)]);
                    double ut = 0.5 * (u[AT(i, j, k)] + u[AT(i, j, k + 1)]), ub = 0.5 * (u[AT(i, j, k - 1)] + u[AT(i, j, k)]);
                    double vn = 0.5 * (v[AT(i, j, k)] + v[AT(i + 1, j, k)]), vs_ = 0.5 * (v[AT(i, j - 1, k)] + v[AT(i + 1, j - 1, k)]);
                    double wt = 0.5 * (w[AT(i, j, k)] + w[AT(i + 1, j, k)]), wb = 0.5 * (w[AT(i, j, k - 1)] + w[AT(i + 1, j, k - 1)]);
                    double conv = -((ue * ue - uw * uw) / dx + (un * vn - us_ * vs_) / dy + (ut * wt - ub * wb) / dz);
                    double txx_e = 2.0 * MU(i + 1, j, k) * (u[AT(i + 1, j, k)] - u[AT(i, j, k)]) / dx;
                    double txx_w = 2.0 * MU(i, j, k) * (u[AT(i, j, k)] - u[AT(i - 1, j, k)]) / dx;
                    double mu_n = 0.25 * (MU(i, j, k) + MU(i + 1, j, k) + MU(i, j + 1, k) + MU(i + 1, j + 1, k));
                    double mu_s = 0.25 * (MU(i, j - 1, k) + MU(i + 1, j - 1, k) + MU(i, j, k) + MU(i + 1, j, k));
                    double mu_t = 0.25 * (MU(i, j, k) + MU(i + 1, j, k) + MU(i, j, k + 1) + MU(i + 1, j, k + 1));
                    double mu_b = 0.25 * (MU(i, j, k - 1) + MU(i + 1, j, k - 1) + MU(i, j, k) + MU(i + 1, j, k));
                    double txy_n = mu_n * ((u[AT(i, j + 1, k)] - u[AT(i, j, k)]) / dy + (v[AT(i + 1, j, k)] - v[AT(i, j, k)]) / dx);
                    double txy_s = mu_s * ((u[AT(i, j, k)] - u[AT(i, j - 1, k)]) / dy + (v[AT(i + 1, j - 1, k)] - v[AT(i, j - 1, k)]) / dx);
                    double txz_t = mu_t * ((u[AT(i, j, k + 1)] - u[AT(i, j, k)]) / dz + (w[AT(i + 1, j, k)] - w[AT(i, j, k)]) / dx);
                    double txz_b = mu_b * ((u[AT(i, j, k)] - u[AT(i, j, k - 1)]) / dz + (w[AT(i + 1, j, k - 1)] - w[AT(i, j, k - 1)]) / dx);
                    double rf = rho_fx(&g, phi, i, j, k);
                    double diff = ((txx_e - txx_w) / dx + (txy_n - txy_s) / dy + (txz_t - txz_b) / dz) / rf;
                    double src = gx;
                    if (kappa) src += sigma * 0.5 * (kappa[AT(i, j, k)] + kappa[AT(i + 1, j, k)]) * (phi[AT(i + 1, j, k)] - phi[AT(i, j, k)]) / dx / rf;
                    double m = conv + diff;
                    mnew_u[q] = m;
                    us[q] = u[q] + dt * (f1 * m - f2 * mold_u[q] + src);
                }
                /* ------------------------------------------------ y component, north face (i, j+1/2, k) */
                {
                    double vn = 0.5 * (v[AT(i, j, k)] + v[AT(i, j + 1, k)]), vs_ = 0.5 * (v[AT(i, j - 1, k)] + v[AT(i, j, k)]);
                    double ve = 0.5 * (v[AT(i, j, k)] + v[AT(i + 1, j, k)]), vw = 0.5 * (v[AT(i - 1, j, k)] + v[AT(i, j, k)]);
                    double vt = 0.5 * (v[AT(i, j, k)] + v[AT(i, j, k + 1)]), vb = 0.5 * (v[AT(i, j, k - 1)] + v[AT(i, j, k)]);
                    double ue = 0.5 * (u[AT(i, j, k)] + u[AT(i, j + 1, k)]), uw = 0.5 * (u[AT(i - 1, j, k)] + u[AT(i - 1, j + 1, k)]);
                    double wt = 0.5 * (w[AT(i, j, k)] + w[AT(i, j + 1, k)]), wb = 0.5 * (w[AT(i, j, k - 1)] + w[AT(i, j + 1, k - 1)]);
                    double conv = -((ve * ue - vw * uw) / dx + (vn * vn - vs_ * vs_) / dy + (vt * wt - vb * wb) / dz);
                    double tyy_n = 2.0 * MU(i, j + 1, k) * (v[AT(i, j + 1, k)] - v[AT(i, j, k)]) / dy;
                    double tyy_s = 2.0 * MU(i, j, k) * (v[AT(i, j, k)] - v[AT(i, j - 1, k)]) / dy;
                    double mu_e = 0.25 * (MU(i, j, k) + MU(i + 1, j, k) + MU(i, j + 1, k) + MU(i + 1, j + 1, k));
                    double mu_w = 0.25 * (MU(i - 1, j, k) + MU(i, j, k) + MU(i - 1, j + 1, k) + MU(i, j + 1, k));
                    double mu_t = 0.25 * (MU(i, j, k) + MU(i, j + 1, k) + MU(i, j, k + 1) + MU(i, j + 1, k + 1));
                    double mu_b = 0.25 * (MU(i, j, k - 1) + MU(i, j + 1, k - 1) + MU(i, j, k) + MU(i, j + 1, k));
                    double tyx_e = mu_e * ((v[AT(i + 1, j, k)] - v[AT(i, j, k)]) / dx + (u[AT(i, j + 1, k)] - u[AT(i, j, k)]) / dy);
                    double tyx_w = mu_w * ((v[AT(i, j, k)] - v[AT(i - 1, j, k)]) / dx + (u[AT(i - 1, j + 1, k)] - u[AT(i - 1, j, k)]) / dy);
                    double tyz_t = mu_t * ((v[AT(i, j, k + 1)] - v[AT(i, j, k)]) / dz + (w[AT(i, j + 1, k)] - w[AT(i, j, k)]) / dy);
                    double tyz_b = mu_b * ((v[AT(i, j, k)] - v[AT(i, j, k - 1)]) / dz + (w[AT(i, j + 1, k - 1)] - w[AT(i, j, k - 1)]) / dy);
                    double rf = rho_fy(&g, phi, i, j, k);
                    double diff = ((tyx_e - tyx_w) / dx + (tyy_n - tyy_s) / dy + (tyz_t - tyz_b) / dz) / rf;
                    double src = gy;
                    if (kappa) src += sigma * 0.5 * (kappa[AT(i, j, k)] + kappa[AT(i, j + 1, k)]) * (phi[AT(i, j + 1, k)] - phi[AT(i, j, k)]) / dy / rf;
                    double m = conv + diff;
                    mnew_v[q] = m;
                    vs[q] = v[q] + dt * (f1 * m - f2 * mold_v[q] + src);
                }
                /* ------------------------------------------------ z component, top face (i, j, k+1/2) */
                {
                    double wt = 0.5 * (w[AT(i, j, k)] + w[AT(i, j, k + 1)]), wb = 0.5 * (w[AT(i, j, k - 1)] + w[AT(i, j, k)]);
                    double we = 0.5 * (w[AT(i, j, k)] + w[AT(i + 1, j, k)]), ww = 0.5 * (w[AT(i - 1, j, k)] + w[AT(i, j, k)]);
                    double wn = 0.5 * (w[AT(i, j, k)] + w[AT(i, j + 1, k)]), ws_ = 0.5 * (w[AT(i, j - 1, k)] + w[AT(i, j, k)]);
                    double ue = 0.5 * (u[AT(i, j, k)] + u[AT(i, j, k + 1)]), uw = 0.5 * (u[AT(i - 1, j, k)] + u[AT(i - 1, j, k + 1)]);
                    double vn = 0.5 * (v[AT(i, j, k)] + v[AT(i, j, k + 1)]), vs_ = 0.5 * (v[AT(i, j - 1, k)] + v[AT(i, j - 1, k + 1)]);
                    double conv = -((we * ue - ww * uw) / dx + (wn * vn - ws_ * vs_) / dy + (wt * wt - wb * wb) / dz);
                    double tzz_t = 2.0 * MU(i, j, k + 1) * (w[AT(i, j, k + 1)] - w[AT(i, j, k)]) / dz;
                    double tzz_b = 2.0 * MU(i, j, k) * (w[AT(i, j, k)] - w[AT(i, j, k - 1)]) / dz;
                    double mu_e = 0.25 * (MU(i, j, k) + MU(i + 1, j, k) + MU(i, j, k + 1) + MU(i + 1, j, k + 1));
                    double mu_w = 0.25 * (MU(i - 1, j, k) + MU(i, j, k) + MU(i - 1, j, k + 1) + MU(i, j, k + 1));
                    double mu_n = 0.25 * (MU(i, j, k) + MU(i, j + 1, k) + MU(i, j, k + 1) + MU(i, j + 1, k + 1));
                    double mu_s = 0.25 * (MU(i, j - 1, k) + MU(i, j, k) + MU(i, j - 1, k + 1) + MU(i, j, k + 1));
                    double tzx_e = mu_e * ((w[AT(i + 1, j, k)] - w[AT(i, j, k)]) / dx + (u[AT(i, j, k + 1)] - u[AT(i, j, k)]) / dz);
                    double tzx_w = mu_w * ((w[AT(i, j, k)] - w[AT(i - 1, j, k)]) / dx + (u[AT(i - 1, j, k + 1)] - u[AT(i - 1, j, k)]) / dz);
                    double tzy_n = mu_n * ((w[AT(i, j + 1, k)] - w[AT(i, j, k)]) / dy + (v[AT(i, j, k + 1)] - v[AT(i, j, k)]) / dz);
                    double tzy_s = mu_s * ((w[AT(i, j, k)] - w[AT(i, j - 1, k)]) / dy + (v[AT(i, j - 1, k + 1)] - v[AT(i, j - 1, k)]) / dz);
                    double rf = rho_fz(&g, phi, i, j, k);
                    double diff = ((tzx_e - tzx_w) / dx + (tzy_n - tzy_s) / dy + (tzz_t - tzz_b) / dz) / rf;
                    double src = gz;
                    if (kappa) src += sigma * 0.5 * (kappa[AT(i, j, k)] + kappa[AT(i, j, k + 1)]) * (phi[AT(i, j, k + 1)] - phi[AT(i, j, k)]) / dz / rf;
                    double m = conv + diff;
                    mnew_w[q] = m;
                    ws[q] = w[q] + dt * (f1 * m - f2 * mold_w[q] + src);
                }
            }
#undef AT
#undef MU
    return 0;
}

/* ------------------------------------------------------ MTHINC volume of fluid */

/* SURVEY.md sec. 8(f) NEXT-4.  PAPER.md:104-132 (sec. 3.1, eqs. 8-12) and Appendix A, triply periodic,
 * with the LINEAR reconstruction T(x~) = n . x~ (the curvature tensor of eqs. A.3-A.5 set to zero) -- readings
 * R21-R26 of DESIGN.md.  One step, directional splitting x -> y -> z (Algorithm 2):
 *   for p = x, y, z  (s = n, x, y):
 *     in every cell reconstruct  H^(x~) = 1/2 [1 + tanh(beta (n . x~ + d))]  from phi^s          (eq. 10)
 *        n  = m~ / |m~|,  m~ = the Youngs gradient of phi^s in cell units (corner values averaged)  (A.6)
 *        d  from the volume constraint  int_cell H^ = phi^s  (A.8), the integral being exact along the direction of the
 *           largest |n| and a 2 x 2 Gauss quadrature across it (A.9-A.13)
 *        cells with phi^s outside (eps, 1 - eps) or without a gradient keep the constant state H^ = phi^s
 *     on every face along p the flux is the integral of the UPWIND cell's H^ over the part of that cell swept through the face
 *        in dt, exact along p and 2 x 2 Gauss across it (A.23-A.31)
 *     phi^p = [phi^s - (F_+ - F_-) / dl] / [1 - dt/dl (u_+ - u_-)]                                   (eq. 11)
 *   phi^(n+1) = phi^z - sum_p dt/dl_p phi^p (u^p_+ - u^p_-)                                            (eq. 12)
 * d is found here by bisection on the constraint itself (the definition; the paper's route is the quartic A.15). */
#define VOF_EPS 1e-8

/* ln cosh(x), stable for large |x| */
static double ln_cosh(double x) {
    double a = fabs(x);
    return a + log1p(exp(-2.0 * a)) - 0.69314718055994530941723212145818;
}
/* int_a^b 1/2 [1 + tanh(beta (alpha x + gamma))] dx */
static double tanh_integral(double a, double b, double alpha, double gamma, double beta) {
    if (fabs(alpha) < 1e-12) return (b - a) * 0.5 * (1.0 + tanh(beta * gamma));
    /* the antiderivative of tanh is ln cosh: int = 1/2 [(b - a) + (ln cosh z_b - ln cosh z_a) / (beta alpha)], z = beta (alpha x + gamma).
     * When the increment delta = z_b - z_a is small (a normal almost perpendicular to the direction of integration, or a
     * small swept interval) the two logarithms agree in their leading digits and their difference, divided by beta alpha,
     * would lose them: |alpha| = 1e-9 leaves 7 digits.  The same difference without cancellation:
     *   ln cosh z_b - ln cosh z_a = ln(cosh delta + tanh z_a sinh delta) = log1p(2 sinh^2(delta/2) + tanh z_a sinh delta) */
    double za = beta * (alpha * a + gamma), delta = beta * alpha * (b - a);
    if (fabs(delta) < 0.1) {
        double sh = sinh(0.5 * delta);
        return 0.5 * ((b - a) + log1p(2.0 * sh * sh + tanh(za) * sinh(delta)) / (beta * alpha));
    }
    return 0.5 * ((b - a) + (ln_cosh(beta * (alpha * b + gamma)) - ln_cosh(za)) / (beta * alpha));
}
/* the function above, for the pins (tests/test_oracle_pins_vof.py V9) */
double oracle_tanh_integral(double a, double b, double alpha, double gamma, double beta) { return tanh_integral(a, b, alpha, gamma, beta); }
static const double GAUSS2[2] = {0.5 - 0.28867513459481288225457439025098, 0.5 + 0.28867513459481288225457439025098};

/* mean of H^ over x~_dir in [a, b] and the full unit square across: exact along dir, 2 x 2 Gauss across (n: normal, d: offset) */
static double hat_integral(const double n[3], double d, int dir, double a, double b, double beta) {
    int t1 = (dir + 1) % 3, t2 = (dir + 2) % 3;
    double s = 0.0;
    for (int p = 0; p < 2; ++p)
        for (int q = 0; q < 2; ++q) s += tanh_integral(a, b, n[dir], n[t1] * GAUSS2[p] + n[t2] * GAUSS2[q] + d, beta);
    return 0.25 * s;
}

typedef struct { double n[3]; double d; int flat; } recon_t;   /* flat: H^ is the constant phi of the cell */

static void reconstruct_cell(const grid_t *g, const double *phi, int i, int j, int k, double beta, recon_t *r) {
    const int nx = g->nx, ny = g->ny, nz = g->nz;
    const double f = phi[at(g, i, j, k)];
    r->flat = 1; r->d = 0.0; r->n[0] = r->n[1] = r->n[2] = 0.0;
    if (!(f > VOF_EPS && f < 1.0 - VOF_EPS)) return;
    /* Youngs: the gradient at each of the 8 corners of the cell from the 8 cells around that corner (differences in
     * cell units: the reconstruction lives in the unit cube), then the mean of the 8 corner values */
    double m[3] = {0.0, 0.0, 0.0};
    for (int ck = 0; ck < 2; ++ck)
        for (int cj = 0; cj < 2; ++cj)
            for (int ci = 0; ci < 2; ++ci) {
                /* corner between cells (i-1+ci .. i+ci) x (j-1+cj .. j+cj) x (k-1+ck .. k+ck) */
                int i0 = wrap(i - 1 + ci, nx), i1 = wrap(i + ci, nx);
                int j0 = wrap(j - 1 + cj, ny), j1 = wrap(j + cj, ny);
                int k0 = wrap(k - 1 + ck, nz), k1 = wrap(k + ck, nz);
                double p000 = phi[at(g, i0, j0, k0)], p100 = phi[at(g, i1, j0, k0)], p010 = phi[at(g, i0, j1, k0)], p110 = phi[at(g, i1, j1, k0)];
                double p001 = phi[at(g, i0, j0, k1)], p101 = phi[at(g, i1, j0, k1)], p011 = phi[at(g, i0, j1, k1)], p111 = phi[at(g, i1, j1, k1)];
                m[0] += 0.25 * ((p100 - p000) + (p110 - p010) + (p101 - p001) + (p111 - p011));
                m[1] += 0.25 * ((p010 - p000) + (p110 - p100) + (p011 - p001) + (p111 - p101));
                m[2] += 0.25 * ((p001 - p000) + (p101 - p100) + (p011 - p010) + (p111 - p110));
            }
    m[0] *= 0.125; m[1] *= 0.125; m[2] *= 0.125;
    double mag = sqrt(m[0] * m[0] + m[1] * m[1] + m[2] * m[2]);
    if (!(mag > 1e-12)) return;
    r->flat = 0;
    for (int c = 0; c < 3; ++c) r->n[c] = m[c] / mag;
    /* direction of the exact integration: the largest |n|, ties to x, then y (cases 1-3) */
    double ax = fabs(r->n[0]), ay = fabs(r->n[1]), az = fabs(r->n[2]);
    int dir = (ax >= ay && ax >= az) ? 0 : ((ay >= az) ? 1 : 2);
    /* volume constraint (A.8, A.10): the cell mean of H^ equals phi; monotone in d -> bisection */
    double lo = -(2.0 + 40.0 / beta), hi = 2.0 + 40.0 / beta;
    for (int it = 0; it < 200; ++it) {
        double mid = 0.5 * (lo + hi);
        if (hat_integral(r->n, mid, dir, 0.0, 1.0, beta) < f) lo = mid; else hi = mid;
    }
    r->d = 0.5 * (lo + hi);
}

/* the flux (phase-1 volume per unit face area) through the face between cell (i,j,k) and its next neighbour along dir */
static double face_flux_vof(const grid_t *g, const double *phi, const recon_t *rec, int i, int j, int k, int dir,
                            double vel, double dl, double dt, double beta) {
    double c = vel * dt / dl;                                   /* local CFL number, A.26 / A.30 / A.31 */
    int iu = i, ju = j, ku = k;
    double a, b, sign;
    if (c >= 0.0) { a = 1.0 - c; b = 1.0; sign = 1.0; }          /* donor = this cell, its last c of the way */
    else {
        if (dir == 0) iu = wrap(i + 1, g->nx); else if (dir == 1) ju = wrap(j + 1, g->ny); else ku = wrap(k + 1, g->nz);
        a = 0.0; b = -c; sign = -1.0;                            /* donor = the next cell, its first |c| */
    }
    const recon_t *r = &rec[at(g, iu, ju, ku)];
    double vol = r->flat ? (b - a) * phi[at(g, iu, ju, ku)] : hat_integral(r->n, r->d, dir, a, b, beta);
    return sign * dl * vol;
}

int oracle_vof_step(int nx, int ny, int nz, double lx, double ly, double lz, double beta, double dt,
                    const double *phi, const double *u, const double *v, const double *w, double *phi_out, int nthreads) {
    grid_t g;
    if (grid_init(&g, nx, ny, nz, lx, ly, lz, ORACLE_BC_Z_PERIODIC, 1.0, 1.0, dt)) return 1;
    if (!(beta > 0.0) || !(dt > 0.0)) return 1;
    set_threads(nthreads);
    const size_t n = (size_t)nx * ny * nz;
    recon_t *rec = (recon_t *)malloc(sizeof(recon_t) * n);
    double *cur = (double *)malloc(sizeof(double) * n), *flux = (double *)malloc(sizeof(double) * n);
    double *ps[3] = {(double *)malloc(sizeof(double) * n), (double *)malloc(sizeof(double) * n), (double *)malloc(sizeof(double) * n)};
    int rc = 0;
    if (!rec || !cur || !flux || !ps[0] || !ps[1] || !ps[2]) { rc = 2; goto done; }
    memcpy(cur, phi, sizeof(double) * n);
    const double *vel[3] = {u, v, w};
    const double dl[3] = {g.dx, g.dy, g.dz};
    for (int dir = 0; dir < 3; ++dir) {
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) reconstruct_cell(&g, cur, i, j, k, beta, &rec[at(&g, i, j, k)]);
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i)
                    flux[at(&g, i, j, k)] = face_flux_vof(&g, cur, rec, i, j, k, dir, vel[dir][at(&g, i, j, k)], dl[dir], dt, beta);
#pragma omp parallel for collapse(2) schedule(static)
        for (int k = 0; k < nz; ++k)
            for (int j = 0; j < ny; ++j)
                for (int i = 0; i < nx; ++i) {
                    size_t q = at(&g, i, j, k);
                    size_t qm = dir == 0 ? at(&g, wrap(i - 1, nx), j, k) : (dir == 1 ? at(&g, i, wrap(j - 1, ny), k) : at(&g, i, j, wrap(k - 1, nz)));
                    double du = vel[dir][q] - vel[dir][qm];
                    ps[dir][q] = (cur[q] - (flux[q] - flux[qm]) / dl[dir]) / (1.0 - dt / dl[dir] * du);      /* eq. (11) */
                }
        memcpy(cur, ps[dir], sizeof(double) * n);
    }
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                size_t q = at(&g, i, j, k);
                double du = u[q] - u[at(&g, wrap(i - 1, nx), j, k)], dv = v[q] - v[at(&g, i, wrap(j - 1, ny), k)];
                double dw = w[q] - w[at(&g, i, j, wrap(k - 1, nz))];
                phi_out[q] = ps[2][q] - (dt / g.dx * ps[0][q] * du + dt / g.dy * ps[1][q] * dv + dt / g.dz * ps[2][q] * dw);   /* eq. (12) */
            }
done:
    free(rec); free(cur); free(flux); free(ps[0]); free(ps[1]); free(ps[2]);
    return rc;
}

/* the reconstruction alone, for the pins: n (3 doubles per cell, x fastest over cells), d and the flat flag per cell */
int oracle_vof_reconstruct(int nx, int ny, int nz, double beta, const double *phi, double *n_out, double *d_out, int *flat_out, int nthreads) {
    grid_t g;
    if (grid_init(&g, nx, ny, nz, 1.0, 1.0, 1.0, ORACLE_BC_Z_PERIODIC, 1.0, 1.0, 1.0)) return 1;
    if (!(beta > 0.0)) return 1;
    set_threads(nthreads);
#pragma omp parallel for collapse(2) schedule(static)
    for (int k = 0; k < nz; ++k)
        for (int j = 0; j < ny; ++j)
            for (int i = 0; i < nx; ++i) {
                recon_t r;
                reconstruct_cell(&g, phi, i, j, k, beta, &r);
                size_t q = at(&g, i, j, k);
                n_out[3 * q] = r.n[0]; n_out[3 * q + 1] = r.n[1]; n_out[3 * q + 2] = r.n[2];
                d_out[q] = r.d; flat_out[q] = r.flat;
            }
    return 0;
}
