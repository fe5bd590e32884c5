/*
 * oracle.h -- TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Plain, slow, fp64 CPU statement of the pressure-correction (projection) step of
 * the FluTAS two-fluid method, written from the paper (PAPER.md = arxiv 2204.08834):
 *   PAPER.md:76   eq. (2)       one-fluid density  rho = rho1*phi + rho2*(1-phi)
 *   PAPER.md:102  sec. 3        staggered MAC grid, uniform spacing, scalars at centres
 *   PAPER.md:153-159 eqs.16-19  splitting terms, constant-coefficient Poisson equation,
 *                               velocity correction, pressure update
 *   PAPER.md:161                rho0 = min density, p_hat = time-extrapolated pressure,
 *                               wall remark (normal gradient vanishes at a wall)
 *   PAPER.md:167, 173-181       Fourier expansion in x, y -> tridiagonal system in z,
 *                               Gauss elimination; order of the nine solver steps
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * leg may load this library.  It shares no code with the CUDA path and imports
 * nothing from it.  Every function below is pinned by tests/test_oracle_pins.py
 * (eigenpairs, dense 8^3 bordered solve, residual, gauge, div-free, fixed point,
 * grouping identity, numpy.fft cross-check); none is "parity unpinned".
 *
 * Layout everywhere: x fastest, idx = i + nx*(j + ny*k), no ghost cells.
 * u[i,j,k] lives on the east face x_{i+1/2}, v on the north face, w on the top face;
 * p, phi at cell centres.  bc_z = 0: triply periodic; bc_z = 1: x, y periodic, z walls
 * (no-slip w = 0 at both walls, homogeneous Neumann for p); the bottom wall face is
 * not stored, the top wall face is w[.,.,nz-1] and must be 0 on entry.
 *
 * All functions return 0 on success, non-zero on bad arguments / allocation failure.
 * nthreads <= 0 means "all cores" (OpenMP default).  OpenMP is used only across
 * independent lines / systems / grid points, never inside a recurrence or a sum.
 */
#ifndef FLUTAS_ORACLE_H
#define FLUTAS_ORACLE_H

#ifdef __cplusplus
extern "C" {
#endif

enum { ORACLE_BC_Z_PERIODIC = 0, ORACLE_BC_Z_WALL = 1 };
/* per-direction boundary conditions of the *_bc functions below (homogeneous pressure conditions, PAPER.md:61, 163,
 * 167): PERIODIC; NEUMANN = a wall (u_n = 0, dp/dn = 0 on the boundary faces); DIRICHLET = p = 0 ON the boundary
 * faces (Poisson problem and operators only: the step needs the boundary-normal velocity on both boundary faces, which
 * the nx-faces-per-line layout does not store). */
enum { ORACLE_BC_PERIODIC = 0, ORACLE_BC_NEUMANN = 1, ORACLE_BC_DIRICHLET = 2 };

/* rhs = rho0/dt * div(u*) + div[(1 - rho0/rho_f) grad p_hat],  p_hat = 2 p - p_old
 * (north_star grouping of eqs. 16-17; reading R1 of DESIGN.md). */
int oracle_rhs(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
               double rho1, double rho2, double dt,
               const double *u, const double *v, const double *w, const double *phi,
               const double *p, const double *p_old, double *rhs_out, int nthreads);

/* Solve L p = rhs, L = div grad (7-point Laplacian), zero-mean gauge, by the
 * eigen-expansion of PAPER.md:167, 173-181 with NAIVE O(n^2) DFTs along x and y and
 * (periodic z) a naive DFT along z + division by lambda_x+lambda_y+lambda_z with the
 * (0,0,0) mode set to 0, or (wall z) textbook Thomas per (kx,ky) with the singular
 * (0,0) column pinned (x_{nz-1} = 0) and its mean removed.
 * imag_residue_out (nullable): max |Im p| / max |Re p| before the real part is taken. */
int oracle_poisson(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                   const double *rhs, double *p_out, double *imag_residue_out, int nthreads);

/* One full step, in place on u, v, w, p (phi, p_old untouched):
 *   rhs as above;  L p_new = rhs;
 *   u = u* - dt [ (1/rho0) grad p_new + (1/rho_f - 1/rho0) grad p_hat ];  p = p_new.
 * rhs_out nullable (receives the right-hand side). */
int oracle_projection_step(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                           double rho1, double rho2, double dt,
                           double *u, double *v, double *w, const double *phi,
                           double *p, const double *p_old, double *rhs_out, int nthreads);

/* The same two calls for a variable time step:
 *   p_hat = (1 + r) p^n - r p^(n-1),  r = dt_ratio = dt^(n+1) / dt^n >= 0;  dt = dt^(n+1).
 * dt_ratio = 1 is the constant-dt step above, bit for bit.  dt_ratio = 0 (the same formulas, no special case) is the
 * start-up step when no level n-1 exists: p_hat = p^n, and in the momentum prediction f1 = 1, f2 = 0, explicit Euler
 * (PAPER.md:140, 161 give the coefficients as functions of r; the paper does not describe its first step: DESIGN.md R29). */
int oracle_rhs_vdt(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                   double rho1, double rho2, double dt, double dt_ratio,
                   const double *u, const double *v, const double *w, const double *phi,
                   const double *p, const double *p_old, double *rhs_out, int nthreads);
int oracle_projection_step_vdt(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                               double rho1, double rho2, double dt, double dt_ratio,
                               double *u, double *v, double *w, const double *phi,
                               double *p, const double *p_old, double *rhs_out, int nthreads);

/* The last part of the step alone (eq. 18 in the north_star grouping), in place on u, v, w:
 *   u = u* - dt [ (1/rho0) grad p_new + (1/rho_f - 1/rho0) grad p_hat ],  p_hat = 2 p - p_old.
 * Lets a test check the velocity correction at full size given any p_new. */
int oracle_correction(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                      double rho1, double rho2, double dt,
                      double *u, double *v, double *w, const double *phi,
                      const double *p, const double *p_old, const double *p_new, int nthreads);

/* Same step in the paper's own incremental grouping, eqs. (16)-(19):
 *   u' = u* - dt/rho0 [ grad p^n - (1 - rho0/rho_f) grad p_hat ];  L psi = rho0/dt div u';
 *   u = u' - dt/rho0 grad psi;  p = p^n + psi - mean(p^n + psi).
 * Exact-arithmetic identical to oracle_projection_step; used as a cross-check pin. */
int oracle_projection_step_paper(int nx, int ny, int nz, double lx, double ly, double lz,
                                 int bc_z, double rho1, double rho2, double dt,
                                 double *u, double *v, double *w, const double *phi,
                                 double *p, const double *p_old, int nthreads);

/* Naive DFT of complex data along one axis of an (n_outer, n, n_inner) array
 * (C order, n_inner fastest): out[o][k][q] = sum_j in[o][j][q] * exp(sign*2*pi*i*k*j/n),
 * sign = -1 forward, +1 inverse; NOT normalised.  re/im are separate arrays.
 * Exposed so that kernel-level parity tests can compare single transform stages. */
int oracle_dft_axis(long n_outer, int n, long n_inner, int sign,
                    const double *in_re, const double *in_im,
                    double *out_re, double *out_im, int nthreads);

/* Discrete operators, exposed for the pins and for sampled checks at full size. */
int oracle_divergence(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                      const double *u, const double *v, const double *w, double *div_out,
                      int nthreads);
int oracle_laplacian(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                     const double *p, double *lap_out, int nthreads);

/* ---- the same path with non-periodic x / y ("all the possible homogeneous pressure boundary conditions",
 * PAPER.md:163, 167 "Fourier-based expansions [that] depend on the boundary conditions"; closed cavity PAPER.md:287).
 * bc_x, bc_y, bc_z in {ORACLE_BC_PERIODIC, _NEUMANN, _DIRICHLET}; with all-periodic x, y these are the functions above,
 * bit for bit (those call these). */

/* naive cosine (Neumann) / sine (Dirichlet) eigen-expansion of REAL data along one axis of an (n_outer, n, n_inner)
 * array: sign = -1 analysis c_m = <f, e_m> / |e_m|^2, sign = +1 synthesis f = sum_m c_m e_m, with
 * e_m[i] = cos(pi m (2i+1)/(2n)) or sin(pi (m+1)(2i+1)/(2n)): the eigenvectors of the cell-centred second difference. */
int oracle_r2r_axis(long n_outer, int n, long n_inner, int bc, int sign,
                    const double *in, double *out, int nthreads);
/* the eigenvalue of mode m = 0..n-1 of the second difference with spacing d under bc (R6) */
int oracle_eigenvalues(int n, double d, int bc, double *lam_out);

int oracle_divergence_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                         const double *u, const double *v, const double *w, double *div_out, int nthreads);
int oracle_laplacian_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                        const double *p, double *lap_out, int nthreads);
/* L p = rhs with the given conditions; the zero-mean gauge (R5) applies when no direction is Dirichlet, otherwise L is
 * non-singular and nothing is removed.  Non-periodic z: Thomas with first / last diagonal -1/dz^2 + lam (Neumann) or
 * -3/dz^2 + lam (Dirichlet). */
int oracle_poisson_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                      const double *rhs, double *p_out, double *imag_residue_out, int nthreads);
/* rhs / correction / whole step with walls along any direction (no Dirichlet); dt_ratio as in the _vdt calls */
int oracle_rhs_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                  double rho1, double rho2, double dt, double dt_ratio,
                  const double *u, const double *v, const double *w, const double *phi,
                  const double *p, const double *p_old, double *rhs_out, int nthreads);
int oracle_correction_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                         double rho1, double rho2, double dt,
                         double *u, double *v, double *w, const double *phi,
                         const double *p, const double *p_old, const double *p_new, int nthreads);
int oracle_projection_step_bc(int nx, int ny, int nz, double lx, double ly, double lz, int bc_x, int bc_y, int bc_z,
                              double rho1, double rho2, double dt, double dt_ratio,
                              double *u, double *v, double *w, const double *phi,
                              double *p, const double *p_old, double *rhs_out, int nthreads);

/* ---- momentum prediction, eq. (15) (eq. (5)), triply
 * periodic:  u** = u^n + dt [ (1 + r/2) M(u^n) - (r/2) M(u^(n-1)) + g + sigma kappa grad(phi) / rho_f ],  r = dt_ratio,
 * M(u) = -div(u u) + (1/rho_f) div[ mu (grad u + grad u^T) ], central differences on the staggered grid, mu = mu1 phi +
 * mu2 (1 - phi) (see oracle.c for every face formula).  In: u, v, w = u^n, mold_* = M(u^(n-1)), kappa (nullable) the
 * cell-centred curvature.  Out: us, vs, ws = u**, mnew_* = M(u^n).  No array may alias another. */
int oracle_momentum_prediction(int nx, int ny, int nz, double lx, double ly, double lz,
                               double rho1, double rho2, double mu1, double mu2, double sigma,
                               double gx, double gy, double gz, double dt, double dt_ratio,
                               const double *u, const double *v, const double *w, const double *phi, const double *kappa,
                               const double *mold_u, const double *mold_v, const double *mold_w,
                               double *us, double *vs, double *ws,
                               double *mnew_u, double *mnew_v, double *mnew_w, int nthreads);

/* ---- MTHINC volume-of-fluid step (eqs. 8-12; Appendix A),
 * triply periodic, linear reconstruction T = n . x~, directional splitting x -> y -> z, one step:
 * phi (cell centres) and u, v, w (faces) in, phi_out = phi^(n+1).  See oracle.c for every formula and DESIGN.md R21-R26
 * for the readings (Gauss points, flat cells, normalised normal, flux quadrature). */
int oracle_vof_step(int nx, int ny, int nz, double lx, double ly, double lz, double beta, double dt,
                    const double *phi, const double *u, const double *v, const double *w, double *phi_out, int nthreads);
/* the reconstruction of every cell alone: unit normal (3 per cell), offset d, and whether the cell keeps a constant state */
int oracle_vof_reconstruct(int nx, int ny, int nz, double beta, const double *phi, double *n_out, double *d_out,
                           int *flat_out, int nthreads);

/* int_a^b 1/2 [1 + tanh(beta (alpha x + gamma))] dx, the one-dimensional integral every volume and flux of the MTHINC
 * reconstruction is made of (eq. 10 integrated along one direction; A.9-A.13, A.27): exposed for the pins. */
double oracle_tanh_integral(double a, double b, double alpha, double gamma, double beta);

/* number of OpenMP threads a call with this nthreads argument would use */
int oracle_threads(int nthreads);

#ifdef __cplusplus
}
#endif
#endif
