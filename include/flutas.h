/*
 * flutas.h -- C ABI of libflutas_b200.so: the pressure-correction (projection) step of the
 * FluTAS two-fluid incompressible solver (arxiv 2204.08834; PAPER.md = the paper's text),
 * hand-written CUDA for NVIDIA B200 (sm_100a), fp64, one GPU.
 *
 * What one step computes (sec. 3.3 + 3.3.1; Algorithm 1 lines 10-13,
 * PAPER.md:211-218), in the grouping fixed by BASELINE.json's north_star (R1):
 *
 *   rho_c  = rho1*phi + rho2*(1-phi)                         eq. (2),
 *   rho_f  = mean of the two adjacent cell densities          (R2)
 *   p_hat  = 2 p^n - p^(n-1)                                  PAPER.md:161 (constant dt)
 *   rhs    = rho0/dt * div(u*) + div[(1 - rho0/rho_f) grad p_hat],  rho0 = min(rho1,rho2)
 *                                                             eqs. (16)-(17)
 *   L p^(n+1) = rhs, zero mean; L = 7-point Laplacian, solved by Fourier expansion in x, y
 *            and (periodic z) in z / (wall z) a tridiagonal solve per (kx,ky)
 *                                                             PAPER.md:163-167, 173-181
 *   u = u* - dt [ (1/rho0) grad p^(n+1) + (1/rho_f - 1/rho0) grad p_hat ]
 *                                                             eqs. (18)-(19)
 *
 * Grid and layout (R10): uniform spacing dx = lx/nx etc.; every field is
 * nx*ny*nz contiguous doubles, x fastest: idx = i + nx*(j + ny*k); no ghost cells.  p, phi live at
 * cell centres; u / v / w[i,j,k] live on the east / north / top face of cell (i,j,k).
 * x and y are periodic.  bc_z = FLUTAS_BC_Z_PERIODIC: z periodic.  bc_z = FLUTAS_BC_Z_WALL:
 * no-slip walls at z = 0 and z = lz (w = 0 there), homogeneous Neumann for p; the bottom wall face
 * is not stored; the top wall face is w[.,.,nz-1], MUST be 0 on entry (not checked) and is left
 * unchanged.
 *
 * All functions are extern "C", never throw and never call exit().  Unless a parameter says HOST,
 * pointers are DEVICE pointers.  The library never prints, reads no environment variable and has no
 * CPU fallback: without a CUDA device every call below fails with FLUTAS_ERR_CUDA / NULL.
 *
 * Arithmetic: fp64 throughout, no --use_fast_math.  The two reciprocals on the path -- 1/(rho_a + rho_b) of a face and
 * 1/(lambda_x + lambda_y + lambda_z) of a mode -- are the hardware seed (rcp.approx.ftz.f64) refined by two Newton
 * steps: relative error <= ~1 ulp, not the correctly rounded IEEE quotient (measured against the divide-based
 * CPU definition: <= 1e-14 relative L2 on every field).  The seed flushes subnormals, hence the density range below.
 */
#ifndef FLUTAS_H
#define FLUTAS_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct flutas_plan flutas_plan;

enum { FLUTAS_BC_Z_PERIODIC = 0, FLUTAS_BC_Z_WALL = 1 };
/* boundary conditions per direction (flutas_plan_create_ex): the homogeneous pressure conditions the FFT-based solver
 * covers.
 *   PERIODIC
 *   NEUMANN    a wall at both ends: u_n = 0, dp/dn = 0 on the boundary faces (what FLUTAS_BC_Z_WALL is along z).  The last
 *              stored face of the direction (u[nx-1,.,.], v[.,ny-1,.], w[.,.,nz-1]) is the wall face: it MUST be 0 on entry
 *              (not checked) and is left unchanged; the first wall face is not stored.  Closed cavity:
 *              NEUMANN in all three directions.
 *   DIRICHLET  p = 0 ON both boundary faces (ghost value = -interior value).  flutas_poisson_solve only: the step would
 *              need the boundary-normal velocity on both boundary faces and a line of n cells stores n faces.
 * Expansions: cosine (NEUMANN) / sine (DIRICHLET) series computed with the real-to-complex FFT machinery and pre- / post-
 * processing fused into the transform kernels; eigenvalues -2 (1 - cos(pi m / n)) / d^2 and
 * -2 (1 - cos(pi (m+1) / n)) / d^2.  With any DIRICHLET direction the operator is non-singular and no mean is removed. */
enum { FLUTAS_BC_PERIODIC = 0, FLUTAS_BC_NEUMANN = 1, FLUTAS_BC_DIRICHLET = 2 };

/* flags of flutas_plan_create_ex */
enum { FLUTAS_PLAN_CALLER_WORKSPACE = 1 };   /* do not allocate the workspace: flutas_plan_set_workspace supplies it */

enum {
    FLUTAS_OK = 0,
    FLUTAS_ERR_INVALID_ARG = 1,       /* NULL pointer, non-positive length / density / dt, bad bc_z   */
    FLUTAS_ERR_UNSUPPORTED_SIZE = 2,  /* see flutas_plan_create                                      */
    FLUTAS_ERR_ALLOC = 3,             /* cudaMalloc / host allocation failed                          */
    FLUTAS_ERR_CUDA = 4,              /* any other CUDA runtime error (message: flutas_last_error)    */
    FLUTAS_ERR_ALIAS = 5              /* two field arguments overlap, or are not 16-byte aligned      */
};

/* Create a plan for an nx x ny x nz grid on a box lx x ly x lz, on the CURRENT CUDA device.
 *   sizes:  nx, ny powers of two, 8 <= nx, ny <= 2048;
 *           bc_z periodic: nz a power of two, 8 <= nz <= 2048;  bc_z wall: any 2 <= nz <= 4096.
 *   rho1, rho2 in [1e-100, 1e100]: densities of phase 1 (phi = 1) and phase 2 (phi = 0);
 *           rho0 = min(rho1, rho2) (R3, R11).  With rho1 == rho2 the splitting
 *           coefficient (1 - rho0/rho_f) is exactly 0 (the classical constant-density projection).
 * The plan owns, on the device: twiddle and (permuted) eigenvalue tables (kilobytes), and -- unless
 * flutas_plan_create_ex was told FLUTAS_PLAN_CALLER_WORKSPACE -- a workspace of flutas_plan_workspace_bytes()
 * (one padded half-spectrum, four intermediate fields and, with walls, the elimination-coefficient table).
 * Returns NULL on failure; flutas_last_error() / flutas_last_error_code() say why.
 * A plan may be reused for any number of steps; one step in flight per plan (shared workspace). */
flutas_plan *flutas_plan_create(int nx, int ny, int nz, double lx, double ly, double lz,
                                int bc_z, double rho1, double rho2);

/* flutas_plan_create with boundary conditions per direction and flags (same problem;
 * "all the possible homogeneous pressure boundary conditions").
 *   bc_x, bc_y, bc_z: FLUTAS_BC_PERIODIC / _NEUMANN / _DIRICHLET (flutas_plan_create passes PERIODIC, PERIODIC, bc_z).
 *   sizes, beyond those of flutas_plan_create: non-periodic y: ny <= 1024; non-periodic x: 16 <= nx <= 1024, ny <= 1024,
 *          z not periodic and nz <= 444 (put a periodic direction first); otherwise FLUTAS_ERR_UNSUPPORTED_SIZE.
 *   FLUTAS_PLAN_CALLER_WORKSPACE: the plan allocates its small tables only; before the first step the caller hands it
 *   a device buffer with flutas_plan_set_workspace (e.g. one torch tensor, so that the framework's allocator
 *   accounts for every large byte).  A step on a plan without a workspace fails with FLUTAS_ERR_INVALID_ARG. */
flutas_plan *flutas_plan_create_ex(int nx, int ny, int nz, double lx, double ly, double lz,
                                   int bc_x, int bc_y, int bc_z, double rho1, double rho2, unsigned flags);

/* Bytes of workspace a plan for this grid needs (no plan, no device needed; 0 for an unsupported grid):
 * the number flutas_plan_workspace_bytes returns for such a plan.  PAPER.md:146-163 (sizes the solve of eq. 17). */
size_t flutas_workspace_bytes(int nx, int ny, int nz, int bc_x, int bc_y, int bc_z);

/* Make the plan use the caller's device buffer [dev_ptr, dev_ptr + bytes) as its workspace (the
 * intermediate arrays of eqs. 16-18 and of the solver steps 1-9).
 *   dev_ptr: device memory, 256-byte aligned, bytes >= flutas_plan_workspace_bytes(plan); the caller keeps
 *            ownership and must keep it alive and otherwise unused while the plan may run; contents need not be
 *            preserved between steps by the caller, but are (the coefficient table of the wall solve lives there).
 *   dev_ptr == NULL: go back to a plan-owned workspace (allocated here).
 * Synchronises the device, releases a plan-owned workspace, rebuilds the tensor maps and the wall coefficient
 * table.  FLUTAS_ERR_INVALID_ARG for a misaligned or too small buffer. */
int flutas_plan_set_workspace(flutas_plan *plan, void *dev_ptr, size_t bytes);

/* One projection step, enqueued on `stream` (a cudaStream_t passed as void*; NULL = legacy
 * default stream).  Returns without synchronising; no device<->host copy is made.
 *   in : u, v, w = provisional velocity u* (the paper's u**, before the splitting terms);
 *        phi = VoF colour phi^(n+1);  p = p^n;  p_old = p^(n-1);  dt > 0.
 *   out: u, v, w = u^(n+1) in place;  p = p^(n+1) (zero mean) in place;  phi, p_old untouched.
 * The six arrays must be 16-byte aligned and pairwise non-overlapping (FLUTAS_ERR_ALIAS).
 * Launch errors are returned as FLUTAS_ERR_CUDA; asynchronous faults surface at the caller's
 * next synchronisation. */
int flutas_projection_step(flutas_plan *plan, double *u, double *v, double *w, const double *phi,
                           double *p, const double *p_old, double dt, void *stream);

/* The time-stepping form of the same step:
 *   dt_ratio = r = dt^(n+1) / dt^n > 0 selects the variable-time-step extrapolation
 *              p_hat = (1 + r) p^n - r p^(n-1)   (r = 1: p_hat = 2 p^n - p^(n-1), the call above, bit for bit);
 *              dt = dt^(n+1).
 *   p_out    receives p^(n+1) (zero mean).  It may be
 *              == p      in place (what flutas_projection_step does),
 *              == p_old  ping-pong: a time loop then just swaps the two pointers for the next step
 *                        (p^(n-1) is dead once the right-hand side has been formed) -- no copy of p per step,
 *              or a seventh array (p and p_old are then left untouched).
 *            Any other overlap between the seven arrays is FLUTAS_ERR_ALIAS.
 * Everything else as flutas_projection_step.  The call only enqueues kernels on `stream` (no allocation,
 * no synchronisation, no host<->device copy), so it may be recorded into a CUDA graph by stream capture
 * (per-kernel timing must be off while capturing). */
int flutas_projection_step_ex(flutas_plan *plan, double *u, double *v, double *w, const double *phi,
                              const double *p, const double *p_old, double *p_out, double dt,
                              double dt_ratio, void *stream);

/* The same step for HOST arrays (same layout; pinned memory makes the copies asynchronous):
 * copies the six inputs host->device into plan-owned staging buffers (allocated on first use,
 * 6 fields), runs flutas_projection_step, copies u, v, w, p back and SYNCHRONISES `stream`.
 * This is the end-to-end entry point that bench.py times as `e2e`. */
int flutas_projection_step_host(flutas_plan *plan, double *u_host, double *v_host, double *w_host,
                                const double *phi_host, double *p_host, const double *p_old_host,
                                double dt, void *stream);

/* One whole velocity / pressure update: the momentum prediction of eq. (15) fused with the projection step
 * (Algorithm 1 lines 10-13):
 *     u** = u^n + dt [ (1 + r/2) M(u^n) - (r/2) M(u^(n-1)) + g + sigma kappa grad(phi) / rho_f ],   r = dt_ratio
 *     M(u) = - div(u u) + (1/rho_f) div[ mu (grad u + grad u^T) ],  mu = mu1 phi + mu2 (1 - phi)     (eqs. 5, 15, 2)
 * (central differences on the staggered grid: divergence-form convection with two-point means, normal stresses with
 * the cell viscosity, shear stresses with the mean viscosity of the four cells around an edge, 1/rho on the face with
 * the face density of the projection; surface tension as the continuum surface force with a given cell-centred
 * curvature field; gravity with rho_hat = rho: DESIGN.md R18-R20), then exactly flutas_projection_step_ex on u**.
 * ONE kernel forms u**, the splitting terms and the right-hand side, so u** never travels through HBM.
 *   in : u, v, w = u^n;  phi = phi^(n+1);  kappa = curvature at cell centres, or NULL (no surface tension);
 *        p = p^n, p_old = p^(n-1);  m_old_* = M(u^(n-1));  mu1, mu2 >= 0, sigma, g: plain numbers;  dt > 0, dt_ratio >= 0.
 *        FIRST STEP of a run (no level n-1 yet): pass dt_ratio = 0.  The Adams-Bashforth weights are then 1 and 0 (explicit
 *        Euler) and p_hat = p^n, so m_old_* and p_old are multiplied by zero: they must be valid arrays of finite numbers
 *        (e.g. zeros), their values do not matter.  m_new_* = M(u^0) comes back for the second step (R29).
 *   out: u, v, w = u^(n+1) in place;  p_out = p^(n+1) (may be p or p_old, as in flutas_projection_step_ex);
 *        m_new_* = M(u^n) (the caller swaps the two sets for the next step).
 * Triply periodic plans with nx a multiple of 32 only (FLUTAS_ERR_UNSUPPORTED_SIZE otherwise).  All arrays are N doubles on
 * the device, 16-byte aligned, pairwise distinct except p_out.  Enqueues on `stream`, no synchronisation. */
int flutas_time_step(flutas_plan *plan, double *u, double *v, double *w, const double *phi, const double *kappa,
                     const double *p, const double *p_old, double *p_out,
                     const double *m_old_u, const double *m_old_v, const double *m_old_w,
                     double *m_new_u, double *m_new_v, double *m_new_w,
                     double mu1, double mu2, double sigma, double gx, double gy, double gz,
                     double dt, double dt_ratio, void *stream);

/* The first kernel of flutas_time_step alone (kernel-level parity tests): us/vs/ws_out = u' = u** + the splitting term
 * (u** itself when p == NULL: no splitting terms), rhs_out = rho0/dt div(u'), m_new_* = M(u^n).  Inputs are not modified. */
int flutas_momentum_rhs(flutas_plan *plan, const double *u, const double *v, const double *w, const double *phi,
                        const double *kappa, const double *p, const double *p_old,
                        const double *m_old_u, const double *m_old_v, const double *m_old_w,
                        double *m_new_u, double *m_new_v, double *m_new_w,
                        double mu1, double mu2, double sigma, double gx, double gy, double gz,
                        double dt, double dt_ratio, double *us_out, double *vs_out, double *ws_out, double *rhs_out,
                        void *stream);

/* One step of the MTHINC volume-of-fluid method (eqs. 8-12; Appendix A,
 * PAPER.md:446-653; Algorithm 1 line 6, Algorithm 2): phi^n -> phi^(n+1) with the velocity u^n, directional splitting
 * x -> y -> z, hyperbolic-tangent reconstruction with sharpness beta (the paper's runs use 2 and 3) and the
 * LINEAR surface T = n . x~ (curvature tensor zero), Youngs normals, the volume constraint solved in the
 * paper's polynomial form (A.14-A.16), fluxes by exact integration along the sweep and 2 x 2 Gauss points across it,
 * the divergence correction of eq. (12).  Cells with phi outside (1e-8, 1 - 1e-8) or without a gradient carry a constant
 * state (R21-R26).  Triply periodic plans only (FLUTAS_ERR_UNSUPPORTED_SIZE otherwise).
 *   phi, u, v, w: N doubles each on the device (phi at cell centres, u / v / w on east / north / top faces); not modified
 *   phi_out: N doubles; may be phi itself (in place).  beta > 0, dt > 0.
 * Uses four fields of the plan's workspace (one step of anything in flight per plan).  Enqueues on `stream`. */
int flutas_vof_step(flutas_plan *plan, const double *phi, const double *u, const double *v, const double *w,
                    double *phi_out, double beta, double dt, void *stream);

/* flutas_vof_step for callers that must not allocate device memory (same method, same kernels: eqs. 8-12;
 * Appendix A; Algorithm 2).
 *
 * For whom: a solver embedded in an application whose own memory pool already owns the whole GPU (any further cudaMalloc
 * fails there), a routine called from inside a latency-critical pipeline (cudaMalloc synchronises the device, so every
 * stream of the host application would stall on it), or code bound by a "nothing is allocated after start-up" rule.
 * Such a caller cannot use flutas_vof_step: that one needs a plan, flutas_plan_create allocates the plan's tables, and
 * the step works in four fields of the plan's workspace.
 *
 * This call takes NO plan and allocates NOTHING, neither on the device nor on the host (no cudaMalloc / cudaFree, no
 * allocating library routine).  The grid is described by its arguments, and the step's four intermediate fields
 * (the fluxes of one sweep, phi after each of the three sweeps) are kept in one statically sized array inside the library:
 * 4 x FLUTAS_VOF_NOALLOC_MAX_CELLS doubles = 64 MiB, which every GPU that loads this part of the library holds until the
 * process exits.  The price of "no allocation" is therefore a size limit:
 *   nx * ny * nz <= FLUTAS_VOF_NOALLOC_MAX_CELLS (2^21, e.g. 128^3), else FLUTAS_ERR_UNSUPPORTED_SIZE and nothing is
 *   launched;  nx, ny, nz >= 3, any value (not only powers of two);  triply periodic;  lx, ly, lz, beta, dt > 0.
 *   phi, u, v, w, phi_out: caller-owned DEVICE arrays of nx*ny*nz doubles on the current device, layout and alignment as
 *   for flutas_vof_step; inputs are not modified; phi_out may be phi itself, any other overlap is FLUTAS_ERR_ALIAS.
 * Enqueues seven kernels on `stream` and returns without synchronising; results agree with flutas_vof_step on the same
 * grid to round-off.
 *
 * First call on a device: the entry point looks up, once per device and with that device current, the address its
 * static array has on that GPU (cudaGetSymbolAddress; this is also when the driver places the array in that GPU's
 * memory).  Make that first call during start-up, before any stream capture begins.
 * Shared scratch: there is ONE array per GPU for the whole process, and it keeps what the last call left in it.  A call
 * needs none of it cleared (every element it reads it has written itself first), but two calls whose kernels can
 * overlap on the same GPU -- different streams without an ordering between them, or several host threads -- overwrite
 * each other's intermediate fields and give wrong results: keep all calls on one GPU ordered one after the other. */
#define FLUTAS_VOF_NOALLOC_MAX_CELLS 2097152
int flutas_vof_step_noalloc(int nx, int ny, int nz, double lx, double ly, double lz, const double *phi, const double *u,
                            const double *v, const double *w, double *phi_out, double beta, double dt, void *stream);
/* FLUTAS_VOF_NOALLOC_MAX_CELLS as the loaded library was built with (no device needed). */
size_t flutas_vof_step_noalloc_max_cells(void);

/* NULL is a no-op.  Frees every device and host resource of the plan (synchronises the device). */
void flutas_plan_destroy(flutas_plan *plan);

/* ---- the two halves of the step as calls of their own (used by the kernel-level parity tests) */

/* Part (a) of the step alone: rhs_out[idx] = rho0/dt div(u*) + div[(1-rho0/rho_f) grad p_hat]
 * (N doubles, device).  Inputs are not modified. */
int flutas_splitting_rhs(flutas_plan *plan, const double *u, const double *v, const double *w,
                         const double *phi, const double *p, const double *p_old, double dt,
                         double *rhs_out, void *stream);

/* flutas_splitting_rhs with the variable-time-step p_hat (dt_ratio as in flutas_projection_step_ex). */
int flutas_splitting_rhs_ex(flutas_plan *plan, const double *u, const double *v, const double *w,
                            const double *phi, const double *p, const double *p_old, double dt,
                            double dt_ratio, double *rhs_out, void *stream);

/* Part (b) alone: solve L p = rhs in the zero-mean gauge.  rhs and p_out are
 * N doubles on the device; p_out may alias rhs. */
int flutas_poisson_solve(flutas_plan *plan, const double *rhs, double *p_out, void *stream);

/* ---- introspection ---------------------------------------------------------------------- */

/* Thread-local, NUL-terminated description / code of the last failure in this thread. */
const char *flutas_last_error(void);
int flutas_last_error_code(void);

/* Bytes of workspace the plan needs (== flutas_workspace_bytes of its grid), whoever owns it; the plan's tables
 * (kilobytes) and the staging buffers of the _host entry are not included. */
size_t flutas_plan_workspace_bytes(const flutas_plan *plan);

/* Number of kernel launches one flutas_projection_step enqueues, and their names
 * (idx in [0, launches); returns NULL outside). */
int flutas_plan_kernel_launches(const flutas_plan *plan);
const char *flutas_plan_kernel_name(const flutas_plan *plan, int idx);
/* The device function launch idx runs with the plan as it is configured now (the name a profiler shows, without
 * template arguments), so that stored profiler captures can be matched to the code that is running. */
const char *flutas_plan_kernel_symbol(const flutas_plan *plan, int idx);

/* Per-kernel device timing.  flutas_plan_set_timing(plan, 1) makes every following step record a
 * CUDA event before and after each of its kernels on the step's stream (events only; no
 * synchronisation).  flutas_plan_read_timing SYNCHRONISES the events, adds up the elapsed time of
 * every kernel since the last read, writes ms_out[idx] = total milliseconds of kernel idx
 * (n_out >= flutas_plan_kernel_launches) and steps_out = number of steps covered, then resets.
 * At most 256 steps can be pending between two reads (older ones are dropped from the totals). */
int flutas_plan_set_timing(flutas_plan *plan, int enabled);
int flutas_plan_read_timing(flutas_plan *plan, float *ms_out, int n_out, int *steps_out);

/* Algorithmic (modelled) HBM bytes kernel idx moves per launch: 8 bytes x the fields it must read
 * and write once; used by bench.py for the roofline line. */
double flutas_plan_kernel_bytes(const flutas_plan *plan, int idx);

/* Kernel variants a plan can switch between (never needed for correctness; every value of every option is held to
 * the same parity tests in tests/test_gpu_variants.py and tests/test_gpu_momentum.py).  FLUTAS_ERR_INVALID_ARG for an unknown name or a value the plan
 * cannot take.
 *   "y16" = 0 | 1                 ny = 1024 only: 1 (default) = 16 x 8 x 8 register-resident kernel, 0 = 4-column path.
 *                                 Switching re-orders the eigenvalue tables (synchronises the device).
 *   "thomas" = 0 | 1              wall only: 1 (default when nz <= 512) = one-pass shared-memory elimination,
 *                                 0 = two sweeps through HBM (allocates its c' array, half a spectrum, on first use;
 *                                 plan-owned, outside the workspace)
 *   "thomas_warps" = 1 | 2        solving warps per CTA of the one-pass kernel (default 2)
 *   "mom_ty16" = 0 | 1            flutas_time_step / flutas_momentum_rhs: tiles of 32 x 16 cells (1, default; used when ny is a
 *                                 multiple of 16) or of 32 x 8 cells per CTA
 *   "chunk" = n >= 0              planes per launch group of the step (0, default: every kernel covers the grid)
 *   "overlap" = 0 | 1             chunked only: run the three kernels of a group on three internal streams */
int flutas_plan_set_option(flutas_plan *plan, const char *name, int value);

/* ---- the step on a z-slab decomposition over several GPUs ---------------------------
 *
 * PAPER.md:169-183 (sec. 3.3.1: slabs for the transforms along x and y, "all-to-all" transposes to make z local for the
 * Gauss elimination and back), PAPER.md:313, 364-368 (the transposes are the measured bottleneck of the multi-GPU runs).
 * Here the two all-to-alls are the STORE stage of the kernel before them: the last pass of the forward transform along
 * y writes every row straight into the z-local spectrum of the rank that owns it, and the z stage writes every plane
 * straight into the slab spectrum of the rank that owns it -- plain / TMA stores into peer memory over NVLink (or into
 * the same device when ranks share one).  No transpose kernel, no pack / unpack buffer, no NCCL data path.
 *
 * Decomposition: rank r of n_ranks owns planes r*nzl .. (r+1)*nzl - 1, nzl = nz / n_ranks.  Every field argument is a
 * LOCAL array of (nzl + 2) planes of nx*ny doubles (x fastest): plane 0 = the plane below the slab (owned by rank r-1),
 * planes 1 .. nzl = the slab, plane nzl + 1 = the plane above (rank r+1); periodic z wraps around, beyond a wall the
 * halo plane is never read.  On entry the halo planes of phi, p, p_old (both) and of w (plane 0) must hold the
 * neighbours' values; u, v need none.  On exit u, v, w are corrected on planes 1 .. nzl and p_out holds p^(n+1) on ALL
 * planes 0 .. nzl + 1 that exist (the z stage sends the two boundary planes of every slab to the neighbours as well), so
 * a time loop never exchanges pressure halos; phi and w* arrive with the halos their producers gave them.
 *
 * Buffers (caller-owned device memory, 256-byte aligned):
 *   workspace  flutas_slab_workspace_bytes: private to the rank;
 *   exchange   flutas_slab_exchange_bytes: the rank's two spectra; PEERS WRITE INTO IT, so it must be mapped in every
 *              rank's address space (CUDA IPC, torch symmetric memory, or one process) -- flutas_slab_plan_attach takes
 *              the n_ranks device pointers as THIS process sees them (a HOST array; entry `rank` is the own buffer).
 *              attach clears the own buffer: synchronise all ranks between attach and the first step.
 * A step is three calls, phase = 0, 1, 2, each only enqueueing kernels on `stream`; BETWEEN phases 0 -> 1 and 1 -> 2 all
 * ranks must have finished the earlier phase before any starts the later one (a stream-ordered barrier, e.g. an NCCL
 * all-reduce of one element; nothing when the ranks are driven phase by phase on one stream of one device):
 *   phase 0  right-hand side, transform along x, transform along y -> rows to their owners
 *   phase 1  z stage on the own rows of ky -> planes to their owners
 *   phase 2  inverse transforms along y and x, correction
 * Phases 0 and 2 take the fields (p_out may be p, p_old or a seventh array, as in flutas_projection_step_ex); phase 1
 * ignores them (NULL allowed).
 * Sizes: n_ranks a power of two <= 16 dividing ny and nz, nz / n_ranks a power of two; nx a power of two in [128, 1024];
 *        ny a power of two in [8, 1024]; periodic z: nz a power of two in [8, 1024]; wall z: nz <= 512.
 * Results equal flutas_projection_step on the assembled fields up to round-off (same kernels, same arithmetic). */
typedef struct flutas_slab_plan flutas_slab_plan;
flutas_slab_plan *flutas_slab_plan_create(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                                          double rho1, double rho2, int n_ranks, int rank);
size_t flutas_slab_workspace_bytes(int nx, int ny, int nz, int bc_z, int n_ranks);   /* 0: unsupported decomposition */
size_t flutas_slab_exchange_bytes(int nx, int ny, int nz, int bc_z, int n_ranks);
int flutas_slab_plan_attach(flutas_slab_plan *plan, void *workspace, size_t workspace_bytes,
                            void *const *exchange /* HOST array of n_ranks DEVICE pointers */, size_t exchange_bytes);
int flutas_slab_step_phase(flutas_slab_plan *plan, int phase, double *u, double *v, double *w, const double *phi,
                           const double *p, const double *p_old, double *p_out, double dt, double dt_ratio, void *stream);
void flutas_slab_plan_destroy(flutas_slab_plan *plan);

#ifdef __cplusplus
}
#endif
#endif /* FLUTAS_H */
