// flutas_slab.inl -- SURVEY.md sec. 8(f) NEXT-3: the projection step on a z-slab decomposition over several GPUs
// (slabs for the x and y transforms, "all-to-all" transposes around the Gauss elimination along z;
// the transposes are the measured bottleneck).  Included at the end of flutas.cu.
//
// Rank r of P owns planes r nzl .. (r + 1) nzl - 1 (nzl = nz / P) of the six fields and, for the z stage, rows
// r rpp .. (r + 1) rpp - 1 (rpp = ny / P) of the ky axis of the half-spectrum with ALL planes.  It holds two plans of
// reduced geometry (flutas_plan::role):
//   A  ROLE_SLAB    nx x ny x (nzl + 2): the local arrays with one halo plane below and one above; right-hand side,
//                   x and y transforms, correction -- the kernels of the one-GPU step, called on plane ranges;
//   B  ROLE_ZLOCAL  nx x rpp x nz: the z stage (transform along z / Gauss elimination) on its rows.
// There is no transpose kernel and no pack / unpack buffer: the last pass of the forward transform along y stores each
// row into the z-local spectrum of the rank that owns it, and the z stage stores each plane into the slab spectrum
// of the rank that owns it (plus the two halo planes of its neighbours), as plain stores / TMA stores into the peers'
// memory (kernels.cuh PeerScatter).  What is left of the two all-to-alls is one synchronisation after each, which the
// CALLER provides between the three phases (a stream-ordered barrier over all ranks: bench.py / slab.py use an NCCL
// all-reduce of one element; ranks that share a device and a stream need nothing).
//
// Because the z stage writes the solution into the neighbours' halo planes as well, the inverse transforms give
// p^(n+1) on planes 0 .. nzl + 1 of every rank: the correction needs no halo exchange, and in a time loop the halos of
// p and p_old are always in place; phi and w* arrive with the halos their producers (VoF, momentum) gave them.
struct flutas_slab_plan {
    int nx, ny, nz, bc_z, n_ranks, rank, nzl, rpp;
    flutas_plan *A, *B;
    size_t off_specz, off_specs, ex_bytes;   // layout of the exchange buffer (the same on every rank)
    bool attached;
    double norm;
};

static bool slab_sizes_supported(int nx, int ny, int nz, int bc_z, int P) {
    if (bc_z != FLUTAS_BC_Z_PERIODIC && bc_z != FLUTAS_BC_Z_WALL) return false;
    if (!is_pow2(P) || P < 1 || P > kMaxRanks) return false;
    if (!is_pow2(nx) || nx < Rhs3Geom::X || nx > 1024) return false;          // bulk-copy-fed RHS kernel, persistent x kernels
    if (!is_pow2(ny) || ny < 8 || ny > 1024 || ny % P != 0) return false;     // one-butterfly-per-thread y kernel
    if (nz % P != 0 || !is_pow2(nz / P)) return false;
    if (bc_z == FLUTAS_BC_Z_PERIODIC) return is_pow2(nz) && nz >= 8 && nz <= 1024;
    return nz >= 2 && ThomasGeom::smem_bytes(nz, ThomasGeom::C) <= 227 * 1024;   // one-pass elimination: nz <= 512
}

// a plan of reduced geometry: tables only, the workspace and the spectrum come with flutas_slab_plan_attach
static flutas_plan *slab_subplan(int role, int nx, int ny, int nz, double lx, double ly, double lz, int bc_z, double rho1,
                                 double rho2, int ny_full, int row0) {
    flutas_plan *pl = new (std::nothrow) flutas_plan();
    if (!pl) { fail(FLUTAS_ERR_ALLOC, "host allocation failed"); return nullptr; }
    memset(pl, 0, sizeof(*pl));
    pl->role = role;
    pl->nx = nx; pl->ny = ny; pl->nz = nz;
    pl->ny_full = ny_full; pl->row0 = row0;
    pl->bc[0] = pl->bc[1] = FLUTAS_BC_PERIODIC;
    pl->bc[2] = bc_z == FLUTAS_BC_Z_PERIODIC ? FLUTAS_BC_PERIODIC : FLUTAS_BC_NEUMANN;
    pl->bc_z = bc_z;
    pl->lx = lx; pl->ly = ly; pl->lz = lz; pl->rho1 = rho1; pl->rho2 = rho2;
    if (plan_build(pl, FLUTAS_PLAN_CALLER_WORKSPACE) != FLUTAS_OK) {
        flutas_plan_destroy(pl);
        return nullptr;
    }
    return pl;
}

static void slab_geometry(flutas_slab_plan *sp) {
    flutas_plan a, b;
    memset(&a, 0, sizeof(a)); memset(&b, 0, sizeof(b));
    a.role = ROLE_SLAB; a.nx = sp->nx; a.ny = a.ny_full = sp->ny; a.nz = sp->nzl + 2; a.bc_z = sp->bc_z;
    b.role = ROLE_ZLOCAL; b.nx = sp->nx; b.ny = sp->rpp; b.ny_full = sp->ny; b.nz = sp->nz; b.bc_z = sp->bc_z;
    plan_geometry(&a); plan_geometry(&b);
    sp->off_specz = 0;
    sp->off_specs = align_up(sizeof(double2) * (size_t)b.nspec);
    sp->ex_bytes = sp->off_specs + align_up(sizeof(double2) * (size_t)a.nspec);
}

extern "C" size_t flutas_slab_exchange_bytes(int nx, int ny, int nz, int bc_z, int n_ranks) {
    if (!slab_sizes_supported(nx, ny, nz, bc_z, n_ranks)) return 0;
    flutas_slab_plan sp{};
    sp.nx = nx; sp.ny = ny; sp.nz = nz; sp.bc_z = bc_z; sp.n_ranks = n_ranks; sp.nzl = nz / n_ranks; sp.rpp = ny / n_ranks;
    slab_geometry(&sp);
    return sp.ex_bytes;
}

extern "C" size_t flutas_slab_workspace_bytes(int nx, int ny, int nz, int bc_z, int n_ranks) {
    if (!slab_sizes_supported(nx, ny, nz, bc_z, n_ranks)) return 0;
    flutas_plan a, b;
    memset(&a, 0, sizeof(a)); memset(&b, 0, sizeof(b));
    a.role = ROLE_SLAB; a.nx = nx; a.ny = a.ny_full = ny; a.nz = nz / n_ranks + 2; a.bc_z = bc_z;
    b.role = ROLE_ZLOCAL; b.nx = nx; b.ny = ny / n_ranks; b.ny_full = ny; b.nz = nz; b.bc_z = bc_z;
    plan_geometry(&a); plan_geometry(&b);
    return a.bytes + b.bytes + 1024;
}

extern "C" void flutas_slab_plan_destroy(flutas_slab_plan *sp) {
    if (!sp) return;
    flutas_plan_destroy(sp->A);
    flutas_plan_destroy(sp->B);
    delete sp;
}

extern "C" flutas_slab_plan *flutas_slab_plan_create(int nx, int ny, int nz, double lx, double ly, double lz, int bc_z,
                                                     double rho1, double rho2, int n_ranks, int rank) {
    if (!(lx > 0.0) || !(ly > 0.0) || !(lz > 0.0) || !std::isfinite(lx + ly + lz)) {
        fail(FLUTAS_ERR_INVALID_ARG, "box lengths must be positive and finite");
        return nullptr;
    }
    if (!(rho1 >= 1e-100 && rho1 <= 1e100) || !(rho2 >= 1e-100 && rho2 <= 1e100)) {
        fail(FLUTAS_ERR_INVALID_ARG, "densities must lie in [1e-100, 1e100]");
        return nullptr;
    }
    if (rank < 0 || rank >= n_ranks) {
        fail(FLUTAS_ERR_INVALID_ARG, "rank %d outside [0, %d)", rank, n_ranks);
        return nullptr;
    }
    if (!slab_sizes_supported(nx, ny, nz, bc_z, n_ranks)) {
        fail(FLUTAS_ERR_UNSUPPORTED_SIZE,
             "unsupported slab decomposition of %d x %d x %d over %d ranks: n_ranks a power of two <= %d dividing ny and nz with "
             "nz / n_ranks a power of two; nx a power of two in [128, 1024]; ny a power of two in [8, 1024]; periodic z: nz a "
             "power of two in [8, 1024]; wall z: nz <= 512", nx, ny, nz, n_ranks, kMaxRanks);
        return nullptr;
    }
    int ndev = 0;
    if (cudaGetDeviceCount(&ndev) != cudaSuccess || ndev == 0) {
        cudaGetLastError();
        fail(FLUTAS_ERR_CUDA, "no CUDA device available (there is no CPU fallback)");
        return nullptr;
    }
    flutas_slab_plan *sp = new (std::nothrow) flutas_slab_plan();
    if (!sp) { fail(FLUTAS_ERR_ALLOC, "host allocation failed"); return nullptr; }
    sp->nx = nx; sp->ny = ny; sp->nz = nz; sp->bc_z = bc_z; sp->n_ranks = n_ranks; sp->rank = rank;
    sp->nzl = nz / n_ranks; sp->rpp = ny / n_ranks;
    sp->norm = 1.0 / ((double)nx * (double)ny * (bc_z == FLUTAS_BC_Z_WALL ? 1.0 : (double)nz));
    slab_geometry(sp);
    // A sees nzl + 2 planes of the same spacing: lz_A / (nzl + 2) is replaced by the exact lz / nz below
    sp->A = slab_subplan(ROLE_SLAB, nx, ny, sp->nzl + 2, lx, ly, lz, bc_z, rho1, rho2, ny, 0);
    sp->B = sp->A ? slab_subplan(ROLE_ZLOCAL, nx, sp->rpp, nz, lx, ly, lz, bc_z, rho1, rho2, ny, rank * sp->rpp) : nullptr;
    if (!sp->A || !sp->B) {
        flutas_slab_plan_destroy(sp);
        return nullptr;
    }
    sp->A->grid.inv_dz = 1.0 / (lz / nz);
    return sp;
}

static int upload_scatter(flutas_plan *pl, const PeerScatter &h) {
    if (!pl->sc_dev) CUDA_TRY(cudaMalloc((void **)&pl->sc_dev, sizeof(PeerScatter)));
    CUDA_TRY(cudaMemcpy(pl->sc_dev, &h, sizeof(PeerScatter), cudaMemcpyHostToDevice));
    return FLUTAS_OK;
}

extern "C" int flutas_slab_plan_attach(flutas_slab_plan *sp, void *workspace, size_t workspace_bytes, void *const *exchange,
                                       size_t exchange_bytes) {
    if (!sp || !workspace || !exchange) return fail(FLUTAS_ERR_INVALID_ARG, "NULL argument");
    const size_t need_ws = sp->A->bytes + sp->B->bytes + 1024;
    if (workspace_bytes < need_ws) return fail(FLUTAS_ERR_INVALID_ARG, "the workspace is too small: %zu bytes given, %zu needed", workspace_bytes, need_ws);
    if (exchange_bytes < sp->ex_bytes) return fail(FLUTAS_ERR_INVALID_ARG, "the exchange buffer is too small: %zu bytes given, %zu needed", exchange_bytes, sp->ex_bytes);
    if (((size_t)workspace) & 255) return fail(FLUTAS_ERR_INVALID_ARG, "the workspace must be 256-byte aligned");
    for (int r = 0; r < sp->n_ranks; ++r)
        if (!exchange[r] || (((size_t)exchange[r]) & 255))
            return fail(FLUTAS_ERR_INVALID_ARG, "exchange buffer %d is NULL or not 256-byte aligned", r);
    CUDA_TRY(cudaDeviceSynchronize());
    flutas_plan *A = sp->A, *B = sp->B;
    char *own = (char *)exchange[sp->rank];
    A->spec_ext = (double2 *)(own + sp->off_specs);
    B->spec_ext = (double2 *)(own + sp->off_specz);
    if (int rc = plan_attach_workspace(A, workspace, false)) return rc;
    if (int rc = plan_attach_workspace(B, (char *)workspace + align_up(A->bytes), false)) return rc;

    // forward: row j of the y transform of plane k (array index k_loc = 1 .. nzl) -> rank j / rpp, row j % rpp, plane
    // rank nzl + k_loc - 1 of its z-local spectrum
    PeerScatter fy{};
    int sh = 0;
    while ((1 << sh) < sp->rpp) ++sh;
    fy.shift = sh; fy.lead = 0; fy.halo = 0; fy.wrap = 0; fy.n_peers = sp->n_ranks;
    fy.row_stride = B->pitch; fy.outer_stride = B->plane; fy.outer_off = (long long)sp->rank * sp->nzl - 1;
    for (int r = 0; r < sp->n_ranks; ++r) fy.base[r] = (double2 *)((char *)exchange[r] + sp->off_specz);
    if (int rc = upload_scatter(A, fy)) return rc;
    // backward: plane k of the z stage's row j_loc -> rank k / nzl, plane k % nzl + 1, row rank rpp + j_loc of its slab
    // spectrum; the first / last plane of a slab also to the halo plane of the rank below / above
    PeerScatter bz{};
    sh = 0;
    while ((1 << sh) < sp->nzl) ++sh;
    bz.shift = sh; bz.lead = 1; bz.halo = 1; bz.wrap = sp->bc_z == FLUTAS_BC_Z_PERIODIC ? 1 : 0; bz.n_peers = sp->n_ranks;
    bz.row_stride = A->plane; bz.outer_stride = A->pitch; bz.outer_off = (long long)sp->rank * sp->rpp;
    for (int r = 0; r < sp->n_ranks; ++r) bz.base[r] = (double2 *)((char *)exchange[r] + sp->off_specs);
    if (int rc = upload_scatter(B, bz)) return rc;
    B->sc_npeers = sp->n_ranks; B->sc_nzl = sp->nzl; B->sc_srows = sp->nzl < 256 ? sp->nzl : 256;
    if (sp->bc_z == FLUTAS_BC_Z_WALL) {   // tensor maps of the peers' slab spectra for the tile stores of the elimination
        if (!B->tpm) B->tpm = new (std::nothrow) ThomasPeerMaps();
        if (!B->tpm) return fail(FLUTAS_ERR_ALLOC, "host allocation failed");
        for (int r = 0; r < sp->n_ranks; ++r)
            if (int rc = make_spectrum_map(A, &B->tpm->m[r], ThomasGeom::C, 2, A->nz, B->sc_srows, bz.base[r])) return rc;
    }
    sp->attached = true;
    return FLUTAS_OK;
}

extern "C" int flutas_slab_step_phase(flutas_slab_plan *sp, int phase, double *u, double *v, double *w, const double *phi,
                                      const double *p, const double *p_old, double *p_out, double dt, double dt_ratio,
                                      void *stream) {
    if (!sp) return fail(FLUTAS_ERR_INVALID_ARG, "NULL plan");
    if (!sp->attached) return fail(FLUTAS_ERR_INVALID_ARG, "the plan has no buffers (flutas_slab_plan_attach)");
    if (phase < 0 || phase > 2) return fail(FLUTAS_ERR_INVALID_ARG, "phase must be 0, 1 or 2");
    if (!(dt > 0.0) || !std::isfinite(dt)) return fail(FLUTAS_ERR_INVALID_ARG, "dt must be positive and finite");
    if (!(dt_ratio > 0.0) || !std::isfinite(dt_ratio)) return fail(FLUTAS_ERR_INVALID_ARG, "dt_ratio must be positive and finite");
    flutas_plan *A = sp->A, *B = sp->B;
    cudaStream_t st = (cudaStream_t)stream;
    const int nzl = sp->nzl;
    const bool wall = sp->bc_z == FLUTAS_BC_Z_WALL, bottom = wall && sp->rank == 0, top = wall && sp->rank == sp->n_ranks - 1;
    const long long plane = (long long)sp->nx * sp->ny;
    if (phase != 1)
        if (int rc = check_step_fields(A, u, v, w, phi, p, p_old, p_out)) return rc;   // npts of A: nzl + 2 planes each
    if (phase == 0) {
        // The kernel's plane index q and the array's plane index differ by `sh` for the rank at the bottom wall: the
        // wall form of the kernel takes q = 0 for the first plane above the wall and q = g.nz for the wall at the top.
        GridParams g = A->grid;
        const int sh = bottom ? 1 : 0;
        g.wall = (bottom || top) ? 1 : 0;
        g.nz = bottom ? (top ? nzl : nzl + 1) : (top ? nzl + 1 : nzl + 2);
        const long long o = sh * plane;
        if (int rc = enqueue_rhs_g(A, g, u + o, v + o, w + o, phi + o, p + o, p_old + o, dt, dt_ratio, A->rhs + o, A->up + o,
                                   A->vp + o, A->wp + o, st, 1 - sh, nzl + 1 - sh)) return rc;
        if (int rc = check_launch(launch_r2c(A, A->rhs, st, 1, nzl + 1), "fft_x_r2c")) return rc;
        return enqueue_y<MODE_FWD>(A, st, 1, nzl + 1);
    }
    if (phase == 1) return enqueue_z(B, st, nullptr);
    // phase 2: planes 0 .. nzl + 1 of p^(n+1) (the halo planes too, except beyond a wall), then the correction
    const int kb0 = bottom ? 1 : 0, kb1 = top ? nzl + 1 : nzl + 2;
    if (int rc = enqueue_y<MODE_INV>(A, st, kb0, kb1)) return rc;
    if (int rc = check_launch(launch_c2r(A, p_out, sp->norm, st, kb0, kb1), "fft_x_c2r")) return rc;
    GridParams g = A->grid;
    g.wall = top ? 1 : 0;
    g.nz = top ? nzl + 1 : nzl + 2;
    return enqueue_correction_g(A, g, dt, p_out, u, v, w, st, 1, nzl + 1);
}
