"""Thin ctypes binding of libflutas_b200.so (include/flutas.h): argument marshalling only.

Every step of the path runs in the library's CUDA kernels; torch is used for device memory and
streams.  Importing this module fails loudly if the library cannot be built or loaded: there is
no CPU fallback.
"""
import ctypes

from .build import build as _build

BC_Z_PERIODIC = 0
BC_Z_WALL = 1
BC_PERIODIC = 0
BC_NEUMANN = 1
BC_DIRICHLET = 2
PLAN_CALLER_WORKSPACE = 1

_vp, _ci, _cd = ctypes.c_void_p, ctypes.c_int, ctypes.c_double
lib = ctypes.CDLL(_build())

lib.flutas_plan_create.argtypes = [_ci, _ci, _ci, _cd, _cd, _cd, _ci, _cd, _cd]
lib.flutas_plan_create.restype = _vp
lib.flutas_plan_create_ex.argtypes = [_ci, _ci, _ci, _cd, _cd, _cd, _ci, _ci, _ci, _cd, _cd, ctypes.c_uint]
lib.flutas_plan_create_ex.restype = _vp
lib.flutas_workspace_bytes.argtypes = [_ci] * 6
lib.flutas_workspace_bytes.restype = ctypes.c_size_t
lib.flutas_plan_set_workspace.argtypes = [_vp, _vp, ctypes.c_size_t]
lib.flutas_plan_set_workspace.restype = _ci
lib.flutas_plan_kernel_symbol.argtypes = [_vp, _ci]
lib.flutas_plan_kernel_symbol.restype = ctypes.c_char_p
lib.flutas_time_step.argtypes = [_vp] * 15 + [_cd] * 8 + [_vp]
lib.flutas_time_step.restype = _ci
lib.flutas_momentum_rhs.argtypes = [_vp] * 14 + [_cd] * 8 + [_vp] * 5
lib.flutas_momentum_rhs.restype = _ci
lib.flutas_vof_step.argtypes = [_vp] * 6 + [_cd, _cd, _vp]
lib.flutas_vof_step.restype = _ci
lib.flutas_vof_step_noalloc.argtypes = [_ci] * 3 + [_cd] * 3 + [_vp] * 5 + [_cd, _cd, _vp]
lib.flutas_vof_step_noalloc.restype = _ci
lib.flutas_vof_step_noalloc_max_cells.argtypes = []
lib.flutas_vof_step_noalloc_max_cells.restype = ctypes.c_size_t
lib.flutas_plan_destroy.argtypes = [_vp]
lib.flutas_plan_destroy.restype = None
lib.flutas_projection_step.argtypes = [_vp] * 7 + [_cd, _vp]
lib.flutas_projection_step.restype = _ci
lib.flutas_projection_step_ex.argtypes = [_vp] * 8 + [_cd, _cd, _vp]
lib.flutas_projection_step_ex.restype = _ci
lib.flutas_splitting_rhs_ex.argtypes = [_vp] * 7 + [_cd, _cd, _vp, _vp]
lib.flutas_splitting_rhs_ex.restype = _ci
lib.flutas_projection_step_host.argtypes = [_vp] * 7 + [_cd, _vp]
lib.flutas_projection_step_host.restype = _ci
lib.flutas_splitting_rhs.argtypes = [_vp] * 7 + [_cd, _vp, _vp]
lib.flutas_splitting_rhs.restype = _ci
lib.flutas_poisson_solve.argtypes = [_vp, _vp, _vp, _vp]
lib.flutas_poisson_solve.restype = _ci
lib.flutas_last_error.argtypes = []
lib.flutas_last_error.restype = ctypes.c_char_p
lib.flutas_last_error_code.argtypes = []
lib.flutas_last_error_code.restype = _ci
lib.flutas_plan_workspace_bytes.argtypes = [_vp]
lib.flutas_plan_workspace_bytes.restype = ctypes.c_size_t
lib.flutas_plan_kernel_launches.argtypes = [_vp]
lib.flutas_plan_kernel_launches.restype = _ci
lib.flutas_plan_kernel_name.argtypes = [_vp, _ci]
lib.flutas_plan_kernel_name.restype = ctypes.c_char_p
lib.flutas_plan_kernel_bytes.argtypes = [_vp, _ci]
lib.flutas_plan_kernel_bytes.restype = _cd
lib.flutas_plan_set_timing.argtypes = [_vp, _ci]
lib.flutas_plan_set_timing.restype = _ci
lib.flutas_plan_read_timing.argtypes = [_vp, ctypes.POINTER(ctypes.c_float), _ci, ctypes.POINTER(_ci)]
lib.flutas_plan_read_timing.restype = _ci
lib.flutas_plan_set_option.argtypes = [_vp, ctypes.c_char_p, _ci]
lib.flutas_plan_set_option.restype = _ci

lib.flutas_slab_plan_create.argtypes = [_ci, _ci, _ci, _cd, _cd, _cd, _ci, _cd, _cd, _ci, _ci]
lib.flutas_slab_plan_create.restype = _vp
lib.flutas_slab_workspace_bytes.argtypes = [_ci] * 5
lib.flutas_slab_workspace_bytes.restype = ctypes.c_size_t
lib.flutas_slab_exchange_bytes.argtypes = [_ci] * 5
lib.flutas_slab_exchange_bytes.restype = ctypes.c_size_t
lib.flutas_slab_plan_attach.argtypes = [_vp, _vp, ctypes.c_size_t, ctypes.POINTER(_vp), ctypes.c_size_t]
lib.flutas_slab_plan_attach.restype = _ci
lib.flutas_slab_step_phase.argtypes = [_vp, _ci] + [_vp] * 7 + [_cd, _cd, _vp]
lib.flutas_slab_step_phase.restype = _ci
lib.flutas_slab_plan_destroy.argtypes = [_vp]
lib.flutas_slab_plan_destroy.restype = None

EXPORTS = [
    "flutas_plan_create", "flutas_projection_step", "flutas_projection_step_host", "flutas_plan_destroy",
    "flutas_splitting_rhs", "flutas_poisson_solve", "flutas_last_error", "flutas_last_error_code",
    "flutas_plan_workspace_bytes", "flutas_plan_kernel_launches", "flutas_plan_kernel_name",
    "flutas_plan_set_timing", "flutas_plan_read_timing", "flutas_plan_kernel_bytes", "flutas_plan_set_option",
    "flutas_projection_step_ex", "flutas_splitting_rhs_ex",
    "flutas_plan_create_ex", "flutas_workspace_bytes", "flutas_plan_set_workspace", "flutas_plan_kernel_symbol",
    "flutas_time_step", "flutas_momentum_rhs", "flutas_vof_step", "flutas_vof_step_noalloc",
    "flutas_vof_step_noalloc_max_cells",
    "flutas_slab_plan_create", "flutas_slab_workspace_bytes", "flutas_slab_exchange_bytes", "flutas_slab_plan_attach",
    "flutas_slab_step_phase", "flutas_slab_plan_destroy",
]


class FlutasError(RuntimeError):
    def __init__(self, code, message):
        super().__init__(f"flutas error {code}: {message}")
        self.code = code


def _raise_last():
    raise FlutasError(lib.flutas_last_error_code(), lib.flutas_last_error().decode())


def _check(rc):
    if rc != 0:
        raise FlutasError(rc, lib.flutas_last_error().decode())


def _dev_ptr(t, npts):
    import torch
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == torch.float64 and t.is_contiguous()
            and t.numel() == npts):
        raise ValueError("expected a contiguous float64 CUDA tensor with nx*ny*nz elements")
    return t.data_ptr()


def _stream():
    import torch
    return torch.cuda.current_stream().cuda_stream


def workspace_bytes(nx, ny, nz, bc_z, bc_x=BC_PERIODIC, bc_y=BC_PERIODIC):
    """flutas_workspace_bytes: what a plan for this grid needs (0 = unsupported grid); no device needed"""
    return lib.flutas_workspace_bytes(int(nx), int(ny), int(nz), int(bc_x), int(bc_y), int(bc_z))


def vof_step_noalloc(shape, box, phi, u, v, w, phi_out, beta, dt, stream=None):
    """flutas_vof_step_noalloc: one MTHINC step without a plan and without any allocation by the library (for callers that
    may not call cudaMalloc; the scratch is a static array in the library, hence shape = (nx, ny, nz) with
    nx*ny*nz <= vof_noalloc_max_cells()).  One array per GPU is shared by all calls: keep them ordered on the device."""
    nx, ny, nz = (int(n) for n in shape)
    ptrs = [_dev_ptr(t, nx * ny * nz) for t in (phi, u, v, w, phi_out)]
    _check(lib.flutas_vof_step_noalloc(nx, ny, nz, float(box[0]), float(box[1]), float(box[2]), *ptrs, float(beta), float(dt),
                                       _stream() if stream is None else stream))


def vof_noalloc_max_cells():
    return lib.flutas_vof_step_noalloc_max_cells()


class Plan:
    """flutas_plan_create / flutas_projection_step / flutas_plan_destroy with the same argument order.

    workspace="torch" (default): the plan is created with FLUTAS_PLAN_CALLER_WORKSPACE and handed one uint8 torch
    tensor (flutas_plan_set_workspace), so that every large device byte goes through torch's allocator;
    workspace="library": flutas_plan_create allocates it with cudaMalloc (what a C caller of the three north-star
    calls gets); workspace=<uint8 CUDA tensor>: that buffer."""

    def __init__(self, nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, bc_x=BC_PERIODIC, bc_y=BC_PERIODIC, workspace="torch"):
        self._h = None
        self._ws = None
        args = (int(nx), int(ny), int(nz), float(lx), float(ly), float(lz))
        if isinstance(workspace, str) and workspace == "library":
            if bc_x == BC_PERIODIC and bc_y == BC_PERIODIC:
                h = lib.flutas_plan_create(*args, int(bc_z), float(rho1), float(rho2))
            else:
                h = lib.flutas_plan_create_ex(*args, int(bc_x), int(bc_y), int(bc_z), float(rho1), float(rho2), 0)
        else:
            h = lib.flutas_plan_create_ex(*args, int(bc_x), int(bc_y), int(bc_z), float(rho1), float(rho2),
                                          PLAN_CALLER_WORKSPACE)
        if not h:
            _raise_last()
        self._h = h
        self.nx, self.ny, self.nz, self.bc_z = int(nx), int(ny), int(nz), int(bc_z)
        self.npts = self.nx * self.ny * self.nz
        if not (isinstance(workspace, str) and workspace == "library"):
            import torch
            ws = torch.empty(self.workspace_bytes, dtype=torch.uint8, device="cuda") if isinstance(workspace, str) else workspace
            self.set_workspace(ws)

    def set_workspace(self, ws):
        """ws: a contiguous uint8 CUDA tensor of at least workspace_bytes (kept alive by the plan), or None = library-owned"""
        if ws is None:
            _check(lib.flutas_plan_set_workspace(self._h, None, 0))
        else:
            _check(lib.flutas_plan_set_workspace(self._h, ws.data_ptr(), ws.numel() * ws.element_size()))
        self._ws = ws

    def destroy(self):
        if self._h:
            lib.flutas_plan_destroy(self._h)
            self._h = None
            self._ws = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass

    # --- the step (device tensors, in place on u, v, w, p)
    def projection_step(self, u, v, w, phi, p, p_old, dt, stream=None):
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi, p, p_old)]
        _check(lib.flutas_projection_step(self._h, *ptrs, float(dt), _stream() if stream is None else stream))

    # --- time-stepping form: variable dt (dt_ratio = dt_new / dt_old) and p_out = p | p_old | a seventh tensor
    def projection_step_ex(self, u, v, w, phi, p, p_old, p_out, dt, dt_ratio=1.0, stream=None):
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi, p, p_old, p_out)]
        _check(lib.flutas_projection_step_ex(self._h, *ptrs, float(dt), float(dt_ratio),
                                             _stream() if stream is None else stream))

    def splitting_rhs_ex(self, u, v, w, phi, p, p_old, dt, dt_ratio, rhs_out, stream=None):
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi, p, p_old)]
        _check(lib.flutas_splitting_rhs_ex(self._h, *ptrs, float(dt), float(dt_ratio),
                                           _dev_ptr(rhs_out, self.npts), _stream() if stream is None else stream))

    # --- momentum prediction (eq. 15) fused with the projection: one velocity / pressure update
    def time_step(self, u, v, w, phi, kappa, p, p_old, p_out, m_old, m_new, mu1, mu2, sigma, grav, dt, dt_ratio=1.0, stream=None):
        """u, v, w in place; m_old / m_new: 3-tuples of tensors (M of the previous / this step); kappa may be None"""
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi)] + [None if kappa is None else _dev_ptr(kappa, self.npts)]
        ptrs += [_dev_ptr(t, self.npts) for t in (p, p_old, p_out, *m_old, *m_new)]
        _check(lib.flutas_time_step(self._h, *ptrs, float(mu1), float(mu2), float(sigma), float(grav[0]), float(grav[1]),
                                    float(grav[2]), float(dt), float(dt_ratio), _stream() if stream is None else stream))

    def momentum_rhs(self, u, v, w, phi, kappa, p, p_old, m_old, m_new, mu1, mu2, sigma, grav, dt, dt_ratio, us, vs, ws, rhs,
                     stream=None):
        """the first kernel of time_step alone; p = p_old = None gives u** without the splitting terms"""
        opt = lambda t: None if t is None else _dev_ptr(t, self.npts)
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi)] + [opt(kappa), opt(p), opt(p_old)]
        ptrs += [_dev_ptr(t, self.npts) for t in (*m_old, *m_new)]
        outs = [_dev_ptr(t, self.npts) for t in (us, vs, ws, rhs)]
        _check(lib.flutas_momentum_rhs(self._h, *ptrs, float(mu1), float(mu2), float(sigma), float(grav[0]), float(grav[1]),
                                       float(grav[2]), float(dt), float(dt_ratio), *outs, _stream() if stream is None else stream))

    # --- one MTHINC volume-of-fluid step (phi_out may be phi)
    def vof_step(self, phi, u, v, w, phi_out, beta, dt, stream=None):
        ptrs = [_dev_ptr(t, self.npts) for t in (phi, u, v, w, phi_out)]
        _check(lib.flutas_vof_step(self._h, *ptrs, float(beta), float(dt), _stream() if stream is None else stream))

    # --- the step for host arrays (numpy float64 or pinned torch CPU tensors), in place, synchronous
    def projection_step_host(self, u, v, w, phi, p, p_old, dt, stream=None):
        ptrs = [_host_ptr(a, self.npts) for a in (u, v, w, phi, p, p_old)]
        _check(lib.flutas_projection_step_host(self._h, *ptrs, float(dt), _stream() if stream is None else stream))

    def splitting_rhs(self, u, v, w, phi, p, p_old, dt, rhs_out, stream=None):
        ptrs = [_dev_ptr(t, self.npts) for t in (u, v, w, phi, p, p_old)]
        _check(lib.flutas_splitting_rhs(self._h, *ptrs, float(dt), _dev_ptr(rhs_out, self.npts),
                                        _stream() if stream is None else stream))

    def poisson_solve(self, rhs, p_out, stream=None):
        _check(lib.flutas_poisson_solve(self._h, _dev_ptr(rhs, self.npts), _dev_ptr(p_out, self.npts),
                                        _stream() if stream is None else stream))

    # --- introspection
    @property
    def workspace_bytes(self):
        return lib.flutas_plan_workspace_bytes(self._h)

    @property
    def kernel_names(self):
        n = lib.flutas_plan_kernel_launches(self._h)
        return [lib.flutas_plan_kernel_name(self._h, i).decode() for i in range(n)]

    @property
    def kernel_symbols(self):
        n = lib.flutas_plan_kernel_launches(self._h)
        return [lib.flutas_plan_kernel_symbol(self._h, i).decode() for i in range(n)]

    @property
    def kernel_bytes(self):
        n = lib.flutas_plan_kernel_launches(self._h)
        return [lib.flutas_plan_kernel_bytes(self._h, i) for i in range(n)]

    def set_timing(self, enabled):
        _check(lib.flutas_plan_set_timing(self._h, 1 if enabled else 0))

    def read_timing(self):
        """returns (list of total ms per kernel, number of steps covered)"""
        n = lib.flutas_plan_kernel_launches(self._h)
        ms = (ctypes.c_float * n)()
        steps = _ci(0)
        _check(lib.flutas_plan_read_timing(self._h, ms, n, ctypes.byref(steps)))
        return list(ms), steps.value

    def set_option(self, name, value):
        _check(lib.flutas_plan_set_option(self._h, name.encode(), int(value)))


class SlabPlan:
    """flutas_slab_plan_create / _attach / _step_phase / _destroy for ONE rank of a z-slab decomposition (include/flutas.h).
    Fields are local tensors of (nz / n_ranks + 2) * ny * nx doubles (one halo plane below and above the slab).
    `exchange_ptrs`: the device addresses of every rank's exchange buffer as this process sees them (entry `rank` is the
    own one); slab.py builds them for ranks that share a process and for torchrun ranks (symmetric memory)."""

    def __init__(self, nx, ny, nz, lx, ly, lz, bc_z, rho1, rho2, n_ranks, rank):
        self._h = None
        h = lib.flutas_slab_plan_create(int(nx), int(ny), int(nz), float(lx), float(ly), float(lz), int(bc_z), float(rho1),
                                        float(rho2), int(n_ranks), int(rank))
        if not h:
            _raise_last()
        self._h = h
        self.nx, self.ny, self.nz, self.bc_z, self.n_ranks, self.rank = int(nx), int(ny), int(nz), int(bc_z), int(n_ranks), int(rank)
        self.nzl = self.nz // self.n_ranks
        self.npts_local = self.nx * self.ny * (self.nzl + 2)
        self.workspace_bytes = lib.flutas_slab_workspace_bytes(self.nx, self.ny, self.nz, self.bc_z, self.n_ranks)
        self.exchange_bytes = lib.flutas_slab_exchange_bytes(self.nx, self.ny, self.nz, self.bc_z, self.n_ranks)
        self._keep = None

    def attach(self, workspace, exchange_ptrs, keep=None):
        """workspace: uint8 CUDA tensor of workspace_bytes; exchange_ptrs: n_ranks ints; keep: objects to keep alive"""
        arr = (_vp * self.n_ranks)(*[int(q) for q in exchange_ptrs])
        _check(lib.flutas_slab_plan_attach(self._h, workspace.data_ptr(), workspace.numel(), arr, self.exchange_bytes))
        self._keep = (workspace, keep)

    def step_phase(self, phase, u, v, w, phi, p, p_old, p_out, dt, dt_ratio=1.0, stream=None):
        if phase == 1:
            ptrs = [None] * 7
        else:
            ptrs = [_dev_ptr(t, self.npts_local) for t in (u, v, w, phi, p, p_old, p_out)]
        _check(lib.flutas_slab_step_phase(self._h, int(phase), *ptrs, float(dt), float(dt_ratio),
                                          _stream() if stream is None else stream))

    def destroy(self):
        if self._h:
            lib.flutas_slab_plan_destroy(self._h)
            self._h = None
            self._keep = None

    def __del__(self):
        try:
            self.destroy()
        except Exception:
            pass


def _host_ptr(a, npts):
    import numpy as np
    try:
        import torch
        if isinstance(a, torch.Tensor):
            if a.is_cuda or a.dtype != torch.float64 or not a.is_contiguous() or a.numel() != npts:
                raise ValueError("expected a contiguous float64 CPU tensor with nx*ny*nz elements")
            return a.data_ptr()
    except ImportError:
        pass
    if not (isinstance(a, np.ndarray) and a.dtype == np.float64 and a.flags["C_CONTIGUOUS"] and a.size == npts):
        raise ValueError("expected a C-contiguous float64 numpy array with nx*ny*nz elements")
    return a.ctypes.data
