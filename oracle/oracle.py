"""ctypes wrapper around liboracle.so -- TEST INFRASTRUCTURE, NOT PRODUCT.

numpy arrays in, numpy arrays out; fields have shape (nz, ny, nx), C-contiguous, float64
(x fastest, matching oracle.h).  Argument marshalling only: all arithmetic is in oracle.c.
"""
import ctypes

import numpy as np

from .build import build as _build

BC_Z_PERIODIC = 0
BC_Z_WALL = 1
BC_PERIODIC, BC_NEUMANN, BC_DIRICHLET = 0, 1, 2

_lib = ctypes.CDLL(_build())
_dp = ctypes.POINTER(ctypes.c_double)
_ci, _cd, _cl = ctypes.c_int, ctypes.c_double, ctypes.c_long

_GRID = [_ci, _ci, _ci, _cd, _cd, _cd, _ci]
_lib.oracle_rhs.argtypes = _GRID + [_cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_poisson.argtypes = _GRID + [_dp, _dp, _dp, _ci]
_lib.oracle_projection_step.argtypes = _GRID + [_cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_rhs_vdt.argtypes = _GRID + [_cd, _cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_projection_step_vdt.argtypes = _GRID + [_cd, _cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_projection_step_paper.argtypes = _GRID + [_cd, _cd, _cd] + [_dp] * 6 + [_ci]
_lib.oracle_correction.argtypes = _GRID + [_cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_correction.restype = _ci
_lib.oracle_dft_axis.argtypes = [_cl, _ci, _cl, _ci, _dp, _dp, _dp, _dp, _ci]
_lib.oracle_divergence.argtypes = _GRID + [_dp] * 4 + [_ci]
_lib.oracle_laplacian.argtypes = _GRID + [_dp] * 2 + [_ci]
_GRID3 = [_ci, _ci, _ci, _cd, _cd, _cd, _ci, _ci, _ci]
_lib.oracle_r2r_axis.argtypes = [_cl, _ci, _cl, _ci, _ci, _dp, _dp, _ci]
_lib.oracle_eigenvalues.argtypes = [_ci, _cd, _ci, _dp]
_lib.oracle_divergence_bc.argtypes = _GRID3 + [_dp] * 4 + [_ci]
_lib.oracle_laplacian_bc.argtypes = _GRID3 + [_dp] * 2 + [_ci]
_lib.oracle_poisson_bc.argtypes = _GRID3 + [_dp, _dp, _dp, _ci]
_lib.oracle_rhs_bc.argtypes = _GRID3 + [_cd, _cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_correction_bc.argtypes = _GRID3 + [_cd, _cd, _cd] + [_dp] * 7 + [_ci]
_lib.oracle_projection_step_bc.argtypes = _GRID3 + [_cd, _cd, _cd, _cd] + [_dp] * 7 + [_ci]
for _f in ("oracle_r2r_axis", "oracle_eigenvalues", "oracle_divergence_bc", "oracle_laplacian_bc", "oracle_poisson_bc",
           "oracle_rhs_bc", "oracle_correction_bc", "oracle_projection_step_bc"):
    getattr(_lib, _f).restype = _ci
_lib.oracle_momentum_prediction.argtypes = [_ci, _ci, _ci, _cd, _cd, _cd] + [_cd] * 10 + [_dp] * 14 + [_ci]
_lib.oracle_momentum_prediction.restype = _ci
_lib.oracle_vof_step.argtypes = [_ci, _ci, _ci, _cd, _cd, _cd, _cd, _cd] + [_dp] * 5 + [_ci]
_lib.oracle_vof_step.restype = _ci
_lib.oracle_vof_reconstruct.argtypes = [_ci, _ci, _ci, _cd, _dp, _dp, _dp, ctypes.POINTER(_ci), _ci]
_lib.oracle_vof_reconstruct.restype = _ci
_lib.oracle_tanh_integral.argtypes = [_cd] * 5
_lib.oracle_tanh_integral.restype = _cd
_lib.oracle_threads.argtypes = [_ci]
for _f in ("oracle_rhs_vdt", "oracle_projection_step_vdt", "oracle_rhs", "oracle_poisson", "oracle_projection_step", "oracle_projection_step_paper",
           "oracle_dft_axis", "oracle_divergence", "oracle_laplacian", "oracle_threads"):
    getattr(_lib, _f).restype = _ci


def _p(a):
    return a.ctypes.data_as(_dp)


def _field(a, shape=None):
    a = np.ascontiguousarray(a, dtype=np.float64)
    if a.ndim != 3 or (shape is not None and a.shape != shape):
        raise ValueError("oracle fields must be float64 arrays of shape (nz, ny, nx)")
    return a


def _grid(shape, box, bc_z):
    nz, ny, nx = shape
    lx, ly, lz = box
    return [nx, ny, nz, float(lx), float(ly), float(lz), int(bc_z)]


def _grid3(shape, box, bc):
    """bc = (bc_x, bc_y, bc_z)"""
    nz, ny, nx = shape
    lx, ly, lz = box
    return [nx, ny, nz, float(lx), float(ly), float(lz), int(bc[0]), int(bc[1]), int(bc[2])]


def _check(rc, name):
    if rc != 0:
        raise RuntimeError(f"{name} failed with code {rc}")


def threads(nthreads=0):
    return _lib.oracle_threads(int(nthreads))


def rhs(u, v, w, phi, p, p_old, box, bc_z, rho1, rho2, dt, nthreads=0, dt_ratio=None):
    """dt_ratio = dt^(n+1)/dt^n selects the variable-time-step p_hat; None = constant dt."""
    u = _field(u)
    f = [_field(a, u.shape) for a in (v, w, phi, p, p_old)]
    out = np.empty_like(u)
    if dt_ratio is None:
        _check(_lib.oracle_rhs(*_grid(u.shape, box, bc_z), rho1, rho2, dt, _p(u), *[_p(a) for a in f],
                               _p(out), nthreads), "oracle_rhs")
    else:
        _check(_lib.oracle_rhs_vdt(*_grid(u.shape, box, bc_z), rho1, rho2, dt, float(dt_ratio), _p(u),
                                   *[_p(a) for a in f], _p(out), nthreads), "oracle_rhs_vdt")
    return out


def poisson(rhs_field, box, bc_z, nthreads=0, return_imag_residue=False):
    r = _field(rhs_field)
    out = np.empty_like(r)
    res = ctypes.c_double(0.0)
    _check(_lib.oracle_poisson(*_grid(r.shape, box, bc_z), _p(r), _p(out), ctypes.byref(res), nthreads),
           "oracle_poisson")
    return (out, res.value) if return_imag_residue else out


def projection_step(u, v, w, phi, p, p_old, box, bc_z, rho1, rho2, dt, nthreads=0, return_rhs=False,
                    dt_ratio=None):
    """Returns new (u, v, w, p) [and rhs]; inputs are not modified.  dt_ratio as in rhs()."""
    u = _field(u).copy()
    v, w, p = (_field(a, u.shape).copy() for a in (v, w, p))
    phi, p_old = _field(phi, u.shape), _field(p_old, u.shape)
    r = np.empty_like(u) if return_rhs else None
    if dt_ratio is None:
        _check(_lib.oracle_projection_step(*_grid(u.shape, box, bc_z), rho1, rho2, dt, _p(u), _p(v), _p(w),
                                           _p(phi), _p(p), _p(p_old), _p(r) if return_rhs else None,
                                           nthreads), "oracle_projection_step")
    else:
        _check(_lib.oracle_projection_step_vdt(*_grid(u.shape, box, bc_z), rho1, rho2, dt, float(dt_ratio),
                                               _p(u), _p(v), _p(w), _p(phi), _p(p), _p(p_old),
                                               _p(r) if return_rhs else None, nthreads),
               "oracle_projection_step_vdt")
    return (u, v, w, p, r) if return_rhs else (u, v, w, p)


def correction(u, v, w, phi, p, p_old, p_new, box, bc_z, rho1, rho2, dt, nthreads=0):
    """Returns corrected (u, v, w) given p_new; inputs are not modified."""
    u = _field(u).copy()
    v, w = (_field(a, u.shape).copy() for a in (v, w))
    phi, p, p_old, p_new = (_field(a, u.shape) for a in (phi, p, p_old, p_new))
    _check(_lib.oracle_correction(*_grid(u.shape, box, bc_z), rho1, rho2, dt, _p(u), _p(v), _p(w), _p(phi),
                                  _p(p), _p(p_old), _p(p_new), nthreads), "oracle_correction")
    return u, v, w


def projection_step_paper(u, v, w, phi, p, p_old, box, bc_z, rho1, rho2, dt, nthreads=0):
    u = _field(u).copy()
    v, w, p = (_field(a, u.shape).copy() for a in (v, w, p))
    phi, p_old = _field(phi, u.shape), _field(p_old, u.shape)
    _check(_lib.oracle_projection_step_paper(*_grid(u.shape, box, bc_z), rho1, rho2, dt, _p(u), _p(v),
                                             _p(w), _p(phi), _p(p), _p(p_old), nthreads),
           "oracle_projection_step_paper")
    return u, v, w, p


def dft_axis(x, axis, sign, nthreads=0):
    """Naive, unnormalised DFT of a complex array along one axis (sign=-1 forward, +1 inverse)."""
    x = np.asarray(x)
    n = x.shape[axis]
    n_outer = int(np.prod(x.shape[:axis], dtype=np.int64))
    n_inner = int(np.prod(x.shape[axis + 1:], dtype=np.int64))
    re = np.ascontiguousarray(x.real, dtype=np.float64)
    im = np.ascontiguousarray(x.imag, dtype=np.float64) if np.iscomplexobj(x) else np.zeros_like(re)
    o_re, o_im = np.empty_like(re), np.empty_like(re)
    _check(_lib.oracle_dft_axis(n_outer, n, n_inner, sign, _p(re), _p(im), _p(o_re), _p(o_im), nthreads),
           "oracle_dft_axis")
    return o_re + 1j * o_im


def divergence(u, v, w, box, bc_z, nthreads=0):
    u = _field(u)
    v, w = _field(v, u.shape), _field(w, u.shape)
    out = np.empty_like(u)
    _check(_lib.oracle_divergence(*_grid(u.shape, box, bc_z), _p(u), _p(v), _p(w), _p(out), nthreads),
           "oracle_divergence")
    return out


def laplacian(p, box, bc_z, nthreads=0):
    p = _field(p)
    out = np.empty_like(p)
    _check(_lib.oracle_laplacian(*_grid(p.shape, box, bc_z), _p(p), _p(out), nthreads), "oracle_laplacian")
    return out


# ---------------------------------------------------------------- non-periodic x / y (bc = (bc_x, bc_y, bc_z))

def r2r_axis(x, axis, bc, sign, nthreads=0):
    """naive cosine (bc = 1) / sine (bc = 2) eigen-expansion of a real array along one axis; sign = -1 analysis
    (normalised coefficients), +1 synthesis"""
    x = np.ascontiguousarray(x, dtype=np.float64)
    n = x.shape[axis]
    n_outer = int(np.prod(x.shape[:axis], dtype=np.int64))
    n_inner = int(np.prod(x.shape[axis + 1:], dtype=np.int64))
    out = np.empty_like(x)
    _check(_lib.oracle_r2r_axis(n_outer, n, n_inner, int(bc), int(sign), _p(x), _p(out), nthreads), "oracle_r2r_axis")
    return out


def eigenvalues(n, d, bc):
    out = np.empty(n)
    _check(_lib.oracle_eigenvalues(int(n), float(d), int(bc), _p(out)), "oracle_eigenvalues")
    return out


def divergence_bc(u, v, w, box, bc, nthreads=0):
    u = _field(u)
    v, w = _field(v, u.shape), _field(w, u.shape)
    out = np.empty_like(u)
    _check(_lib.oracle_divergence_bc(*_grid3(u.shape, box, bc), _p(u), _p(v), _p(w), _p(out), nthreads), "oracle_divergence_bc")
    return out


def laplacian_bc(p, box, bc, nthreads=0):
    p = _field(p)
    out = np.empty_like(p)
    _check(_lib.oracle_laplacian_bc(*_grid3(p.shape, box, bc), _p(p), _p(out), nthreads), "oracle_laplacian_bc")
    return out


def poisson_bc(rhs_field, box, bc, nthreads=0, return_imag_residue=False):
    r = _field(rhs_field)
    out = np.empty_like(r)
    res = ctypes.c_double(0.0)
    _check(_lib.oracle_poisson_bc(*_grid3(r.shape, box, bc), _p(r), _p(out), ctypes.byref(res), nthreads), "oracle_poisson_bc")
    return (out, res.value) if return_imag_residue else out


def rhs_bc(u, v, w, phi, p, p_old, box, bc, rho1, rho2, dt, nthreads=0, dt_ratio=1.0):
    u = _field(u)
    f = [_field(a, u.shape) for a in (v, w, phi, p, p_old)]
    out = np.empty_like(u)
    _check(_lib.oracle_rhs_bc(*_grid3(u.shape, box, bc), rho1, rho2, dt, float(dt_ratio), _p(u), *[_p(a) for a in f],
                              _p(out), nthreads), "oracle_rhs_bc")
    return out


def correction_bc(u, v, w, phi, p, p_old, p_new, box, bc, rho1, rho2, dt, nthreads=0):
    u = _field(u).copy()
    v, w = (_field(a, u.shape).copy() for a in (v, w))
    phi, p, p_old, p_new = (_field(a, u.shape) for a in (phi, p, p_old, p_new))
    _check(_lib.oracle_correction_bc(*_grid3(u.shape, box, bc), rho1, rho2, dt, _p(u), _p(v), _p(w), _p(phi),
                                     _p(p), _p(p_old), _p(p_new), nthreads), "oracle_correction_bc")
    return u, v, w


def projection_step_bc(u, v, w, phi, p, p_old, box, bc, rho1, rho2, dt, nthreads=0, return_rhs=False, dt_ratio=1.0):
    """the step with walls along any direction: bc = (bc_x, bc_y, bc_z), each PERIODIC or NEUMANN"""
    u = _field(u).copy()
    v, w, p = (_field(a, u.shape).copy() for a in (v, w, p))
    phi, p_old = _field(phi, u.shape), _field(p_old, u.shape)
    r = np.empty_like(u) if return_rhs else None
    _check(_lib.oracle_projection_step_bc(*_grid3(u.shape, box, bc), rho1, rho2, dt, float(dt_ratio), _p(u), _p(v), _p(w),
                                          _p(phi), _p(p), _p(p_old), _p(r) if return_rhs else None, nthreads),
           "oracle_projection_step_bc")
    return (u, v, w, p, r) if return_rhs else (u, v, w, p)


def momentum_prediction(u, v, w, phi, kappa, m_old, box, rho1, rho2, mu1, mu2, sigma, grav, dt, dt_ratio=1.0, nthreads=0):
    """eq. (15), triply periodic.  m_old = (Mu, Mv, Mw) of the previous step; kappa may be None.
    Returns (u**, v**, w**), (Mu, Mv, Mw) of this step."""
    u = _field(u)
    v, w, phi = (_field(a, u.shape) for a in (v, w, phi))
    mo = [_field(a, u.shape) for a in m_old]
    kap = None if kappa is None else _field(kappa, u.shape)
    out = [np.empty_like(u) for _ in range(6)]
    nz, ny, nx = u.shape
    _check(_lib.oracle_momentum_prediction(nx, ny, nz, float(box[0]), float(box[1]), float(box[2]), rho1, rho2, mu1, mu2,
                                           sigma, float(grav[0]), float(grav[1]), float(grav[2]), dt, float(dt_ratio),
                                           _p(u), _p(v), _p(w), _p(phi), None if kap is None else _p(kap),
                                           *[_p(a) for a in mo], *[_p(a) for a in out], nthreads),
           "oracle_momentum_prediction")
    return tuple(out[:3]), tuple(out[3:])


def vof_step(phi, u, v, w, box, beta, dt, nthreads=0):
    """one MTHINC step (x -> y -> z), triply periodic; returns phi^(n+1)"""
    phi = _field(phi)
    u, v, w = (_field(a, phi.shape) for a in (u, v, w))
    out = np.empty_like(phi)
    nz, ny, nx = phi.shape
    _check(_lib.oracle_vof_step(nx, ny, nz, float(box[0]), float(box[1]), float(box[2]), float(beta), float(dt),
                                _p(phi), _p(u), _p(v), _p(w), _p(out), nthreads), "oracle_vof_step")
    return out


def tanh_integral(a, b, alpha, gamma, beta):
    """int_a^b 1/2 [1 + tanh(beta (alpha x + gamma))] dx"""
    return _lib.oracle_tanh_integral(float(a), float(b), float(alpha), float(gamma), float(beta))


def vof_reconstruct(phi, beta, nthreads=0):
    """per cell: unit normal (nz, ny, nx, 3), offset d, flat flag"""
    phi = _field(phi)
    nz, ny, nx = phi.shape
    n = np.empty(phi.shape + (3,))
    d = np.empty_like(phi)
    flat = np.empty(phi.shape, dtype=np.int32)
    _check(_lib.oracle_vof_reconstruct(nx, ny, nz, float(beta), _p(phi), _p(n), _p(d),
                                       flat.ctypes.data_as(ctypes.POINTER(_ci)), nthreads), "oracle_vof_reconstruct")
    return n, d, flat
