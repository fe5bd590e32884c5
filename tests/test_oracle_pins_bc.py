"""Pins for the oracle's non-periodic x / y path (oracle *_bc functions; PAPER.md:61, 163,
167, 287).  As in test_oracle_pins.py, everything is checked against what the mathematics fixes, never against the
CUDA path:
  B0  the naive cosine / sine expansions against closed forms (a single eigenvector), against scipy's DCT-II / DST-II
      (a library routine they reduce to) and analysis-synthesis round trips
  B1  exact eigenpairs of the 7-point Laplacian for every combination of periodic / Neumann / Dirichlet directions
  B2  dense direct solve (bordered when there is a null space) on tiny grids for all 27 combinations
  B3  operators against independent numpy statements
  B4  the step with walls: div-free, residual, gauge, wall faces untouched, fixed point, and all-periodic x, y == the
      original entry points bit for bit
"""
import itertools

import numpy as np
import pytest
import scipy.fft as sfft

import workloads as wl
from tests import np_ops as ops

P, N, D = 0, 1, 2


def _mode(n, m, bc, phase=0.4):
    i = np.arange(n)
    if bc == P:
        return np.cos(2 * np.pi * m * i / n + phase)
    if bc == N:
        return np.cos(np.pi * m * (2 * i + 1) / (2 * n))
    return np.sin(np.pi * (m + 1) * (2 * i + 1) / (2 * n))


def _lam(n, m, d, bc):
    f = {P: 2.0 * m, N: float(m), D: m + 1.0}[bc]
    return -2.0 * (1.0 - np.cos(np.pi * f / n)) / d ** 2


# ----------------------------------------------------------------------------- B0
@pytest.mark.parametrize("n", [2, 3, 8, 13])
@pytest.mark.parametrize("bc", [N, D])
def test_b0_expansions_closed_forms_and_scipy(oracle_mod, n, bc):
    rng = np.random.default_rng(n + bc)
    # a single eigenvector analyses to a unit coefficient (orthogonality + the norms n and n/2)
    for m in range(n):
        x = np.tile(_mode(n, m, bc)[None, :, None], (2, 1, 3))
        c = oracle_mod.r2r_axis(x, 1, bc, -1)
        want = np.zeros(n); want[m] = 1.0
        assert np.allclose(c[1, :, 2], want, atol=1e-13)
    x = rng.standard_normal((3, n, 4))
    c = oracle_mod.r2r_axis(x, 1, bc, -1)
    # scipy's unnormalised DCT-II / DST-II: X_m = 2 sum_i x_i cos / sin(...) = 2 |e_m|^2 c_m
    X = sfft.dct(x, type=2, axis=1) if bc == N else sfft.dst(x, type=2, axis=1)
    norm2 = np.full(n, n / 2.0)
    norm2[0 if bc == N else n - 1] = n
    assert ops.rel_l2(c, X / (2.0 * norm2[None, :, None])) < 1e-14
    # synthesis inverts analysis, on every axis
    for ax in range(3):
        y = rng.standard_normal((n, n, n))
        assert ops.rel_l2(oracle_mod.r2r_axis(oracle_mod.r2r_axis(y, ax, bc, -1), ax, bc, +1), y) < 1e-13
    # eigenvalue table: applying the second difference (ghost = +-interior) to mode m scales it by lam_m
    d = 0.37
    lam = oracle_mod.eigenvalues(n, d, bc)
    for m in range(n):
        e = _mode(n, m, bc)
        ghost = e if bc == N else -e
        ext = np.concatenate(([ghost[0]], e, [ghost[-1]]))
        assert np.allclose((ext[:-2] - 2 * ext[1:-1] + ext[2:]) / d ** 2, lam[m] * e, atol=1e-11 / d ** 2)
        assert np.isclose(lam[m], _lam(n, m, d, bc), rtol=1e-14, atol=1e-300)


# ----------------------------------------------------------------------------- B1
@pytest.mark.parametrize("bc", list(itertools.product((P, N, D), repeat=3)))
def test_b1_eigenpairs_every_combination(oracle_mod, bc):
    shape, box = (6, 8, 10), (1.3, 0.9, 0.7)
    nz, ny, nx = shape
    dx, dy, dz = ops.spacings(shape, box)
    for (a, b, c) in ((1, 2, 1), (0, 0, 2), (3, 0, 0), (2, 3, 4)):
        f = _mode(nz, c, bc[2], 0.7)[:, None, None] * _mode(ny, b, bc[1], 1.1)[None, :, None] * _mode(nx, a, bc[0], 0.3)[None, None, :]
        lam = _lam(nx, a, dx, bc[0]) + _lam(ny, b, dy, bc[1]) + _lam(nz, c, dz, bc[2])
        assert np.linalg.norm(oracle_mod.laplacian_bc(f, box, bc) - lam * f) < 1e-11 * np.linalg.norm(lam * f)
        got, imag = oracle_mod.poisson_bc(lam * f, box, bc, return_imag_residue=True)
        assert ops.rel_l2(got, f) < 1e-12 and imag < 1e-13


# ----------------------------------------------------------------------------- B2
def _dense(shape, box, bc):
    n = int(np.prod(shape))
    L = np.empty((n, n))
    e = np.zeros(n)
    for q in range(n):
        e[q] = 1.0
        L[:, q] = ops.lap_bc(e.reshape(shape), box, bc).ravel()
        e[q] = 0.0
    return L


@pytest.mark.parametrize("bc", list(itertools.product((P, N, D), repeat=3)))
def test_b2_dense_direct_solve_every_combination(oracle_mod, bc):
    shape, box = (5, 6, 8), (1.0, 1.5, 0.8)
    rng = np.random.default_rng(3 + 9 * bc[0] + 3 * bc[1] + bc[2])
    rhs = rng.standard_normal(shape)
    n = rhs.size
    L = _dense(shape, box, bc)
    assert np.allclose(L, L.T, atol=1e-9)
    p = oracle_mod.poisson_bc(rhs - rhs.mean() if D not in bc else rhs, box, bc)
    if D in bc:                                   # non-singular: plain LU
        sol = np.linalg.solve(L, rhs.ravel())
    else:                                         # null space of constants: bordered system, zero-mean gauge (R5)
        assert np.allclose(L.sum(axis=1), 0.0, atol=1e-9)
        K = np.zeros((n + 1, n + 1))
        K[:n, :n] = L
        K[:n, n] = 1.0
        K[n, :n] = 1.0
        sol = np.linalg.solve(K, np.append((rhs - rhs.mean()).ravel(), 0.0))
        assert abs(sol[n]) < 1e-10
        sol = sol[:n]
    assert ops.rel_l2(p.ravel(), sol) < 1e-12


# ----------------------------------------------------------------------------- B3
@pytest.mark.parametrize("bc", [(N, N, N), (P, N, N), (N, P, P), (D, D, N), (D, N, P), (P, D, D)])
def test_b3_operators_match_independent_numpy(oracle_mod, bc):
    rng = np.random.default_rng(17)
    shape, box = (5, 6, 8), (1.3, 0.7, 2.1)
    a, b, c, f = (rng.standard_normal(shape) for _ in range(4))
    assert ops.rel_l2(oracle_mod.laplacian_bc(f, box, bc), ops.lap_bc(f, box, bc)) < 1e-13
    if D not in bc:
        assert ops.rel_l2(oracle_mod.divergence_bc(a, b, c, box, bc), ops.div_bc(a, b, c, box, bc)) < 1e-14


# ----------------------------------------------------------------------------- B4
def _walled_case(nx, ny, nz, bc, ratio, seed):
    W = wl.random_case(nx, ny, nz, bc[2], ratio, seed, box=(2.0, 1.5, 1.0))
    if bc[0] == N:
        W.u[:, :, -1] = 0.0
    if bc[1] == N:
        W.v[:, -1, :] = 0.0
    if bc[2] == N:
        W.w[-1] = 0.0
    return W


@pytest.mark.parametrize("bc", [(N, N, N), (P, N, N), (N, P, N), (N, N, P), (N, P, P)])
@pytest.mark.parametrize("ratio", [1000.0, 0.05])
def test_b4_step_with_walls(oracle_mod, bc, ratio):
    W = _walled_case(12, 10, 8, bc, ratio, 71)
    u, v, w, p, rhs = oracle_mod.projection_step_bc(*W.fields(), W.box, bc, W.rho1, W.rho2, W.dt, return_rhs=True)
    d0, d1 = ops.div_bc(W.u, W.v, W.w, W.box, bc), ops.div_bc(u, v, w, W.box, bc)
    assert np.linalg.norm(d1) / np.linalg.norm(d0) < 1e-12                                  # div-free (P3)
    assert np.linalg.norm(ops.lap_bc(p, W.box, bc) - (rhs - rhs.mean())) / np.linalg.norm(rhs) < 1e-12    # residual (P4)
    assert abs(p.mean()) < 1e-13 * np.sqrt(np.mean(p ** 2))                                 # gauge (P5)
    assert abs(rhs.sum()) / np.abs(rhs).sum() < 1e-14                                       # compatibility
    if bc[0] == N:
        assert np.array_equal(u[:, :, -1], W.u[:, :, -1])                                   # wall faces pass through (R8)
    if bc[1] == N:
        assert np.array_equal(v[:, -1, :], W.v[:, -1, :])
    if bc[2] == N:
        assert np.array_equal(w[-1], W.w[-1])
    # independent numpy statement of rhs and correction
    rho0 = min(W.rho1, W.rho2)
    rf = ops.face_density_bc(W.phi, W.rho1, W.rho2, bc)
    gh = ops.grad_bc(2.0 * W.p - W.p_old, W.box, bc)
    F = [(1.0 - rho0 / r) * g for r, g in zip(rf, gh)]
    assert ops.rel_l2(rhs, rho0 / W.dt * d0 + ops.div_bc(*F, W.box, bc)) < 1e-12
    gn = ops.grad_bc(p, W.box, bc)
    for a, us, r, g1, g2 in zip((u, v, w), (W.u, W.v, W.w), rf, gn, gh):
        assert ops.rel_l2(a, us - W.dt * (g1 / rho0 + (1.0 / r - 1.0 / rho0) * g2)) < 1e-12
    # the pieces on their own are the step's pieces, bit for bit
    assert np.array_equal(oracle_mod.rhs_bc(*W.fields(), W.box, bc, W.rho1, W.rho2, W.dt), rhs)
    assert np.array_equal(oracle_mod.poisson_bc(rhs, W.box, bc), p)
    for a, b in zip(oracle_mod.correction_bc(*W.fields(), p, W.box, bc, W.rho1, W.rho2, W.dt), (u, v, w)):
        assert np.array_equal(a, b)


@pytest.mark.parametrize("bc", [(N, N, N), (P, N, N)])
def test_b4_fixed_point_with_walls(oracle_mod, bc):
    """the steady-state fixed point P3b in a walled box: pins sign / grouping (R1) and the wall-face density"""
    W = _walled_case(10, 12, 8, bc, 50.0, 73)
    ut, vt, wt, _ = oracle_mod.projection_step_bc(W.u, W.v, W.w, W.phi, W.p, W.p_old, W.box, bc, 1.0, 1.0, W.dt)
    p = W.p - W.p.mean()
    rf = ops.face_density_bc(W.phi, W.rho1, W.rho2, bc)
    g = ops.grad_bc(p, W.box, bc)
    us, vs, ws = (a + W.dt * gg / r for a, gg, r in zip((ut, vt, wt), g, rf))
    u, v, w, pn = oracle_mod.projection_step_bc(us, vs, ws, W.phi, p, p, W.box, bc, W.rho1, W.rho2, W.dt)
    assert ops.rel_l2(pn, p) < 1e-10
    for a, b in ((u, ut), (v, vt), (w, wt)):
        assert ops.rel_l2(a, b) < 1e-12


@pytest.mark.parametrize("bcz", [P, N])
def test_b4_periodic_xy_is_the_original_entry_point_bit_for_bit(oracle_mod, bcz):
    W = wl.random_case(12, 10, 8, bcz, 50.0, 75)
    a = oracle_mod.projection_step(*W.fields(), W.box, bcz, W.rho1, W.rho2, W.dt)
    b = oracle_mod.projection_step_bc(*W.fields(), W.box, (P, P, bcz), W.rho1, W.rho2, W.dt)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
