"""Pins for the CPU oracle (oracle/): everything here checks the oracle against what the paper
and the mathematics fix, never against itself and never against the CUDA path.

The paper prints no worked numbers for the projection step (no table or figure gives a
pressure or a divergence), so the pins are structural:
  P0  naive DFT vs closed forms (delta, single exponential) and numpy.fft
  P1  exact discrete eigenpairs of the 7-point Laplacian
  P2  dense bordered direct solve on tiny grids, both BCs (brute force)
  P3  div u^(n+1) = 0 to round-off for ANY density ratio
  P3b steady-state fixed point: pins sign/grouping of eq. 16 (R1) and the face density (R2)
  P4  residual || L p - (rhs - mean rhs) || / || rhs ||
  P5  zero-mean gauge and compatibility (R5)
  P6  rho1 = rho2: classical projection, independent of p, p_old; idempotent; wall faces
  P7  linearity and shift covariance
  P8  the paper's incremental grouping (eqs. 16-19) == the north_star grouping
  P9  independent numpy.fft + vectorised-Thomas restatement of the whole step
  P10 variable time step: p_hat is the linear extrapolation of the pressure history to
      t^(n+1); r = 1 is the constant-dt step bit for bit; a pressure linear in time is extrapolated exactly
"""
import numpy as np
import pytest

import workloads as wl
from tests import np_ops as ops

PER, WALL = 0, 1


def _step(oracle, W, **kw):
    return oracle.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt, **kw)


# --------------------------------------------------------------------------- P0: DFT
@pytest.mark.parametrize("n", [1, 2, 5, 8, 12])
def test_dft_closed_forms(oracle_mod, n):
    # delta at j0 -> pure phase exp(-2 pi i k j0 / n)
    for j0 in range(min(n, 3)):
        x = np.zeros((2, n, 3), dtype=complex)
        x[:, j0, :] = 1.0
        X = oracle_mod.dft_axis(x, 1, -1)
        k = np.arange(n)
        assert np.allclose(X, np.exp(-2j * np.pi * k * j0 / n)[None, :, None], atol=1e-14)
    # single exponential with frequency m -> n * delta_{k,m}; inverse sign -> delta at n-m
    for m in range(min(n, 3)):
        x = np.exp(2j * np.pi * m * np.arange(n) / n)[None, :, None] * np.ones((1, 1, 2))
        X = oracle_mod.dft_axis(x, 1, -1)
        want = np.zeros(n); want[m] = n
        assert np.allclose(X[0, :, 0], want, atol=1e-12 * n)
        Xi = oracle_mod.dft_axis(x, 1, +1)
        want = np.zeros(n); want[(n - m) % n] = n
        assert np.allclose(Xi[0, :, 0], want, atol=1e-12 * n)


def test_dft_matches_numpy_fft_on_every_axis(oracle_mod):
    rng = np.random.default_rng(7)
    x = rng.standard_normal((5, 6, 7)) + 1j * rng.standard_normal((5, 6, 7))
    for ax in range(3):
        assert ops.rel_l2(oracle_mod.dft_axis(x, ax, -1), np.fft.fft(x, axis=ax)) < 1e-14
        assert ops.rel_l2(oracle_mod.dft_axis(x, ax, +1), np.fft.ifft(x, axis=ax) * x.shape[ax]) < 1e-14


# ------------------------------------------------------------------- operators vs numpy
@pytest.mark.parametrize("bc", [PER, WALL])
def test_operators_match_independent_numpy(oracle_mod, bc):
    rng = np.random.default_rng(11)
    shape, box = (5, 6, 8), (1.3, 0.7, 2.1)
    a, b, c, f = (rng.standard_normal(shape) for _ in range(4))
    assert ops.rel_l2(oracle_mod.divergence(a, b, c, box, bc), ops.div(a, b, c, box, bc == WALL)) < 1e-14
    assert ops.rel_l2(oracle_mod.laplacian(f, box, bc), ops.lap(f, box, bc == WALL)) < 1e-13


# ------------------------------------------------------------------------ P1: eigenpairs
def _eigen_mode(shape, box, bc, a, b, c, alpha=0.3, beta=1.1):
    nz, ny, nx = shape
    dx, dy, dz = ops.spacings(shape, box)
    i, j, k = np.arange(nx), np.arange(ny), np.arange(nz)
    fx = np.cos(2 * np.pi * a * i / nx + alpha)
    fy = np.cos(2 * np.pi * b * j / ny + beta)
    if bc == PER:
        fz = np.cos(2 * np.pi * c * k / nz + 0.7)
        lz = -2.0 * (1.0 - np.cos(2 * np.pi * c / nz)) / dz ** 2
    else:
        fz = np.cos(np.pi * c * (k + 0.5) / nz)           # Neumann eigenvector (R6)
        lz = -2.0 * (1.0 - np.cos(np.pi * c / nz)) / dz ** 2
    lam = (-2.0 * (1.0 - np.cos(2 * np.pi * a / nx)) / dx ** 2
           - 2.0 * (1.0 - np.cos(2 * np.pi * b / ny)) / dy ** 2 + lz)
    return fz[:, None, None] * fy[None, :, None] * fx[None, None, :], lam


@pytest.mark.parametrize("bc", [PER, WALL])
@pytest.mark.parametrize("abc", [(1, 0, 0), (0, 2, 0), (0, 0, 3), (3, 1, 2), (2, 5, 1), (0, 0, 1)])
def test_p1_eigenpairs(oracle_mod, bc, abc):
    shape, box = (10, 12, 16), (2.0, 3.0, 1.0)          # distinct sizes: catches swapped axes
    f, lam = _eigen_mode(shape, box, bc, *abc)
    # the oracle's Laplacian has this eigenpair ...
    assert ops.rel_l2(oracle_mod.laplacian(f, box, bc), lam * f) < 1e-12
    # ... and its solver inverts it (f has zero mean because (a,b,c) != 0)
    p, imag = oracle_mod.poisson(lam * f, box, bc, return_imag_residue=True)
    assert ops.rel_l2(p, f) < 1e-12
    assert imag < 1e-13


# --------------------------------------------------------------- P2: dense bordered solve
def _dense_laplacian(shape, box, wall):
    n = int(np.prod(shape))
    L = np.empty((n, n))
    e = np.zeros(n)
    for q in range(n):
        e[q] = 1.0
        L[:, q] = ops.lap(e.reshape(shape), box, wall).ravel()
        e[q] = 0.0
    return L


@pytest.mark.parametrize("bc", [PER, WALL])
@pytest.mark.parametrize("shape", [(8, 8, 8), (5, 6, 8)])
def test_p2_dense_bordered_solve(oracle_mod, bc, shape):
    box = (1.0, 1.5, 0.8)
    rng = np.random.default_rng(3)
    rhs = rng.standard_normal(shape)
    rhs -= rhs.mean()
    n = rhs.size
    L = _dense_laplacian(shape, box, bc == WALL)
    assert np.allclose(L, L.T, atol=1e-9) and np.allclose(L.sum(axis=1), 0.0, atol=1e-9)  # P7: symmetric, zero row sums
    K = np.zeros((n + 1, n + 1))
    K[:n, :n] = L
    K[:n, n] = 1.0
    K[n, :n] = 1.0
    sol = np.linalg.solve(K, np.append(rhs.ravel(), 0.0))
    p = oracle_mod.poisson(rhs, box, bc)
    assert ops.rel_l2(p.ravel(), sol[:n]) < 1e-12
    assert abs(sol[n]) < 1e-10


# --------------------------------------------------------------------- P3, P4, P5 on configs
def _cases():
    return [wl.config1(), wl.random_case(16, 12, 10, WALL, 10.0, 5), wl.random_case(12, 16, 8, PER, 1000.0, 6),
            wl.random_case(8, 8, 24, WALL, 1000.0, 7), wl.config3(32, 16, 12)]


@pytest.mark.parametrize("idx", range(5))
def test_p3_p4_p5_divfree_residual_gauge(oracle_mod, idx):
    W = _cases()[idx]
    wall = W.bc_z == WALL
    u, v, w, p, rhs = _step(oracle_mod, W, return_rhs=True)
    d0, d1 = ops.div(W.u, W.v, W.w, W.box, wall), ops.div(u, v, w, W.box, wall)
    assert np.linalg.norm(d1) / np.linalg.norm(d0) < 1e-12                       # P3
    assert np.linalg.norm(ops.lap(p, W.box, wall) - (rhs - rhs.mean())) / np.linalg.norm(rhs) < 1e-12   # P4
    assert abs(p.mean()) < 1e-13 * np.sqrt(np.mean(p ** 2))                      # P5 gauge
    assert abs(rhs.sum()) / np.abs(rhs).sum() < 1e-14                            # P5 compatibility
    if wall:
        assert np.array_equal(w[-1], W.w[-1])                                    # P6/R8: wall face untouched


# ------------------------------------------------------------- P3b: steady-state fixed point
@pytest.mark.parametrize("bc,ratio", [(PER, 50.0), (WALL, 1000.0), (PER, 0.02)])
def test_p3b_fixed_point(oracle_mod, bc, ratio):
    """u* = u_divfree + dt (1/rho_f) grad p with p_old = p  ==>  p^(n+1) = p and u = u_divfree, for any
    density ratio.  The literal (garbled) sign of eq. 16 fails this by O(1) in p (R1)."""
    W = wl.random_case(12, 10, 8, bc, ratio, 21)
    wall = bc == WALL
    # a discretely divergence-free field: project white noise once with rho1 = rho2
    ut, vt, wt, _ = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, W.p, W.p_old, W.box, bc, 1.0, 1.0, W.dt)
    assert np.linalg.norm(ops.div(ut, vt, wt, W.box, wall)) < 1e-11 * np.linalg.norm(ops.div(W.u, W.v, W.w, W.box, wall))
    p = W.p - W.p.mean()
    rx, ry, rz = ops.face_density(W.phi, W.rho1, W.rho2, wall)
    gx, gy, gz = ops.grad(p, W.box, wall)
    us, vs, ws = ut + W.dt * gx / rx, vt + W.dt * gy / ry, wt + W.dt * gz / rz
    u, v, w, pn = oracle_mod.projection_step(us, vs, ws, W.phi, p, p, W.box, bc, W.rho1, W.rho2, W.dt)
    assert ops.rel_l2(pn, p) < 1e-10
    for a, b in ((u, ut), (v, vt), (w, wt)):
        assert ops.rel_l2(a, b) < 1e-12


# ------------------------------------------- P3c: the correction entry point on its own
@pytest.mark.parametrize("bc,ratio", [(PER, 50.0), (WALL, 1000.0)])
def test_p3c_correction_entry_point(oracle_mod, bc, ratio):
    """oracle.correction (the call that certifies u, v, w at full size) against an independent numpy statement of
    eq. 18 in the north_star grouping, against the step it is a part of (bit for bit), and with its pressure
    arguments swapped (must differ: a transposed p / p_old / p_new in the entry point or its wrapper fails here)."""
    W = wl.random_case(12, 10, 8, bc, ratio, 61)
    wall = bc == WALL
    rhs = oracle_mod.rhs(*W.fields(), W.box, bc, W.rho1, W.rho2, W.dt)
    pn = oracle_mod.poisson(rhs, W.box, bc)
    got = oracle_mod.correction(*W.fields(), pn, W.box, bc, W.rho1, W.rho2, W.dt)
    # (a) independent numpy restatement: u = u* - dt [ grad p_new / rho0 + (1/rho_f - 1/rho0) grad p_hat ]
    rho0 = min(W.rho1, W.rho2)
    rf = ops.face_density(W.phi, W.rho1, W.rho2, wall)
    gn, gh = ops.grad(pn, W.box, wall), ops.grad(2.0 * W.p - W.p_old, W.box, wall)
    for a, us, r, g1, g2 in zip(got, (W.u, W.v, W.w), rf, gn, gh):
        assert ops.rel_l2(a, us - W.dt * (g1 / rho0 + (1.0 / r - 1.0 / rho0) * g2)) < 1e-13
    # (b) the same arithmetic as the whole step: bit for bit
    step = _step(oracle_mod, W)
    for a, b in zip(got, step[:3]):
        assert np.array_equal(a, b)
    assert np.array_equal(pn, step[3])
    # (c) every transposition of the three pressure arguments changes the result
    f = W.fields()
    for perm in ((pn, f[5], f[4]), (f[4], pn, f[5]), (f[5], f[4], pn), (f[4], f[5], f[4])):
        bad = oracle_mod.correction(f[0], f[1], f[2], f[3], perm[0], perm[1], perm[2], W.box, bc, W.rho1, W.rho2, W.dt)
        assert ops.rel_l2(bad[0], got[0]) > 1e-6
    if wall:
        assert np.array_equal(got[2][-1], W.w[-1])


# --------------------------------------------------------------------- P6: special cases
@pytest.mark.parametrize("bc", [PER, WALL])
def test_p6_constant_density_is_classical_projection(oracle_mod, bc):
    W = wl.random_case(10, 12, 8, bc, 1.0, 31)
    wall = bc == WALL
    a = _step(oracle_mod, W)
    rng = np.random.default_rng(99)
    b = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, rng.standard_normal(W.shape), rng.standard_normal(W.shape),
                                   W.box, bc, 1.0, 1.0, W.dt)
    for x, y in zip(a, b):
        assert ops.rel_l2(x, y) < 1e-13                      # independent of p, p_old
    # classical Chorin projection: u = u* - dt/rho0 grad p with L p = rho0/dt div u*
    gx, gy, gz = ops.grad(a[3], W.box, wall)
    assert ops.rel_l2(a[0], W.u - W.dt * gx) < 1e-13
    # idempotent: projecting the projected field changes nothing and returns p ~ 0
    c = oracle_mod.projection_step(a[0], a[1], a[2], W.phi, W.p, W.p_old, W.box, bc, 1.0, 1.0, W.dt)
    for x, y in zip(c[:3], a[:3]):
        assert ops.rel_l2(x, y) < 1e-12
    dx = W.box[0] / W.nx
    assert np.max(np.abs(c[3])) < 1e-12 * (1.0 / W.dt) * np.max(np.abs(W.u)) * dx * 100


# ------------------------------------------------------------------------ P7: symmetries
def test_p7_linearity_and_shift(oracle_mod):
    W = wl.random_case(12, 8, 10, PER, 20.0, 41)
    rng = np.random.default_rng(5)
    X = [rng.standard_normal(W.shape) for _ in range(5)]
    Y = [rng.standard_normal(W.shape) for _ in range(5)]
    f = lambda Z: oracle_mod.projection_step(Z[0], Z[1], Z[2], W.phi, Z[3], Z[4], W.box, PER, W.rho1, W.rho2, W.dt)
    a, b = f(X), f(Y)
    c = f([2.0 * x - 3.0 * y for x, y in zip(X, Y)])
    for ra, rb, rc in zip(a, b, c):
        assert ops.rel_l2(rc, 2.0 * ra - 3.0 * rb) < 1e-12
    # periodic shift by one cell in x and two in y of all inputs shifts all outputs
    sh = lambda t: np.roll(np.roll(t, 1, axis=2), 2, axis=1)
    d = oracle_mod.projection_step(sh(X[0]), sh(X[1]), sh(X[2]), sh(W.phi), sh(X[3]), sh(X[4]), W.box, PER,
                                   W.rho1, W.rho2, W.dt)
    for ra, rd in zip(a, d):
        assert ops.rel_l2(rd, sh(ra)) < 1e-12


# ------------------------------------------------------------------ P8: grouping identity
@pytest.mark.parametrize("idx", range(5))
def test_p8_paper_grouping_equals_north_star_grouping(oracle_mod, idx):
    W = _cases()[idx]
    a = _step(oracle_mod, W)
    b = oracle_mod.projection_step_paper(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt)
    for x, y in zip(a, b):
        assert ops.rel_l2(y, x) < 1e-13 * (10 if W.rho2 > 100 else 1)


# ------------------------------------------------------------- P10: variable time step
@pytest.mark.parametrize("bc", [PER, WALL])
def test_p10_unit_ratio_is_the_constant_dt_step_bit_for_bit(oracle_mod, bc):
    W = wl.random_case(12, 10, 8, bc, 50.0, 51)
    a = _step(oracle_mod, W, return_rhs=True)
    b = _step(oracle_mod, W, return_rhs=True, dt_ratio=1.0)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


@pytest.mark.parametrize("bc,r", [(PER, 0.5), (WALL, 1.7), (PER, 2.0)])
def test_p10_variable_dt_is_linear_extrapolation_in_time(oracle_mod, bc, r):
    """p_hat = (1 + r) p^n - r p^(n-1), r = dt^(n+1)/dt^n, is the straight line through
    (t^(n-1), p^(n-1)) and (t^n, p^n) evaluated at t^(n+1).  So for a history p(t) = A + t B sampled at
    t^(n-1) = -dt_n and t^n = 0, the step with ratio r must equal the CONSTANT-dt step fed the history
    resampled at -dt_(n+1) (whose 2 p^n - p^(n-1) is the same p(t^(n+1)) = A + dt_(n+1) B); a wrong sign,
    a swapped coefficient or an inverted ratio all change p_hat by O(1) and fail this."""
    W = wl.random_case(10, 12, 8, bc, 20.0, 52)
    rng = np.random.default_rng(53)
    A, B = rng.uniform(-0.1, 0.1, W.shape), rng.uniform(-30.0, 30.0, W.shape)
    dt_new = W.dt
    dt_old = dt_new / r
    p_n, p_nm1 = A, A - dt_old * B
    got = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, p_n, p_nm1, W.box, bc, W.rho1, W.rho2, dt_new,
                                     return_rhs=True, dt_ratio=r)
    want = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, p_n, A - dt_new * B, W.box, bc, W.rho1, W.rho2,
                                      dt_new, return_rhs=True)
    for x, y in zip(got, want):
        assert ops.rel_l2(x, y) < 1e-12
    # and the two histories really differ: with the wrong ratio the result moves by far more than round-off
    wrong = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, p_n, p_nm1, W.box, bc, W.rho1, W.rho2, dt_new,
                                       dt_ratio=1.0 / r)
    assert ops.rel_l2(wrong[3], want[3]) > 1e-6


def test_p10_fixed_point_and_divfree_hold_for_any_ratio(oracle_mod):
    """p_old = p makes p_hat = p for every r, so the steady state of P3b is a fixed point for every r;
    div u^(n+1) = 0 holds for every r because rhs and correction share the same p_hat."""
    bc, ratio, r = WALL, 100.0, 0.37
    W = wl.random_case(12, 10, 8, bc, ratio, 54)
    ut, vt, wt, _ = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, W.p, W.p_old, W.box, bc, 1.0, 1.0, W.dt)
    p = W.p - W.p.mean()
    rx, ry, rz = ops.face_density(W.phi, W.rho1, W.rho2, True)
    gx, gy, gz = ops.grad(p, W.box, True)
    us, vs, ws = ut + W.dt * gx / rx, vt + W.dt * gy / ry, wt + W.dt * gz / rz
    u, v, w, pn = oracle_mod.projection_step(us, vs, ws, W.phi, p, p, W.box, bc, W.rho1, W.rho2, W.dt, dt_ratio=r)
    assert ops.rel_l2(pn, p) < 1e-10
    for a, b in ((u, ut), (v, vt), (w, wt)):
        assert ops.rel_l2(a, b) < 1e-12
    u, v, w, _ = _step(oracle_mod, W, dt_ratio=r)
    d0, d1 = ops.div(W.u, W.v, W.w, W.box, True), ops.div(u, v, w, W.box, True)
    assert np.linalg.norm(d1) / np.linalg.norm(d0) < 1e-12


# ------------------------------------------------------ P9: independent numpy restatement
def mid_oracle(W):
    """numpy.fft + vectorised Thomas restatement of the whole step (tests only)."""
    wall = W.bc_z == WALL
    dx, dy, dz = ops.spacings(W.shape, W.box)
    rho0 = min(W.rho1, W.rho2)
    rx, ry, rz = ops.face_density(W.phi, W.rho1, W.rho2, wall)
    ph = 2.0 * W.p - W.p_old
    gx, gy, gz = ops.grad(ph, W.box, wall)
    rhs = rho0 / W.dt * ops.div(W.u, W.v, W.w, W.box, wall) + ops.div((1 - rho0 / rx) * gx, (1 - rho0 / ry) * gy,
                                                                     (1 - rho0 / rz) * gz, W.box, wall)
    lam = lambda n, d: -2.0 * (1.0 - np.cos(2 * np.pi * np.arange(n) / n)) / d ** 2
    lx_, ly_ = lam(W.nx, dx)[: W.nx // 2 + 1], lam(W.ny, dy)
    if not wall:
        R = np.fft.rfftn(rhs)
        den = lam(W.nz, dz)[:, None, None] + ly_[None, :, None] + lx_[None, None, :]
        den[0, 0, 0] = 1.0
        R /= den
        R[0, 0, 0] = 0.0
        pn = np.fft.irfftn(R, s=W.shape, axes=(0, 1, 2))
    else:
        R = np.fft.rfft2(rhs, axes=(1, 2))
        lxy = ly_[:, None] + lx_[None, :]
        nz = W.nz
        a = 1.0 / dz ** 2
        b = np.full((nz,) + lxy.shape, -2.0 * a) + lxy[None]
        b[0] += a; b[-1] += a
        cp = np.zeros_like(b); dp = np.zeros_like(R)
        with np.errstate(divide="ignore", invalid="ignore"):
            cp[0] = a / b[0]; dp[0] = R[0] / b[0]
            for k in range(1, nz):
                m = b[k] - a * cp[k - 1]
                cp[k] = a / m
                dp[k] = (R[k] - a * dp[k - 1]) / m
        x = np.zeros_like(R)
        x[-1] = dp[-1]
        x[-1, 0, 0] = 0.0                                 # pinned singular column
        for k in range(nz - 2, -1, -1):
            x[k] = dp[k] - cp[k] * x[k + 1]
        x[:, 0, 0] -= x[:, 0, 0].mean()
        pn = np.fft.irfft2(x, s=W.shape[1:], axes=(1, 2))
    g1, g2, g3 = ops.grad(pn, W.box, wall)
    u = W.u - W.dt * (g1 / rho0 + (1 / rx - 1 / rho0) * gx)
    v = W.v - W.dt * (g2 / rho0 + (1 / ry - 1 / rho0) * gy)
    w = W.w - W.dt * (g3 / rho0 + (1 / rz - 1 / rho0) * gz)
    return u, v, w, pn, rhs


@pytest.mark.parametrize("maker", [lambda: wl.config1(), lambda: wl.config2(32, 3, 3, 4),
                                   lambda: wl.config3(32, 16, 24), lambda: wl.config4(32, 50.0, 3, 0.05, 4),
                                   lambda: wl.config5(32, 16, 24)])
def test_p9_numpy_fft_restatement(oracle_mod, maker):
    W = maker()
    a = _step(oracle_mod, W, return_rhs=True)
    b = mid_oracle(W)
    names = "u v w p rhs".split()
    for name, x, y in zip(names, a, b):
        assert ops.rel_l2(x, y) < 1e-12, name
