"""Pins for the oracle's momentum prediction (oracle.momentum_prediction; eq. 15,
PAPER.md:90 eq. 5).  The paper prints no worked numbers for it, so the pins are what the discretisation
and the continuum equations fix:
  M1  conservation: the convective term and the density-weighted viscous term sum to zero over the periodic box
      (divergence form: every flux / stress appears twice with opposite signs) -- catches any sign or index slip
  M2  kinetic energy: for a discretely divergence-free field the convective term does no work, sum u . conv = 0
      (Harlow-Welch property of the two-point-mean divergence form) -- catches wrong averaging partners
  M3  constant viscosity: div[mu (grad u + grad u^T)] = mu (L u + grad div u) exactly on the staggered grid,
      against independent numpy operators
  M4  Taylor-Green vortex: M(u) -> (-1/2 sin 2x - 2 nu u, -1/2 sin 2y - 2 nu v) with second-order convergence
  M5  variable viscosity, manufactured shear flows: the normal, the shear and the transposed-gradient terms, second order
  M6  the time update: Adams-Bashforth coefficients (1 + r/2, r/2) = linear extrapolation of M to t^(n+1/2);
      gravity and the continuum surface force against a numpy statement
"""
import numpy as np
import pytest

import workloads as wl
from tests import np_ops as ops

TWO_PI = 2.0 * np.pi


def _mp(oracle, u, v, w, phi, box, kappa=None, m_old=None, rho=(1.0, 1.0), mu=(0.0, 0.0), sigma=0.0, grav=(0.0, 0.0, 0.0),
        dt=1e-3, r=1.0):
    if m_old is None:
        m_old = [np.zeros_like(u)] * 3
    return oracle.momentum_prediction(u, v, w, phi, kappa, m_old, box, rho[0], rho[1], mu[0], mu[1], sigma, grav, dt, r)


def _rand(shape, seed):
    rng = np.random.default_rng(seed)
    return [rng.standard_normal(shape) for _ in range(3)], rng.random(shape)


def test_m1_conservation(oracle_mod):
    shape, box = (6, 8, 10), (1.3, 0.9, 0.7)
    (u, v, w), phi = _rand(shape, 1)
    _, conv = _mp(oracle_mod, u, v, w, phi, box)                               # mu = 0: M is the convective term
    for c in conv:
        assert abs(c.sum()) < 1e-12 * np.abs(c).sum()
    _, full = _mp(oracle_mod, u, v, w, phi, box, rho=(1.0, 7.0), mu=(0.3, 2.0))
    rf = ops.face_density_bc(phi, 1.0, 7.0, (0, 0, 0))
    for m, c, r in zip(full, conv, rf):
        visc = (m - c) * r                                                      # rho_f * (1/rho_f) div(stress)
        assert abs(visc.sum()) < 1e-12 * np.abs(visc).sum()


def test_m2_convection_does_no_work_on_a_divergence_free_field(oracle_mod):
    W = wl.random_case(12, 10, 8, 0, 1.0, 91)
    u, v, w, _ = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, W.p, W.p_old, W.box, 0, 1.0, 1.0, W.dt)
    assert np.linalg.norm(ops.div(u, v, w, W.box, False)) < 1e-11 * np.linalg.norm(ops.div(W.u, W.v, W.w, W.box, False))
    _, conv = _mp(oracle_mod, u, v, w, W.phi, W.box)
    work = sum((a * c).sum() for a, c in zip((u, v, w), conv))
    scale = sum((np.abs(a) * np.abs(c)).sum() for a, c in zip((u, v, w), conv))
    assert abs(work) < 1e-12 * scale
    # ... and it does work on a field that is not divergence free (the pin is not vacuous)
    _, conv2 = _mp(oracle_mod, W.u, W.v, W.w, W.phi, W.box)
    assert abs(sum((a * c).sum() for a, c in zip((W.u, W.v, W.w), conv2))) > 1e-3 * scale


def test_m3_constant_viscosity_is_laplacian_plus_grad_div(oracle_mod):
    shape, box = (6, 8, 10), (1.3, 0.9, 0.7)
    (u, v, w), phi = _rand(shape, 3)
    nu, rho = 0.37, 2.5
    _, conv = _mp(oracle_mod, u, v, w, phi, box, rho=(rho, rho))
    _, full = _mp(oracle_mod, u, v, w, phi, box, rho=(rho, rho), mu=(nu * rho, nu * rho))
    gd = ops.grad(ops.div(u, v, w, box, False), box, False)                     # grad(div u) lives on the faces
    for m, c, a, g in zip(full, conv, (u, v, w), gd):
        assert ops.rel_l2(m - c, nu * (ops.lap(a, box, False) + g)) < 1e-12


def _taylor_green(n, nu):
    box = (TWO_PI,) * 3
    d = TWO_PI / n
    xc, xf = (np.arange(n) + 0.5) * d, (np.arange(n) + 1.0) * d
    one = np.ones((n, 1, 1))
    u = one * (np.cos(xc)[None, :, None] * np.sin(xf)[None, None, :])            # u(x_face, y_centre)
    v = -one * (np.sin(xf)[None, :, None] * np.cos(xc)[None, None, :])           # v(x_centre, y_face)
    mu_exact = -0.5 * np.sin(2 * xf)[None, None, :] * np.ones((n, n, 1)) - 2 * nu * u
    mv_exact = -0.5 * np.sin(2 * xf)[None, :, None] * np.ones((n, 1, n)) - 2 * nu * v
    return box, u, v, np.zeros_like(u), mu_exact, mv_exact


def test_m4_taylor_green_second_order(oracle_mod):
    nu, errs = 0.1, []
    for n in (16, 32):
        box, u, v, w, mu_e, mv_e = _taylor_green(n, nu)
        _, (mu_, mv_, mw_) = _mp(oracle_mod, u, v, w, np.ones_like(u), box, mu=(nu, nu))
        errs.append(max(np.abs(mu_ - mu_e).max(), np.abs(mv_ - mv_e).max()))
        assert np.abs(mw_).max() < 1e-14
    assert 3.6 < errs[0] / errs[1] < 4.4 and errs[1] < 1e-2


def test_m5_variable_viscosity_manufactured(oracle_mod):
    mu1, mu2 = 3.0, 0.5
    errs = {"shear": [], "transpose": [], "normal": []}
    for n in (16, 32):
        box, d = (TWO_PI,) * 3, TWO_PI / n
        c, f = (np.arange(n) + 0.5) * d, (np.arange(n) + 1.0) * d
        Y, X = c[None, :, None] * np.ones((n, 1, n)), c[None, None, :] * np.ones((n, n, 1))
        Yf, Xf = f[None, :, None] * np.ones((n, 1, n)), f[None, None, :] * np.ones((n, n, 1))
        z = np.zeros((n, n, n))
        phi = 0.5 * (1.0 + 0.8 * np.sin(Y))                                      # mu = mu(y)
        mu = lambda y: mu2 + (mu1 - mu2) * 0.5 * (1.0 + 0.8 * np.sin(y))
        dmu = lambda y: (mu1 - mu2) * 0.4 * np.cos(y)
        # u = sin y: (1/rho) d/dy (mu du/dy), convection vanishes
        _, (a, b, _c) = _mp(oracle_mod, np.sin(Y), z, z, phi, box, mu=(mu1, mu2))
        errs["shear"].append(np.abs(a - (dmu(Y) * np.cos(Y) - mu(Y) * np.sin(Y))).max())
        # v = sin x: the transposed gradient feeds the x equation, d/dy (mu dv/dx), and d/dx (mu dv/dx) the y equation
        _, (a, b, _c) = _mp(oracle_mod, z, np.sin(X), z, phi, box, mu=(mu1, mu2))
        errs["transpose"].append(max(np.abs(a - dmu(Y) * np.cos(Xf)).max(), np.abs(b + mu(Yf) * np.sin(X)).max()))
        # v = sin y: normal stress d/dy (2 mu dv/dy) minus the convective d/dy (v v)
        _, (a, b, _c) = _mp(oracle_mod, z, np.sin(Yf), z, phi, box, mu=(mu1, mu2))
        errs["normal"].append(np.abs(b - (2 * dmu(Yf) * np.cos(Yf) - 2 * mu(Yf) * np.sin(Yf) - np.sin(2 * Yf))).max())
    for k, (e0, e1) in errs.items():
        assert 3.4 < e0 / e1 < 4.6, (k, e0, e1)


def test_m6_time_update_and_sources(oracle_mod):
    shape, box = (6, 8, 10), (1.3, 0.9, 0.7)
    (u, v, w), phi = _rand(shape, 6)
    rng = np.random.default_rng(7)
    kappa = rng.standard_normal(shape)
    rho, mu, sigma, grav, dt = (1.0, 20.0), (0.2, 1.0), 0.07, (0.3, -0.2, -9.81), 2e-3
    _, m_new = _mp(oracle_mod, u, v, w, phi, box, rho=rho, mu=mu)
    b = [rng.standard_normal(shape) for _ in range(3)]                          # dM/dt of a history that is linear in time
    for r in (1.0, 0.5, 1.7):
        dt_old = dt / r
        m_old = [m - bb * dt_old for m, bb in zip(m_new, b)]
        us, m2 = _mp(oracle_mod, u, v, w, phi, box, kappa=kappa, m_old=m_old, rho=rho, mu=mu, sigma=sigma, grav=grav, dt=dt, r=r)
        for x, y in zip(m2, m_new):
            assert np.array_equal(x, y)                                          # M(u^n) does not depend on history or sources
        rf = ops.face_density_bc(phi, rho[0], rho[1], (0, 0, 0))
        gphi = ops.grad(phi, box, False)
        for d, (a, a0, m, bb, r_f, gp) in enumerate(zip(us, (u, v, w), m_new, b, rf, gphi)):
            kf = 0.5 * (kappa + np.roll(kappa, -1, axis=2 - d))
            want = a0 + dt * (m + bb * dt / 2.0 + grav[d] + sigma * kf * gp / r_f)     # M extrapolated to t^n + dt/2
            assert ops.rel_l2(a, want) < 1e-12
    us, _ = _mp(oracle_mod, u, v, w, phi, box, m_old=m_new, rho=rho, mu=mu, grav=grav, dt=dt, r=1.0)
    for d, (a, a0, m) in enumerate(zip(us, (u, v, w), m_new)):
        assert ops.rel_l2(a, a0 + dt * (m + grav[d])) < 1e-13                    # classic AB2: 3/2 - 1/2


def test_m7_start_up_step_is_explicit_euler(oracle_mod):
    """DESIGN.md R29 (PAPER.md:140, 161 with r = 0): f1 = 1, f2 = 0 -- the update is u + dt (M(u) + sources) whatever the
    history holds, and the projection's extrapolated pressure is p^n itself whatever p^(n-1) holds"""
    shape, box = (6, 8, 10), (1.3, 0.9, 0.7)
    (u, v, w), phi = _rand(shape, 8)
    rng = np.random.default_rng(9)
    rho, mu, grav, dt = (1.0, 20.0), (0.2, 1.0), (0.3, -0.2, -9.81), 2e-3
    junk = [1e3 * rng.standard_normal(shape) for _ in range(3)]
    us, m_new = _mp(oracle_mod, u, v, w, phi, box, m_old=junk, rho=rho, mu=mu, grav=grav, dt=dt, r=0.0)
    us0, _ = _mp(oracle_mod, u, v, w, phi, box, rho=rho, mu=mu, grav=grav, dt=dt, r=0.0)
    for d, (a, b, a0, m) in enumerate(zip(us, us0, (u, v, w), m_new)):
        assert np.array_equal(a, b)
        assert ops.rel_l2(a, a0 + dt * (m + grav[d])) < 1e-14
    p, p_old = rng.standard_normal(shape), rng.standard_normal(shape)
    got = oracle_mod.rhs(u, v, w, phi, p, p_old, box, 0, rho[0], rho[1], dt, dt_ratio=0.0)
    same = oracle_mod.rhs(u, v, w, phi, p, 7.0 * p_old + 1.0, box, 0, rho[0], rho[1], dt, dt_ratio=0.0)
    assert np.array_equal(got, same)
    # with p^(n-1) = p^n every r gives p_hat = p^n: r = 0 must agree with r = 1 up to the rounding of (2 p - p)
    ref = oracle_mod.rhs(u, v, w, phi, p, p, box, 0, rho[0], rho[1], dt, dt_ratio=1.0)
    assert ops.rel_l2(got, ref) < 1e-13
    with pytest.raises(Exception):
        _mp(oracle_mod, u, v, w, phi, box, r=-0.5)
