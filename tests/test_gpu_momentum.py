"""-m gpu: the momentum prediction of eq. (15) fused with the projection step
through flutas_momentum_rhs / flutas_time_step, against oracle.momentum_prediction followed by the oracle's projection,
element by element, relative L2 <= 1e-10 (the kernel-level outputs <= 1e-12)."""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests import np_ops as ops
from tests.gpu_util import plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER = 0
PHYS = dict(mu1=0.02, mu2=0.3, sigma=0.07, grav=(0.3, -0.2, -9.81))


def _case(maker, seed, with_kappa=True):
    W = maker()
    rng = np.random.default_rng(seed)
    kappa = rng.standard_normal(W.shape) if with_kappa else None
    m_old = [rng.standard_normal(W.shape) for _ in range(3)]
    return W, kappa, m_old


def _oracle_prediction(oracle, W, kappa, m_old, r):
    return oracle.momentum_prediction(W.u, W.v, W.w, W.phi, kappa, m_old, W.box, W.rho1, W.rho2, PHYS["mu1"], PHYS["mu2"],
                                      PHYS["sigma"] if kappa is not None else 0.0, PHYS["grav"], W.dt, r)


@pytest.mark.parametrize("maker,with_kappa,with_p,r", [
    (lambda: wl.random_case(32, 8, 8, PER, 10.0, 101), True, True, 1.0),          # one tile in x and y: the halo wraps onto the tile
    (lambda: wl.random_case(64, 32, 16, PER, 1000.0, 102), True, True, 0.6),
    (lambda: wl.random_case(128, 16, 64, PER, 0.05, 103), False, True, 1.0),      # more than one z chunk (kc = 32), no surface tension
    (lambda: wl.random_case(64, 8, 16, PER, 50.0, 104), True, False, 1.7),       # u** alone (no splitting terms)
])
def test_momentum_rhs_kernel_matches_oracle(oracle_mod, maker, with_kappa, with_p, r):
    W, kappa, m_old = _case(maker, 7, with_kappa)
    (us, vs, ws), m_new = _oracle_prediction(oracle_mod, W, kappa, m_old, r)
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    dk = None if kappa is None else to_dev(kappa)
    dmo = [to_dev(a) for a in m_old]
    dmn = [torch.empty_like(d[0]) for _ in range(3)]
    out = [torch.empty_like(d[0]) for _ in range(4)]
    plan.momentum_rhs(d[0], d[1], d[2], d[3], dk, d[4] if with_p else None, d[5] if with_p else None, dmo, dmn, PHYS["mu1"],
                      PHYS["mu2"], PHYS["sigma"] if with_kappa else 0.0, PHYS["grav"], W.dt, r, *out)
    torch.cuda.synchronize()
    for t, a in zip(d, W.fields()):
        assert np.array_equal(t.cpu().numpy(), a)                                 # inputs untouched
    for g, want in zip(dmn, m_new):
        assert rel_l2(g.cpu().numpy(), want) <= 1e-12
    rho0 = min(W.rho1, W.rho2)
    if with_p:
        # u' = u** + dt/rho0 (1 - rho0/rho_f) grad p_hat: independent numpy statement on top of the oracle's u**
        rf = ops.face_density(W.phi, W.rho1, W.rho2, False)
        gh = ops.grad((1.0 + r) * W.p - r * W.p_old, W.box, False)
        want_up = [a + W.dt / rho0 * (1.0 - rho0 / rr) * g for a, rr, g in zip((us, vs, ws), rf, gh)]
        want_rhs = oracle_mod.rhs(us, vs, ws, W.phi, W.p, W.p_old, W.box, PER, W.rho1, W.rho2, W.dt, dt_ratio=r)
    else:
        want_up = [us, vs, ws]
        want_rhs = rho0 / W.dt * ops.div(us, vs, ws, W.box, False)
    for g, want in zip(out[:3], want_up):
        assert rel_l2(g.cpu().numpy(), want) <= 1e-12
    assert rel_l2(out[3].cpu().numpy(), want_rhs) <= 1e-10      # rho0/dt div(.) of O(1) fields: cancellation, not a looser kernel
    plan.destroy()


@pytest.mark.parametrize("maker,r", [
    (lambda: wl.config1(), 1.0),
    (lambda: wl.random_case(64, 64, 32, PER, 100.0, 105), 0.8),
    (lambda: wl.config4(128, 50.0, 8, 0.05, 8), 1.0),
])
def test_time_step_matches_oracle_prediction_then_projection(oracle_mod, maker, r):
    W, kappa, m_old = _case(maker, 11)
    (us, vs, ws), m_new = _oracle_prediction(oracle_mod, W, kappa, m_old, r)
    want = oracle_mod.projection_step(us, vs, ws, W.phi, W.p, W.p_old, W.box, PER, W.rho1, W.rho2, W.dt, dt_ratio=r)
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    dk, dmo = to_dev(kappa), [to_dev(a) for a in m_old]
    dmn = [torch.empty_like(d[0]) for _ in range(3)]
    plan.time_step(d[0], d[1], d[2], d[3], dk, d[4], d[5], d[5], dmo, dmn, PHYS["mu1"], PHYS["mu2"], PHYS["sigma"], PHYS["grav"],
                   W.dt, r)                                                        # ping-pong: p^(n+1) over p^(n-1)
    torch.cuda.synchronize()
    got = (d[0], d[1], d[2], d[5])
    errs = {n: rel_l2(g.cpu().numpy(), w_) for n, g, w_ in zip("uvwp", got, want)}
    print(W.name, {k: f"{v:.2e}" for k, v in errs.items()})
    for n, e in errs.items():
        assert e <= TOL, (W.name, n, e)
    for g, w_ in zip(dmn, m_new):
        assert rel_l2(g.cpu().numpy(), w_) <= 1e-12
    assert np.array_equal(d[4].cpu().numpy(), W.p) and np.array_equal(d[3].cpu().numpy(), W.phi)
    un, vn, wn = (t.cpu().numpy() for t in got[:3])
    assert np.linalg.norm(ops.div(un, vn, wn, W.box, False)) <= 1e-11 * np.linalg.norm(ops.div(us, vs, ws, W.box, False))
    plan.destroy()


def test_momentum_tile_variants_agree(oracle_mod):
    """option "mom_ty16": tiles of 32 x 16 cells (default when ny is a multiple of 16) and of 32 x 8 give the same M, u', rhs"""
    W, kappa, m_old = _case(lambda: wl.random_case(64, 32, 40 - 8, PER, 20.0, 107), 13)
    (us, vs, ws), m_new = _oracle_prediction(oracle_mod, W, kappa, m_old, 1.0)
    res = []
    for ty16 in (1, 0):
        plan = plan_for(W)
        plan.set_option("mom_ty16", ty16)
        d = [to_dev(a) for a in W.fields()]
        dmn = [torch.empty_like(d[0]) for _ in range(3)]
        out = [torch.empty_like(d[0]) for _ in range(4)]
        plan.momentum_rhs(d[0], d[1], d[2], d[3], to_dev(kappa), d[4], d[5], [to_dev(a) for a in m_old], dmn, PHYS["mu1"],
                          PHYS["mu2"], PHYS["sigma"], PHYS["grav"], W.dt, 1.0, *out)
        torch.cuda.synchronize()
        for g, want in zip(dmn, m_new):
            assert rel_l2(g.cpu().numpy(), want) <= 1e-12, ty16
        res.append([t.cpu().numpy() for t in dmn + out])
        plan.destroy()
    for a, b in zip(*res):
        assert np.array_equal(a, b)                  # the same arithmetic per face, whatever the tile


def test_time_step_argument_errors():
    W = wl.random_case(64, 16, 8, 1, 2.0, 106)                                      # a wall-bounded plan
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    m = [torch.zeros_like(d[0]) for _ in range(6)]
    with pytest.raises(fl.FlutasError) as e:
        plan.time_step(d[0], d[1], d[2], d[3], None, d[4], d[5], d[4], m[:3], m[3:], 0.1, 0.1, 0.0, (0, 0, 0), 1e-3)
    assert e.value.code == 2
    plan.destroy()
    W = wl.config1()
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    m = [torch.zeros_like(d[0]) for _ in range(6)]
    with pytest.raises(fl.FlutasError) as e:
        plan.time_step(d[0], d[1], d[2], d[3], None, d[4], d[5], d[4], m[:3], [m[0], m[4], m[5]], 0.1, 0.1, 0.0, (0, 0, 0), 1e-3)
    assert e.value.code == 5                                                        # M(u^n) may not overwrite M(u^(n-1))
    with pytest.raises(fl.FlutasError) as e:
        plan.time_step(d[0], d[1], d[2], d[3], None, d[4], d[5], d[4], m[:3], m[3:], -0.1, 0.1, 0.0, (0, 0, 0), 1e-3)
    assert e.value.code == 1
    plan.destroy()


def test_first_step_with_dt_ratio_zero_is_an_euler_step(oracle_mod):
    """DESIGN.md R29: dt_ratio = 0 is the start-up step (f1 = 1, f2 = 0, p_hat = p^n).  M(u^(n-1)) and p^(n-1) are multiplied
    by zero: two different (finite) fillings give bit-identical results, equal to the oracle's step with r = 0."""
    W, kappa, m_old = _case(lambda: wl.random_case(64, 32, 16, PER, 100.0, 108), 17)
    (us, vs, ws), m_new = _oracle_prediction(oracle_mod, W, kappa, m_old, 0.0)
    want = oracle_mod.projection_step(us, vs, ws, W.phi, W.p, W.p_old, W.box, PER, W.rho1, W.rho2, W.dt, dt_ratio=0.0)
    plan = plan_for(W)
    res = []
    for fill in (0.0, 1.0e3):
        d = [to_dev(a) for a in W.fields()]
        d[5] = torch.full_like(d[5], fill)                                          # p^(n-1): does not exist yet
        dmo = [torch.full_like(d[0], -fill) for _ in range(3)]                      # M(u^(n-1)): neither
        dmn = [torch.empty_like(d[0]) for _ in range(3)]
        p_out = torch.empty_like(d[0])
        plan.time_step(d[0], d[1], d[2], d[3], to_dev(kappa), d[4], d[5], p_out, dmo, dmn, PHYS["mu1"], PHYS["mu2"], PHYS["sigma"],
                       PHYS["grav"], W.dt, 0.0)
        torch.cuda.synchronize()
        res.append([t.cpu().numpy() for t in (d[0], d[1], d[2], p_out, *dmn)])
    for a, b in zip(*res):
        assert np.array_equal(a, b)
    for n, g, w_ in zip("uvwp", res[0][:4], want):
        assert rel_l2(g, w_) <= TOL, (n, rel_l2(g, w_))
    for g, w_ in zip(res[0][4:], m_new):
        assert rel_l2(g, w_) <= 1e-12
    with pytest.raises(fl.FlutasError) as e:
        plan.time_step(*[to_dev(a) for a in W.fields()[:4]], None, *[to_dev(a) for a in (W.p, W.p_old, W.p)],
                       [to_dev(a) for a in m_old], [torch.empty(W.npts, dtype=torch.float64, device="cuda") for _ in range(3)],
                       0.1, 0.1, 0.0, (0, 0, 0), W.dt, -1.0)
    assert e.value.code == 1
    plan.destroy()
