"""-m gpu: one step of the MTHINC volume-of-fluid method (Appendix A) through
flutas_vof_step against oracle.vof_step, element by element.  Bar: relative L2 <= 1e-10 on phi^(n+1) (the two sides
find the reconstruction offset d by different algorithms -- bisection on the integral constraint vs the paper's quartic --
and the integer decisions, flat / not flat and the direction of exact integration, are taken on bit-identical normals)."""
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


def _cfl_dt(W, cfl):
    d = ops.spacings(W.shape, W.box)
    return cfl / max(np.abs(a).max() / h for a, h in zip((W.u, W.v, W.w), d))


def _gpu_vof(plan, phi, W, beta, dt, steps=1, in_place=False):
    d = [to_dev(a) for a in (phi, W.u, W.v, W.w)]
    out = d[0] if in_place else torch.empty_like(d[0])
    cur = d[0]
    for _ in range(steps):
        plan.vof_step(cur, d[1], d[2], d[3], out, beta, dt)
        cur = out
    torch.cuda.synchronize()
    if not in_place:
        assert np.array_equal(d[0].cpu().numpy(), phi) or steps > 1
    return out.cpu().numpy()


@pytest.mark.parametrize("maker,beta,cfl", [
    (lambda: wl.config1(), 2.0, 0.3),                                   # one drop, white-noise velocity (not solenoidal)
    (lambda: wl.config2(64, 6, 6, 6), 2.0, 0.4),                        # emulsion-shaped: several drops in a turbulent field
    (lambda: wl.config2(32, 3, 4, 4), 3.0, 0.2),
    (lambda: wl.random_case(64, 16, 8, PER, 1.0, 111), 2.0, 0.5),       # a tilted sheet crossing the periodic boundary
    (lambda: wl.config4(128, 50.0, 8, 0.05, 8), 2.0, 0.3),
])
def test_vof_step_matches_oracle(oracle_mod, maker, beta, cfl):
    W = maker()
    dt = _cfl_dt(W, cfl)
    want = oracle_mod.vof_step(W.phi, W.u, W.v, W.w, W.box, beta, dt)
    plan = plan_for(W)
    got = _gpu_vof(plan, W.phi, W, beta, dt)
    err = rel_l2(got, want)
    print(W.name, f"phi: rel L2 {err:.2e}, max abs {np.abs(got - want).max():.2e}, changed {np.abs(want - W.phi).max():.2e}")
    assert err <= TOL and np.abs(want - W.phi).max() > 1e-3
    same = _gpu_vof(plan, W.phi, W, beta, dt, in_place=True)           # phi_out may be phi
    assert np.array_equal(same, got)
    plan.destroy()


def test_three_steps_and_conservation(oracle_mod):
    W = wl.config2(32, 3, 4, 4)
    # make the velocity discretely solenoidal: one constant-density projection by the oracle
    W.u, W.v, W.w, _ = oracle_mod.projection_step(W.u, W.v, W.w, W.phi, W.p, W.p_old, W.box, PER, 1.0, 1.0, W.dt)
    dt = _cfl_dt(W, 0.3)
    want = W.phi
    for _ in range(3):
        want = oracle_mod.vof_step(want, W.u, W.v, W.w, W.box, 2.0, dt)
    plan = plan_for(W)
    got = _gpu_vof(plan, W.phi, W, 2.0, dt, steps=3, in_place=True)
    assert rel_l2(got, want) <= TOL
    assert abs(got.sum() - W.phi.sum()) <= 1e-12 * W.phi.sum()         # mass conserved to machine precision
    plan.destroy()


def test_vof_argument_errors():
    W = wl.random_case(32, 16, 8, 1, 2.0, 112)
    plan = plan_for(W)
    d = [to_dev(a) for a in (W.phi, W.u, W.v, W.w)]
    with pytest.raises(fl.FlutasError) as e:
        plan.vof_step(*d, torch.empty_like(d[0]), 2.0, 1e-3)
    assert e.value.code == 2
    plan.destroy()
    W = wl.config1()
    plan = plan_for(W)
    d = [to_dev(a) for a in (W.phi, W.u, W.v, W.w)]
    with pytest.raises(fl.FlutasError) as e:
        plan.vof_step(*d, d[1], 2.0, 1e-3)                              # phi_out may only alias phi
    assert e.value.code == 5
    with pytest.raises(fl.FlutasError) as e:
        plan.vof_step(*d, d[0], -2.0, 1e-3)
    assert e.value.code == 1
    plan.destroy()


def test_vof_step_with_nearly_grid_aligned_interfaces(oracle_mod):
    """two sheets normal to z whose height varies by 1e-10 ... 1e-6 of a cell along x and y: the normals have x, y components
    of 1e-11 ... 1e-7, so the sweeps along x and y integrate with |alpha| tiny but above the flat-normal cut-off -- the
    range where a difference of logarithms divided by alpha loses its digits (both sides now use cancellation-free forms,
    each its own; oracle pin V9)"""
    nx, ny, nz = 64, 32, 32
    W = wl.random_case(nx, ny, nz, PER, 1.0, 114)
    z, y, x = np.meshgrid(np.arange(nz) + 0.5, np.arange(ny) + 0.5, np.arange(nx) + 0.5, indexing="ij")
    amp = 10.0 ** (-10.0 + 4.0 * (y // 8) / 3.0)                       # 1e-10, 2e-9, 5e-8, 1e-6 in four bands of y
    ripple = amp * (np.sin(2 * np.pi * x / nx) + 0.5 * np.cos(2 * np.pi * 3 * y / ny))
    W.phi = 0.5 * (np.tanh((z - 9.3 + ripple) / 1.2) - np.tanh((z - 22.6 - ripple) / 1.2))
    dt = _cfl_dt(W, 0.4)
    n, _, flat = oracle_mod.vof_reconstruct(W.phi, 2.0)
    small = (flat == 0) & (np.abs(n[..., 0]) > 1e-12) & (np.abs(n[..., 0]) < 1e-6)
    assert small.sum() > 1000                                           # the case does exercise that range
    want = oracle_mod.vof_step(W.phi, W.u, W.v, W.w, W.box, 2.0, dt)
    plan = plan_for(W)
    got = _gpu_vof(plan, W.phi, W, 2.0, dt)
    err = rel_l2(got, want)
    print(f"nearly aligned: rel L2 {err:.2e}, max abs {np.abs(got - want).max():.2e}, cells with 1e-12 < |n_x| < 1e-6: {small.sum()}")
    assert err <= 1e-12 and np.abs(got - want).max() <= 1e-11
    plan.destroy()
