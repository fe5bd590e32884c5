"""-m gpu: the time-stepping form of the boundary: variable time
step p_hat = (1 + r) p^n - r p^(n-1), p_out aliasing (in place / ping-pong / seventh array), and replay of a
step recorded into a CUDA graph -- all against the CPU oracle, relative L2 <= 1e-10."""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests.gpu_util import gpu_step, plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER, WALL = 0, 1


def _oracle(oracle, W, r):
    return oracle.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt, dt_ratio=r)


@pytest.mark.parametrize("maker,r", [
    (lambda: wl.config1(), 0.5), (lambda: wl.config1(), 1.0), (lambda: wl.config3(64, 32, 24), 1.7),
    (lambda: wl.random_case(128, 16, 32, PER, 50.0, 61), 2.0), (lambda: wl.random_case(32, 64, 33, WALL, 1000.0, 62), 0.25)])
def test_variable_dt_step_matches_oracle(oracle_mod, maker, r):
    W = maker()
    want = _oracle(oracle_mod, W, r)
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    plan.projection_step_ex(*d, d[4], W.dt, r)                 # p_out = p: in place
    torch.cuda.synchronize()
    for n, i, ref in zip("uvwp", (0, 1, 2, 4), want):
        assert rel_l2(d[i].cpu().numpy(), ref) <= TOL, (W.name, n, r)
    assert np.array_equal(d[5].cpu().numpy(), W.p_old) and np.array_equal(d[3].cpu().numpy(), W.phi)
    # kernel level: the right-hand side alone
    d = [to_dev(a) for a in W.fields()]
    out = torch.empty_like(d[0])
    plan.splitting_rhs_ex(*d, W.dt, r, out)
    torch.cuda.synchronize()
    want_rhs = oracle_mod.rhs(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt, dt_ratio=r)
    assert rel_l2(out.cpu().numpy(), want_rhs) <= 1e-13
    plan.destroy()


def test_unit_ratio_is_the_plain_step_bit_for_bit():
    W = wl.random_case(64, 32, 16, WALL, 10.0, 63)
    want = gpu_step(W)
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    plan.projection_step_ex(*d, d[4], W.dt, 1.0)
    torch.cuda.synchronize()
    for i, j in zip((0, 1, 2, 4), range(4)):
        assert np.array_equal(d[i].cpu().numpy(), want[j])
    plan.destroy()


@pytest.mark.parametrize("bc", [PER, WALL])
def test_p_out_ping_pong_and_seventh_array(oracle_mod, bc):
    W = wl.random_case(64, 32, 16, bc, 20.0, 64)
    want = gpu_step(W)
    plan = plan_for(W)
    # ping-pong: p^(n+1) lands in the p_old array, p^n is left untouched
    d = [to_dev(a) for a in W.fields()]
    plan.projection_step_ex(*d, d[5], W.dt, 1.0)
    torch.cuda.synchronize()
    for i, j in zip((0, 1, 2, 5), range(4)):
        assert np.array_equal(d[i].cpu().numpy(), want[j])
    assert np.array_equal(d[4].cpu().numpy(), W.p)
    # seventh array: p and p_old both untouched
    d = [to_dev(a) for a in W.fields()]
    out = torch.full_like(d[0], float("nan"))
    plan.projection_step_ex(*d, out, W.dt, 1.0)
    torch.cuda.synchronize()
    assert np.array_equal(out.cpu().numpy(), want[3])
    assert np.array_equal(d[4].cpu().numpy(), W.p) and np.array_equal(d[5].cpu().numpy(), W.p_old)
    # any other overlap is rejected
    with pytest.raises(fl.FlutasError) as e:
        plan.projection_step_ex(*d, d[0], W.dt, 1.0)
    assert e.value.code == 5
    with pytest.raises(fl.FlutasError) as e:
        plan.projection_step_ex(*d, d[4], W.dt, 0.0)
    assert e.value.code == 1
    plan.destroy()


def test_three_step_time_loop_with_pointer_swap_matches_oracle(oracle_mod):
    """A short time loop the way a solver would run it: variable dt, ping-pong pressure buffers, a fresh
    provisional velocity each step (here: the corrected velocity plus a seeded forcing)."""
    W = wl.random_case(32, 32, 16, WALL, 50.0, 65)
    rng = np.random.default_rng(66)
    forcing = [rng.uniform(-0.1, 0.1, W.shape) for _ in range(3)]
    for f in forcing:
        f[-1] = 0.0                                           # keeps w* = 0 on the top wall face
    dts = [1.0e-3, 1.3e-3, 0.8e-3]
    # oracle loop
    u, v, w, p, po = W.u, W.v, W.w, W.p, W.p_old
    dt_prev = dts[0]
    for dt, f in zip(dts, forcing):
        un, vn, wn, pn = oracle_mod.projection_step(u, v, w, W.phi, p, po, W.box, W.bc_z, W.rho1, W.rho2, dt,
                                                    dt_ratio=dt / dt_prev)
        u, v, w, po, p, dt_prev = un + f, vn + f, wn + f, p, pn, dt
    # GPU loop
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    du, dv, dw, dphi, dp, dpo = d
    dt_prev = dts[0]
    for dt, f in zip(dts, forcing):
        plan.projection_step_ex(du, dv, dw, dphi, dp, dpo, dpo, dt, dt / dt_prev)
        dp, dpo, dt_prev = dpo, dp, dt                        # swap: no copy of p
        ff = to_dev(f)
        du += ff; dv += ff; dw += ff
    torch.cuda.synchronize()
    for got, ref in ((du, u), (dv, v), (dw, w), (dp, p), (dpo, po)):
        assert rel_l2(got.cpu().numpy(), ref) <= TOL
    plan.destroy()


def test_step_replays_from_a_cuda_graph(oracle_mod):
    W = wl.config1()
    want = gpu_step(W)
    plan = plan_for(W)
    pristine = [to_dev(a) for a in W.fields()]
    d = [t.clone() for t in pristine]
    plan.projection_step(*d, W.dt)                            # warm-up outside capture (lazy module loading)
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        for t, src in zip(d, pristine):
            t.copy_(src)
        s.synchronize()
        g.capture_begin()
        plan.projection_step_ex(*d, d[4], W.dt, 1.0, stream=s.cuda_stream)
        g.capture_end()
    torch.cuda.synchronize()
    for rep in range(2):                                      # capture enqueued nothing; each replay is one step
        for t, src in zip(d, pristine):
            t.copy_(src)
        g.replay()
        torch.cuda.synchronize()
        for i, j in zip((0, 1, 2, 4), range(4)):
            assert np.array_equal(d[i].cpu().numpy(), want[j]), rep
    plan.destroy()
