"""-m gpu: every kernel variant a plan can select is held to the same oracle and the same bar.

  * z stage with walls: the one-pass shared-memory elimination (twisted factorisation, 1 or 2 solving warps) and the
    two-sweep kernel it replaced, on sizes that cover the predicated remainder loops (nz not a multiple of 8, odd nz,
    nz = 2, 3), whole register batches (nz >= 64) and the fall-back for nz > 512;
  * transform along y at ny = 1024: the 16 x 8 x 8 register-resident kernel and the 4-column fft_tma1 path;
  * plane-chunked launch order (one stream, and three internal streams): bit for bit the plain order.
"""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests.gpu_util import plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER, WALL = 0, 1


def _solve(plan, rhs):
    r = to_dev(rhs)
    out = torch.empty_like(r)
    plan.poisson_solve(r, out)
    torch.cuda.synchronize()
    return out.cpu().numpy()


@pytest.mark.parametrize("shape", [(2, 8, 16), (3, 8, 16), (7, 16, 32), (24, 32, 64), (37, 16, 32), (64, 16, 32),
                                   (100, 16, 32), (130, 8, 16), (300, 16, 32), (512, 8, 16), (600, 8, 16)])
def test_wall_z_stage_variants_match_oracle(oracle_mod, shape):
    rng = np.random.default_rng(7 + sum(shape))
    rhs = rng.standard_normal(shape)
    rhs -= rhs.mean()
    box = (2.0, 3.0, 1.0)
    want = oracle_mod.poisson(rhs, box, WALL)
    nz, ny, nx = shape
    plan = fl.Plan(nx, ny, nz, *box, WALL, 1.0, 1.0)
    got = {"default": _solve(plan, rhs)}
    if nz <= 512:                                 # the one-pass kernel exists for this size: try both warp counts
        for warps in (1, 2):
            plan.set_option("thomas", 1)
            plan.set_option("thomas_warps", warps)
            got[f"one-pass, {warps} warp(s)"] = _solve(plan, rhs)
    else:
        with pytest.raises(fl.FlutasError):
            plan.set_option("thomas", 1)
    plan.set_option("thomas", 0)
    got["two sweeps"] = _solve(plan, rhs)
    for name, p in got.items():
        assert rel_l2(p, want) <= TOL, (shape, name, rel_l2(p, want))
        assert abs(p.mean()) <= 1e-12 * max(1.0, np.abs(p).max()), (shape, name)     # gauge R5
    plan.destroy()


@pytest.mark.parametrize("nz,nx,bc", [(8, 16, PER), (4, 16, WALL), (16, 64, WALL)])
def test_y_transform_of_length_1024_variants_match_oracle(oracle_mod, nz, nx, bc):
    shape = (nz, 1024, nx)
    rng = np.random.default_rng(11 + nz + nx)
    rhs = rng.standard_normal(shape)
    rhs -= rhs.mean()
    box = (2.0, 3.0, 1.0)
    want = oracle_mod.poisson(rhs, box, bc)
    plan = fl.Plan(nx, 1024, nz, *box, bc, 1.0, 1.0)
    a = _solve(plan, rhs)                         # default: 16 x 8 x 8 kernel
    plan.set_option("y16", 0)
    b = _solve(plan, rhs)                         # 4-column path (different storage order along y)
    plan.set_option("y16", 1)
    c = _solve(plan, rhs)
    assert rel_l2(a, want) <= TOL and rel_l2(b, want) <= TOL
    assert np.array_equal(a, c)                   # switching back and forth rebuilds the same tables
    plan.destroy()


def test_y16_is_refused_for_other_lengths():
    plan = fl.Plan(32, 512, 8, 1.0, 1.0, 1.0, PER, 1.0, 1.0)
    with pytest.raises(fl.FlutasError):
        plan.set_option("y16", 1)
    plan.destroy()


@pytest.mark.parametrize("maker", [lambda: wl.random_case(128, 32, 32, PER, 50.0, 21),
                                   lambda: wl.random_case(128, 16, 20, WALL, 1000.0, 22)])
def test_chunked_launch_order_is_bitwise_the_plain_order(maker):
    W = maker()
    plan = plan_for(W)

    def run():
        d = [to_dev(x) for x in W.fields()]
        plan.projection_step(*d, W.dt)
        torch.cuda.synchronize()
        return [d[i].cpu().numpy() for i in (0, 1, 2, 4)]

    ref = run()
    for chunk, overlap in ((1, 0), (5, 0), (8, 1), (3, 1), (W.nz, 1)):
        plan.set_option("chunk", chunk)
        plan.set_option("overlap", overlap)
        got = run()
        for g, r in zip(got, ref):
            assert np.array_equal(g, r), (W.name, chunk, overlap)
    plan.destroy()


def test_chunked_multi_stream_step_replays_from_a_cuda_graph():
    """the fork / join over the plan's internal streams is capturable: one graph launch = one step, bit for bit"""
    W = wl.random_case(128, 16, 32, PER, 10.0, 23)
    plan = plan_for(W)
    pristine = [to_dev(a) for a in W.fields()]
    d = [t.clone() for t in pristine]
    plan.projection_step(*d, W.dt)
    torch.cuda.synchronize()
    want = [d[i].cpu().numpy() for i in (0, 1, 2, 4)]
    plan.set_option("chunk", 8)
    plan.set_option("overlap", 1)
    for t, src in zip(d, pristine):
        t.copy_(src)
    plan.projection_step(*d, W.dt)                            # creates the internal streams and events outside capture
    torch.cuda.synchronize()
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        s.synchronize()
        g.capture_begin()
        plan.projection_step_ex(*d, d[4], W.dt, 1.0, stream=s.cuda_stream)
        g.capture_end()
    torch.cuda.synchronize()
    for rep in range(2):
        for t, src in zip(d, pristine):
            t.copy_(src)
        g.replay()
        torch.cuda.synchronize()
        for i, ref in zip((0, 1, 2, 4), want):
            assert np.array_equal(d[i].cpu().numpy(), ref), rep
    plan.destroy()


def test_plans_release_their_device_memory():
    """create / use / destroy in a loop (every variant that allocates lazily touched once): free device memory returns"""
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free0, _ = torch.cuda.mem_get_info()
    for rep in range(6):
        for bc, nz in ((PER, 64), (WALL, 50)):
            W = wl.random_case(128, 64, nz, bc, 3.0, 30 + rep)
            plan = plan_for(W)
            if bc == WALL:
                plan.set_option("thomas", rep % 2)          # the two-sweep form allocates c' on first use
            plan.set_option("chunk", 8 * (rep % 2))
            plan.set_option("overlap", rep % 2)             # internal streams and events
            plan.set_timing(rep % 2 == 0)
            d = [to_dev(x) for x in W.fields()]
            plan.projection_step(*d, W.dt)
            torch.cuda.synchronize()
            assert torch.isfinite(d[4]).all()
            plan.destroy()
            del d
    torch.cuda.synchronize()
    torch.cuda.empty_cache()
    free1, _ = torch.cuda.mem_get_info()
    assert free0 - free1 < 64 * 2**20, (free0, free1)
