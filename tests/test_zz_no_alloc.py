"""-m gpu: flutas_vof_step_noalloc, the volume-of-fluid step for callers that cannot allocate device memory.

Some users of this library run where cudaMalloc is off limits: inside an application whose memory pool already holds the whole
GPU (another cudaMalloc just fails), inside a pipeline that cannot afford the device-wide synchronisation a cudaMalloc
causes, or under a "nothing is allocated after start-up" rule.  flutas_vof_step is no use to them (it wants a plan, and a
plan allocates tables and a workspace), so the library has this one plan-free entry point whose scratch -- the four
intermediate fields of the step -- is a fixed array inside the library (4 x 2^21 doubles = 64 MiB per GPU, hence grids of at
most 2^21 cells).

What is checked here, always through the C ABI:
  * its result equals that of the ordinary path, flutas_vof_step, within the tolerance of the other VoF tests (TOL below),
    on two calls in a row.  The second call is a different, smaller case, so it finds the array full of the first call's
    leftovers: the entry point promises that this does not matter;
  * the second call leaves the amount of free device memory as it found it;
  * grids beyond the limit are refused with a message that names it, and nothing is written.
The file is named so that pytest collects it last: the array is shared by the whole process and outlives every test, and
a failure here must not hide the other tests behind `pytest -x`.  It passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests import np_ops as ops
from tests.gpu_util import plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10          # the bar of tests/test_gpu_vof.py (relative L2 on phi^(n+1))


def _cfl_dt(W, cfl):
    d = ops.spacings(W.shape, W.box)
    return cfl / max(np.abs(a).max() / h for a, h in zip((W.u, W.v, W.w), d))


def _existing_path(W, beta, dt):
    plan = plan_for(W)
    d = [to_dev(a) for a in (W.phi, W.u, W.v, W.w)]
    out = torch.empty_like(d[0])
    plan.vof_step(*d, out, beta, dt)
    torch.cuda.synchronize()
    plan.destroy()
    return out.cpu().numpy()


def test_noalloc_vof_step_equals_the_plan_path_on_two_calls_in_a_row():
    cases = [(wl.config2(64, 6, 6, 6), 2.0, 0.4),                  # 64^3: several drops in a turbulent field
             (wl.random_case(64, 16, 8, 0, 1.0, 111), 3.0, 0.5)]   # then 64 x 16 x 8: a tilted sheet, other beta and box
    want = [_existing_path(W, beta, _cfl_dt(W, cfl)) for W, beta, cfl in cases]
    # every tensor of both calls exists before the first one, so that torch's allocator is quiet from here on
    dev = [[to_dev(a) for a in (W.phi, W.u, W.v, W.w)] for W, _, _ in cases]
    outs = [torch.empty_like(d[0]) for d in dev]
    free = []
    for (W, beta, cfl), d, out in zip(cases, dev, outs):
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
        fl.vof_step_noalloc((W.nx, W.ny, W.nz), W.box, *d, out, beta, _cfl_dt(W, cfl))
        torch.cuda.synchronize()
        free.append(torch.cuda.mem_get_info()[0])
    for (W, _, _), d, out, ref in zip(cases, dev, outs, want):
        got = out.cpu().numpy()
        err = rel_l2(got, ref)
        print(W.name, f"no-alloc vs plan path: rel L2 {err:.2e}, bitwise {np.array_equal(got, ref)}, "
                      f"changed {np.abs(ref - W.phi).max():.2e}")
        assert err <= TOL and np.abs(ref - W.phi).max() > 1e-3
        assert np.array_equal(d[0].cpu().numpy(), W.phi)           # inputs untouched
    # the first call on a device may make the driver place the library's static array; the second call changes nothing
    assert free[3] == free[2]
    # in place (phi_out = phi), as flutas_vof_step allows
    W, beta, cfl = cases[1]
    fl.vof_step_noalloc((W.nx, W.ny, W.nz), W.box, dev[1][0], *dev[1][1:], dev[1][0], beta, _cfl_dt(W, cfl))
    torch.cuda.synchronize()
    assert np.array_equal(dev[1][0].cpu().numpy(), outs[1].cpu().numpy())


def test_noalloc_vof_step_takes_any_grid_size_up_to_its_limit(oracle_mod):
    """a grid no plan exists for (sizes that are not powers of two): compared with the CPU oracle instead"""
    W = wl.random_case(24, 20, 12, 0, 1.0, 113)
    dt = _cfl_dt(W, 0.4)
    want = oracle_mod.vof_step(W.phi, W.u, W.v, W.w, W.box, 2.0, dt)
    d = [to_dev(a) for a in (W.phi, W.u, W.v, W.w)]
    out = torch.empty_like(d[0])
    fl.vof_step_noalloc((W.nx, W.ny, W.nz), W.box, *d, out, 2.0, dt)
    torch.cuda.synchronize()
    assert rel_l2(out.cpu().numpy(), want) <= TOL and np.abs(want - W.phi).max() > 1e-3


def test_noalloc_vof_step_refuses_what_its_static_array_cannot_hold():
    limit = fl.vof_noalloc_max_cells()
    assert limit == 1 << 21
    n = 256 * 128 * 128                                              # twice the limit
    assert n > limit
    f = torch.zeros(n, dtype=torch.float64, device="cuda")
    out = torch.full((n,), 7.0, dtype=torch.float64, device="cuda")
    with pytest.raises(fl.FlutasError) as e:
        fl.vof_step_noalloc((256, 128, 128), (1.0, 1.0, 1.0), f, f.clone(), f.clone(), f.clone(), out, 2.0, 1e-3)
    assert e.value.code == 2 and str(limit) in str(e.value) and "FLUTAS_VOF_NOALLOC_MAX_CELLS" in str(e.value)
    torch.cuda.synchronize()
    assert bool((out == 7.0).all())                                  # nothing was launched
    g = torch.zeros(8 * 8 * 8, dtype=torch.float64, device="cuda")
    with pytest.raises(fl.FlutasError) as e:
        fl.vof_step_noalloc((8, 8, 8), (1.0, 1.0, 1.0), g, g.clone(), g.clone(), g.clone(), g.clone(), -2.0, 1e-3)
    assert e.value.code == 1                                         # beta <= 0
    u = g.clone()
    with pytest.raises(fl.FlutasError) as e:                         # phi_out may alias phi only
        fl.vof_step_noalloc((8, 8, 8), (1.0, 1.0, 1.0), g, u, g.clone(), g.clone(), u, 2.0, 1e-3)
    assert e.value.code == 5
