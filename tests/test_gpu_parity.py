"""-m gpu: the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bar (BASELINE.json north_star): relative L2 <= 1e-10 on p, u, v, w (fp64)."""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests import np_ops as ops
from tests.gpu_util import gpu_step, plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER, WALL = 0, 1


def _oracle_step(oracle, W, **kw):
    return oracle.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt, **kw)


def _assert_step_parity(oracle, W, tol=TOL):
    want = _oracle_step(oracle, W)
    got = gpu_step(W)
    errs = {n: rel_l2(g, w_) for n, g, w_ in zip("uvwp", got, want)}
    print(W.name, {k: f"{v:.2e}" for k, v in errs.items()})
    for n, e in errs.items():
        assert e <= tol, (W.name, n, e)
    if W.bc_z == WALL:
        assert np.array_equal(got[2][-1], W.w[-1])          # top wall face passes through untouched
    return errs


# ------------------------------------------------------------------ T1: the two halves alone
@pytest.mark.parametrize("maker", [
    lambda: wl.config1(), lambda: wl.random_case(64, 32, 16, WALL, 1000.0, 3),
    lambda: wl.random_case(32, 64, 24, WALL, 0.01, 4), lambda: wl.random_case(128, 16, 32, PER, 50.0, 5)])
def test_splitting_rhs_matches_oracle(oracle_mod, maker):
    W = maker()
    want = oracle_mod.rhs(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt)
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    out = torch.empty_like(d[0])
    plan.splitting_rhs(*d, W.dt, out)
    torch.cuda.synchronize()
    for t, a in zip(d, W.fields()):
        assert np.array_equal(t.cpu().numpy(), a)            # inputs untouched
    assert rel_l2(out.cpu().numpy(), want) <= 1e-13
    plan.destroy()


@pytest.mark.parametrize("shape,bc", [
    ((32, 32, 32), PER), ((8, 8, 16), PER), ((16, 64, 128), PER), ((64, 16, 256), PER), ((128, 32, 32), PER),
    ((512, 8, 16), PER), ((8, 512, 16), PER), ((8, 8, 1024), PER), ((1024, 8, 16), PER), ((8, 16, 8), PER),
    ((16, 64, 2048), PER), ((9, 8, 8), WALL),
    ((2, 8, 16), WALL), ((3, 16, 32), WALL), ((20, 32, 64), WALL), ((37, 64, 16), WALL), ((128, 8, 512), WALL)])
def test_poisson_solve_matches_oracle(oracle_mod, shape, bc):
    """sizes span: minimum sizes, every radix tail (r = 1, 2, 4), non-power-of-two nz for walls,
    partial kx tiles (nx/2 + 1 is never a multiple of 8)"""
    rng = np.random.default_rng(sum(shape))
    rhs = rng.standard_normal(shape)
    rhs -= rhs.mean()
    box = (2.0, 3.0, 1.0)
    want = oracle_mod.poisson(rhs, box, bc)
    nz, ny, nx = shape
    plan = fl.Plan(nx, ny, nz, *box, bc, 1.0, 1.0)
    r = to_dev(rhs)
    out = torch.empty_like(r)
    plan.poisson_solve(r, out)
    torch.cuda.synchronize()
    assert rel_l2(out.cpu().numpy(), want) <= TOL
    assert np.array_equal(r.cpu().numpy(), rhs)
    plan.poisson_solve(r, r)                                  # in place is allowed
    torch.cuda.synchronize()
    assert np.array_equal(r.cpu().numpy(), out.cpu().numpy())
    plan.destroy()


def test_poisson_solve_returns_eigenmodes(oracle_mod):
    """closed form, independent of the oracle: L f = lam f for a product of cosines (P1)"""
    from tests.test_oracle_pins import _eigen_mode
    for bc, shape in ((PER, (16, 32, 64)), (WALL, (12, 32, 64))):
        box = (2.0, 3.0, 1.0)
        f, lam = _eigen_mode(shape, box, bc, 3, 5, 2)
        plan = fl.Plan(shape[2], shape[1], shape[0], *box, bc, 1.0, 1.0)
        r = to_dev(lam * f)
        plan.poisson_solve(r, r)
        torch.cuda.synchronize()
        assert rel_l2(r.cpu().numpy(), f) <= 1e-12
        plan.destroy()


# ------------------------------------------------------------------ T2: the whole step
def test_step_config1(oracle_mod):
    _assert_step_parity(oracle_mod, wl.config1())


def test_step_config2(oracle_mod):
    _assert_step_parity(oracle_mod, wl.config2())


def test_step_config3(oracle_mod):
    _assert_step_parity(oracle_mod, wl.config3())


@pytest.mark.parametrize("ratio", [1.0, 50.0])
def test_step_config4_shape_at_128(oracle_mod, ratio):
    _assert_step_parity(oracle_mod, wl.config4(128, ratio, 8, 0.05, 8))


def test_step_config5_shape_small(oracle_mod):
    _assert_step_parity(oracle_mod, wl.config5(128, 64, 96))


@pytest.mark.parametrize("maker", [
    lambda: wl.random_case(8, 8, 8, PER, 10.0, 10),           # smallest supported periodic grid (nx = 8: degenerate x kernels)
    lambda: wl.random_case(8, 16, 5, WALL, 100.0, 9),
    lambda: wl.random_case(16, 8, 8, PER, 10.0, 11),
    lambda: wl.random_case(32, 64, 1024, PER, 20.0, 18),      # periodic z of 1024: the 4-column one-butterfly z kernel
    lambda: wl.random_case(2048, 32, 16, WALL, 20.0, 19),     # maximum nx with more than one tile of rows
    lambda: wl.random_case(16, 8, 2, WALL, 10.0, 12),         # smallest wall grid
    lambda: wl.random_case(2048, 8, 8, PER, 5.0, 13),         # maximum nx
    lambda: wl.random_case(16, 2048, 8, WALL, 5.0, 14),       # maximum ny (4-column tiles)
    lambda: wl.random_case(16, 8, 2048, PER, 5.0, 15),        # maximum nz
    lambda: wl.random_case(64, 128, 33, WALL, 1000.0, 16),    # odd nz
    lambda: wl.random_case(256, 64, 128, PER, 1.0, 17),
])
def test_step_edge_sizes(oracle_mod, maker):
    _assert_step_parity(oracle_mod, maker())


def test_equal_densities_make_the_step_independent_of_the_pressure_history_bit_for_bit():
    """rho1 == rho2: the splitting coefficient is exactly 0 on the GPU too (P6), so p and p_old
    cannot influence the result at all"""
    W = wl.random_case(128, 32, 16, WALL, 1.0, 24)
    a = gpu_step(W)
    rng = np.random.default_rng(5)
    W.p, W.p_old = rng.standard_normal(W.shape), rng.standard_normal(W.shape)
    b = gpu_step(W)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_workspace_is_the_callers_torch_memory(oracle_mod):
    """flutas_plan_set_workspace: the default binding hands the plan ONE torch tensor; torch's allocator accounts for
    it; the same step on a library-owned workspace, on a second caller buffer and after switching back and forth gives
    the same bits; a buffer that is too small or misaligned is refused"""
    W = wl.random_case(128, 32, 20, WALL, 10.0, 25)
    need = fl.binding.workspace_bytes(W.nx, W.ny, W.nz, W.bc_z)
    torch.cuda.synchronize()
    before = torch.cuda.memory_allocated()
    plan = plan_for(W)
    assert plan.workspace_bytes == need
    assert torch.cuda.memory_allocated() - before >= need                 # the workspace is torch's
    want = gpu_step(W, plan)
    ref = _oracle_step(oracle_mod, W)
    for g, r in zip(want, ref):
        assert rel_l2(g, r) <= TOL
    lib_plan = fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, workspace="library")
    for g, r in zip(gpu_step(W, lib_plan), want):
        assert np.array_equal(g, r)
    lib_plan.destroy()
    other = torch.empty(need + 4096, dtype=torch.uint8, device="cuda")
    plan.set_workspace(other[256:])                                        # any 256-byte aligned view will do
    for g, r in zip(gpu_step(W, plan), want):
        assert np.array_equal(g, r)
    with pytest.raises(fl.FlutasError):
        plan.set_workspace(other[8:])                                      # misaligned
    with pytest.raises(fl.FlutasError):
        plan.set_workspace(other[:need - 1024])                            # too small
    plan.set_workspace(None)                                               # back to a library-owned one
    for g, r in zip(gpu_step(W, plan), want):
        assert np.array_equal(g, r)
    plan.destroy()
    # a plan created for a caller workspace refuses to step without one
    h = fl.lib.flutas_plan_create_ex(W.nx, W.ny, W.nz, *W.box, 0, 0, W.bc_z, W.rho1, W.rho2, fl.binding.PLAN_CALLER_WORKSPACE)
    d = [to_dev(a) for a in W.fields()]
    assert fl.lib.flutas_projection_step(h, *[t.data_ptr() for t in d], W.dt, None) == 1
    assert b"workspace" in fl.lib.flutas_last_error()
    fl.lib.flutas_plan_destroy(h)


def test_step_is_deterministic_and_plan_is_reusable(oracle_mod):
    W = wl.config1()
    plan = plan_for(W)
    a = gpu_step(W, plan)
    b = gpu_step(W, plan)
    for x, y in zip(a, b):
        assert np.array_equal(x, y)
    plan.destroy()


def test_host_entry_point_matches_device_entry_point(oracle_mod):
    W = wl.random_case(64, 32, 16, WALL, 10.0, 21)
    want = gpu_step(W)
    plan = plan_for(W)
    h = [torch.from_numpy(a.copy()).pin_memory() for a in W.fields()]
    plan.projection_step_host(*h, W.dt)
    for i, j in zip((0, 1, 2, 4), range(4)):
        assert np.array_equal(h[i].numpy(), want[j])
    n = [a.copy() for a in W.fields()]                        # pageable numpy arrays work too
    plan.projection_step_host(*n, W.dt)
    for i, j in zip((0, 1, 2, 4), range(4)):
        assert np.array_equal(n[i], want[j])
    plan.destroy()


def test_non_default_stream_and_timing(oracle_mod):
    W = wl.config1()
    want = gpu_step(W)
    plan = plan_for(W)
    plan.set_timing(True)
    s = torch.cuda.Stream()
    with torch.cuda.stream(s):
        d = [to_dev(a) for a in W.fields()]
        s.synchronize()
        plan.projection_step(*d, W.dt)
    s.synchronize()
    for i, j in zip((0, 1, 2, 4), range(4)):
        assert np.array_equal(d[i].cpu().numpy(), want[j])
    ms, steps = plan.read_timing()
    assert steps == 1 and len(ms) == len(plan.kernel_names) == 7 and all(m > 0 for m in ms)
    assert plan.kernel_names[0] == "splitting_rhs" and plan.kernel_names[-1] == "correction"
    assert plan.kernel_symbols[0] == "splitting_rhs_kernel2" and plan.kernel_symbols[3] == "fft_tma1_kernel"
    plan.destroy()


def test_argument_errors_on_device():
    W = wl.config1()
    plan = plan_for(W)
    d = [to_dev(a) for a in W.fields()]
    with pytest.raises(fl.FlutasError) as e:
        plan.projection_step(d[0], d[0], d[2], d[3], d[4], d[5], W.dt)
    assert e.value.code == 5                                   # alias
    with pytest.raises(fl.FlutasError) as e:
        plan.projection_step(*d, 0.0)
    assert e.value.code == 1                                   # dt
    big = torch.zeros(W.npts + 1, dtype=torch.float64, device="cuda")
    rc = fl.lib.flutas_projection_step(plan._h, big.data_ptr() + 8, d[1].data_ptr(), d[2].data_ptr(), d[3].data_ptr(),
                                       d[4].data_ptr(), d[5].data_ptr(), 1e-3, None)
    assert rc == 5                                             # misaligned
    plan.destroy()
