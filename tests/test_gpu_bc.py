"""-m gpu: non-periodic x / y -- the CUDA path through
flutas_plan_create_ex against the oracle's *_bc functions, element by element, relative L2 <= 1e-10.

  * flutas_poisson_solve for combinations of periodic (P), Neumann / wall (N) and Dirichlet (D) directions, on sizes
    that span partial column tiles, several row tiles, every radix tail along y and odd nz;
  * the whole step with walls (P / N directions), including the closed cavity (N, N, N);
  * a Dirichlet plan refuses the step; unsupported combinations are refused at plan creation.
"""
import numpy as np
import pytest
import torch

import paper_2204_08834_b200 as fl
import workloads as wl
from tests.gpu_util import gpu_step, plan_for, rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
P, N, D = 0, 1, 2


@pytest.mark.parametrize("bc,shape", [
    ((N, N, N), (12, 16, 32)), ((D, D, N), (9, 32, 64)), ((P, N, N), (20, 64, 32)), ((N, P, N), (7, 8, 16)),
    ((N, D, D), (33, 128, 128)), ((D, N, N), (16, 256, 16)), ((P, N, P), (16, 32, 64)), ((P, D, P), (8, 512, 16)),
    ((P, N, D), (5, 16, 8)), ((N, N, N), (64, 1024, 32)), ((P, D, N), (600, 8, 16)), ((P, P, D), (40, 16, 32)),
    ((D, D, D), (2, 8, 1024)), ((N, N, N), (444, 8, 256)), ((P, N, N), (300, 8, 16)), ((P, P, N), (257, 8, 16))])
def test_poisson_solve_with_boundary_conditions_matches_oracle(oracle_mod, bc, shape):
    rng = np.random.default_rng(sum(shape) + 100 * bc[0] + 10 * bc[1] + bc[2])
    rhs = rng.standard_normal(shape)
    if D not in bc:
        rhs -= rhs.mean()
    box = (2.0, 3.0, 1.0)
    want = oracle_mod.poisson_bc(rhs, box, bc)
    nz, ny, nx = shape
    plan = fl.Plan(nx, ny, nz, *box, bc[2], 1.0, 1.0, bc_x=bc[0], bc_y=bc[1])
    r = to_dev(rhs)
    out = torch.empty_like(r)
    plan.poisson_solve(r, out)
    torch.cuda.synchronize()
    got = out.cpu().numpy()
    assert rel_l2(got, want) <= TOL, (bc, shape, rel_l2(got, want))
    assert np.array_equal(r.cpu().numpy(), rhs)
    if D not in bc:
        assert abs(got.mean()) <= 1e-12 * max(1.0, np.abs(got).max())      # gauge R5
    names = plan.kernel_names
    assert ("z_singular" in names) == (bc[2] != P and D not in bc)
    plan.destroy()


@pytest.mark.parametrize("maker", [
    lambda: wl.random_case_bc(32, 16, 12, (N, N, N), 1000.0, 81),
    lambda: wl.random_case_bc(128, 32, 20, (N, N, N), 50.0, 82),          # the bulk-copy-fed RHS kernel with walls
    lambda: wl.random_case_bc(256, 64, 9, (P, N, N), 0.05, 83),
    lambda: wl.random_case_bc(64, 128, 33, (N, P, N), 10.0, 84),
    lambda: wl.random_case_bc(128, 64, 32, (P, N, P), 20.0, 85),
    lambda: wl.random_case_bc(16, 8, 2, (N, N, N), 3.0, 86),              # smallest walled box
    lambda: wl.cavity(64, 64, 16, 1.0),
    lambda: wl.cavity(256, 256, 64, 5.0),                                 # the closed cavity of PAPER.md:287, extruded
])
def test_step_with_walls_matches_oracle(oracle_mod, maker):
    W = maker()
    want = oracle_mod.projection_step_bc(*W.fields(), W.box, W.bc, W.rho1, W.rho2, W.dt)
    got = gpu_step(W)
    errs = {n: rel_l2(g, w_) for n, g, w_ in zip("uvwp", got, want)}
    print(W.name, {k: f"{v:.2e}" for k, v in errs.items()})
    for n, e in errs.items():
        assert e <= TOL, (W.name, n, e)
    if W.bc_x == N:
        assert np.array_equal(got[0][:, :, -1], W.u[:, :, -1])             # wall faces pass through untouched
    if W.bc_y == N:
        assert np.array_equal(got[1][:, -1, :], W.v[:, -1, :])
    if W.bc_z == N:
        assert np.array_equal(got[2][-1], W.w[-1])
    d0 = np.linalg.norm(oracle_mod.divergence_bc(W.u, W.v, W.w, W.box, W.bc))
    assert np.linalg.norm(oracle_mod.divergence_bc(*got[:3], W.box, W.bc)) <= 1e-11 * d0


def test_dirichlet_plans_solve_but_do_not_step_and_unsupported_combinations_are_refused():
    plan = fl.Plan(32, 16, 8, 1.0, 1.0, 1.0, N, 1.0, 2.0, bc_x=D, bc_y=N)
    d = [torch.zeros(8, 16, 32, dtype=torch.float64, device="cuda") for _ in range(6)]
    with pytest.raises(fl.FlutasError) as e:
        plan.projection_step(*d, 1e-3)
    assert e.value.code == 1 and "Dirichlet" in str(e.value)
    plan.destroy()
    for args, kw in (((32, 16, 8, 1.0, 1.0, 1.0, P, 1.0, 1.0), dict(bc_x=N)),          # non-periodic x needs non-periodic z
                     ((2048, 16, 8, 1.0, 1.0, 1.0, N, 1.0, 1.0), dict(bc_x=N)),
                     ((32, 2048, 8, 1.0, 1.0, 1.0, N, 1.0, 1.0), dict(bc_y=D)),
                     ((32, 16, 600, 1.0, 1.0, 1.0, N, 1.0, 1.0), dict(bc_x=N))):
        with pytest.raises(fl.FlutasError) as e:
            fl.Plan(*args, **kw)
        assert e.value.code == 2
        assert fl.binding.workspace_bytes(args[0], args[1], args[2], args[6], kw.get("bc_x", 0), kw.get("bc_y", 0)) == 0
