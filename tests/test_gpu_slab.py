"""-m gpu: the step on a z-slab decomposition (flutas_slab_*), all ranks of the decomposition
driven phase by phase on ONE device, against the CPU oracle on the assembled fields.  The oracle is the plain one-domain
step: the decomposition must not change the result (relative L2 <= 1e-10 per field, the bar of every parity test)."""
import numpy as np
import pytest
import torch

import workloads as wl
from paper_2204_08834_b200 import binding, slab
from tests.gpu_util import rel_l2, to_dev

pytestmark = pytest.mark.gpu
TOL = 1e-10
PER, WALL = 0, 1


def _slab_step(W, n_ranks, p_out_mode="p"):
    periodic = W.bc_z == PER
    parts = [wl.slab_split(a, n_ranks, periodic) for a in W.fields()]            # [field][rank]
    grp = slab.SlabGroup(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, n_ranks)
    dev = [[to_dev(parts[f][r]) for f in range(6)] for r in range(n_ranks)]
    p_out = None
    if p_out_mode == "p_old":
        p_out = [d[5] for d in dev]
    elif p_out_mode == "new":
        p_out = [torch.full_like(d[4], float("nan")) for d in dev]
    grp.step(dev, W.dt, 1.0, p_out)
    torch.cuda.synchronize()
    res_p = [d[4] for d in dev] if p_out is None else p_out
    out = [wl.slab_gather([dev[r][f].cpu().numpy() for r in range(n_ranks)]) for f in (0, 1, 2)]
    p_loc = [t.cpu().numpy() for t in res_p]
    out.append(wl.slab_gather(p_loc))
    grp.destroy()
    return out, p_loc


@pytest.mark.parametrize("shape,bc,ratio,n_ranks", [
    ((128, 16, 32), PER, 10.0, 1), ((128, 16, 32), PER, 10.0, 2), ((128, 16, 32), PER, 10.0, 4),
    ((128, 32, 64), PER, 50.0, 8), ((256, 8, 16), PER, 1.0, 8), ((128, 16, 16), PER, 3.0, 16),
    ((128, 16, 32), WALL, 1000.0, 1), ((128, 16, 32), WALL, 1000.0, 2), ((128, 16, 32), WALL, 1000.0, 4),
    ((256, 32, 64), WALL, 1.2, 8), ((128, 8, 8), WALL, 5.0, 8), ((128, 64, 256), WALL, 20.0, 2),
    # lines of 1024 (four-column tiles of the scatter variants): along y, and along z
    ((128, 1024, 16), WALL, 7.0, 4), ((128, 8, 1024), PER, 2.0, 4), ((1024, 16, 8), PER, 30.0, 2)])
def test_slab_step_matches_oracle(oracle_mod, shape, bc, ratio, n_ranks):
    nx, ny, nz = shape
    W = wl.random_case(nx, ny, nz, bc, ratio, seed=nx + ny + nz + n_ranks)
    want = oracle_mod.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt)
    got, p_loc = _slab_step(W, n_ranks)
    errs = {n: rel_l2(g, w_) for n, g, w_ in zip("uvwp", got, want)}
    print(W.name, n_ranks, {k: f"{v:.2e}" for k, v in errs.items()})
    for n, e in errs.items():
        assert e <= TOL, (W.name, n_ranks, n, e)
    # the halo planes of p^(n+1) every rank was sent are its neighbours' planes (a time loop never exchanges them)
    ref = wl.slab_split(want[3], n_ranks, bc == PER)
    for r in range(n_ranks):
        for pl in (0, -1):
            if np.isfinite(ref[r][pl]).all():
                assert rel_l2(p_loc[r][pl], ref[r][pl]) <= TOL, (r, pl)
    if bc == WALL:
        assert np.array_equal(got[2][-1], W.w[-1])          # the top wall face passes through


@pytest.mark.parametrize("mode", ["p_old", "new"])
def test_slab_step_p_out_variants(oracle_mod, mode):
    W = wl.random_case(128, 16, 32, PER, 10.0, seed=77)
    want = oracle_mod.projection_step(*W.fields(), W.box, W.bc_z, W.rho1, W.rho2, W.dt)
    got, _ = _slab_step(W, 4, mode)
    for n, g, w_ in zip("uvwp", got, want):
        assert rel_l2(g, w_) <= TOL, (mode, n)


def test_slab_equals_one_gpu_step_in_a_time_loop():
    """three steps in a ping-pong loop: the pressure halos a step leaves behind are the next step's inputs (no exchange),
    phi keeps its halos, the velocity halos are refreshed by the test (their producer's job); against flutas_projection_step"""
    import paper_2204_08834_b200 as fl
    W = wl.random_case(128, 16, 32, PER, 10.0, seed=5)
    n_ranks = 4
    plan = fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2)
    d = [to_dev(a) for a in W.fields()]
    grp = slab.SlabGroup(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, n_ranks)
    loc = [[to_dev(q) for q in wl.slab_split(a, n_ranks, True)] for a in W.fields()]      # [field][rank]
    for step in range(3):
        plan.projection_step_ex(d[0], d[1], d[2], d[3], d[4], d[5], d[5], W.dt)           # p^(n+1) into p_old, then swap
        d[4], d[5] = d[5], d[4]
        fields = [[loc[f][r] for f in range(6)] for r in range(n_ranks)]
        grp.step(fields, W.dt, 1.0, [loc[5][r] for r in range(n_ranks)])
        loc[4], loc[5] = loc[5], loc[4]
        torch.cuda.synchronize()
        # the velocity of the next step: the corrected one (w needs its lower halo again)
        wg = wl.slab_gather([t.cpu().numpy() for t in loc[2]])
        loc[2] = [to_dev(q) for q in wl.slab_split(wg, n_ranks, True)]
        for f in (0, 1, 2, 4):
            got = wl.slab_gather([t.cpu().numpy() for t in loc[f]])
            assert rel_l2(got, d[f].cpu().numpy()) <= 1e-12, (step, f)
    grp.destroy()
    plan.destroy()


@pytest.mark.parametrize("bc", [PER, WALL])
def test_slab_time_loop_with_halo_exchange(bc):
    """the same loop with SlabGroup.exchange_halos refreshing plane 0 of w (and the halos of phi) between steps, as a solver
    that feeds the corrected velocity back in would: three steps equal three flutas_projection_step_ex on the whole box"""
    import paper_2204_08834_b200 as fl
    W = wl.random_case(128, 16, 32, bc, 10.0, seed=6)
    n_ranks, periodic = 4, bc == PER
    plan = fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2)
    d = [to_dev(a) for a in W.fields()]
    grp = slab.SlabGroup(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2, n_ranks)
    loc = [[to_dev(q) for q in wl.slab_split(a, n_ranks, periodic)] for a in W.fields()]   # [field][rank]
    for f in (2, 3):                                     # stale halos of w and phi: the exchange must supply them
        for t in loc[f]:
            t[0] = 123.0
            t[-1] = 123.0
    for step in range(3):
        plan.projection_step_ex(d[0], d[1], d[2], d[3], d[4], d[5], d[5], W.dt)
        d[4], d[5] = d[5], d[4]
        fields = [[loc[f][r] for f in range(6)] for r in range(n_ranks)]
        grp.exchange_halos(fields, periodic)
        grp.step(fields, W.dt, 1.0, [loc[5][r] for r in range(n_ranks)])
        loc[4], loc[5] = loc[5], loc[4]
        torch.cuda.synchronize()
        for f in (0, 1, 2, 4):
            got = wl.slab_gather([t.cpu().numpy() for t in loc[f]])
            assert rel_l2(got, d[f].cpu().numpy()) <= 1e-12, (step, f)
    grp.destroy()
    plan.destroy()


def test_slab_rejects_bad_decompositions():
    for args in [(128, 16, 32, PER, 3), (128, 16, 32, PER, 32), (64, 16, 32, PER, 2), (128, 16, 24, PER, 2),
                 (128, 16, 1024, WALL, 2), (128, 4, 32, PER, 2)]:
        assert binding.lib.flutas_slab_workspace_bytes(*args) == 0, args
        with pytest.raises(binding.FlutasError):
            binding.SlabPlan(args[0], args[1], args[2], 1.0, 1.0, 1.0, args[3], 1.0, 2.0, args[4], 0)


def _slab_rank_worker(port, q):
    """one NCCL rank: SlabRank (exchange buffer from torch symmetric memory, all-reduce as the barrier) against flutas_projection_step"""
    import os
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port), RANK="0", WORLD_SIZE="1", LOCAL_RANK="0")
    import numpy as np
    import torch
    import torch.distributed as dist
    import paper_2204_08834_b200 as fl
    import workloads as wl
    from paper_2204_08834_b200 import slab
    torch.cuda.set_device(0)
    dist.init_process_group("nccl", rank=0, world_size=1)
    try:
        W = wl.random_case(128, 16, 32, PER, 10.0, seed=9)
        plan = fl.Plan(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2)
        d = [torch.from_numpy(a).cuda() for a in W.fields()]
        plan.projection_step(*d, W.dt)
        try:
            sr = slab.SlabRank(W.nx, W.ny, W.nz, *W.box, W.bc_z, W.rho1, W.rho2)
        except Exception as e:                                   # symmetric memory not available in this build / on this box
            q.put(("skip", repr(e)))
            return
        loc = [torch.from_numpy(wl.slab_split(a, 1, True)[0]).cuda() for a in W.fields()]
        sr.step(*loc, W.dt)
        torch.cuda.synchronize()
        errs = [float((loc[f][1:-1].reshape(-1) - d[f].reshape(-1)).norm() / d[f].norm()) for f in (0, 1, 2, 4)]
        q.put(("ok", errs))
        sr.destroy()
    finally:
        dist.destroy_process_group()


def test_slab_rank_over_symmetric_memory_one_rank():
    """the torchrun path of slab.py (SlabRank) with a process group of ONE rank: exercises the symmetric-memory allocation,
    the rendezvous, the pointer table and the all-reduce barrier; more ranks need more GPUs than this run has"""
    import socket
    import torch.multiprocessing as mp
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    p = ctx.Process(target=_slab_rank_worker, args=(port, q))
    p.start()
    status, payload = q.get(timeout=240)
    p.join(timeout=60)
    if status == "skip":
        pytest.skip("torch symmetric memory unavailable: " + payload)
    assert max(payload) <= 1e-12, payload
