"""-m "not gpu": host logic of the z-slab decomposition: the partition and the two
destination maps the kernels' store stages implement (paper_2204_08834_b200/slab.py), the size queries of the C ABI, and --
two gloo ranks on CPU -- that the maps are the all-to-all transposes of PAPER.md:169-183: exchanging exactly the
blocks they name turns z-slabs into ky-slabs and back (with the neighbours' boundary planes as halos)."""
import os
import socket

import numpy as np
import pytest
import torch.multiprocessing as mp

from paper_2204_08834_b200 import binding, slab


def test_partition_covers_every_plane_and_row_once():
    for nz, ny, P in ((32, 16, 4), (512, 1024, 8), (16, 16, 16), (8, 8, 1)):
        planes, rows = zip(*(slab.partition(nz, ny, P, r) for r in range(P)))
        assert [a for a, _ in planes] == list(range(0, nz, nz // P)) and planes[-1][1] == nz
        assert [a for a, _ in rows] == list(range(0, ny, ny // P)) and rows[-1][1] == ny
    with pytest.raises(ValueError):
        slab.partition(30, 16, 4, 0)


def test_destination_maps():
    nz, ny, P = 16, 8, 4
    seen = {}
    for k in range(nz):
        for j in range(ny):
            r, kk, jl = slab.forward_destination(k, j, nz, ny, P)
            assert slab.partition(nz, ny, P, r)[1][0] + jl == j and kk == k
            seen[(r, kk, jl)] = seen.get((r, kk, jl), 0) + 1
    assert len(seen) == nz * ny and set(seen.values()) == {1}            # a bijection
    for periodic in (True, False):
        cnt = {}
        for k in range(nz):
            for d in slab.backward_destinations(k, 3, nz, ny, P, periodic):
                cnt[d[:2]] = cnt.get(d[:2], 0) + 1
        nzl = nz // P
        want = P * (nzl + 2) - (0 if periodic else 2)                     # every local plane once; none beyond a wall
        assert len(cnt) == want and set(cnt.values()) == {1}
        assert ((0, 0) in cnt) == periodic and ((P - 1, nzl + 1) in cnt) == periodic


def test_size_queries_need_no_device():
    up = lambda b: (b + 1023) // 1024 * 1024
    nx, ny, nz, P = 256, 64, 128, 4
    nzl, rpp, pitch = nz // P, ny // P, nx // 2 + 8
    ex = binding.lib.flutas_slab_exchange_bytes(nx, ny, nz, 0, P)
    assert ex == up(16 * pitch * (rpp + 1) * nz) + up(16 * pitch * (ny + 1) * (nzl + 2))
    ws = binding.lib.flutas_slab_workspace_bytes(nx, ny, nz, 0, P)
    assert ws == 4 * up(8 * nx * ny * (nzl + 2)) + 1024
    assert binding.lib.flutas_slab_workspace_bytes(nx, ny, nz, 1, P) > ws                 # + the elimination table
    assert binding.lib.flutas_slab_exchange_bytes(nx, ny, nz, 0, 3) == 0
    assert binding.lib.flutas_slab_step_phase(None, 0, *([None] * 7), 1e-3, 1.0, None) == 1
    binding.lib.flutas_slab_plan_destroy(None)


def test_slab_plan_needs_a_device_and_rejects_bad_arguments():
    import torch
    lib = binding.lib
    for args, code in (((128, 16, 32, 1.0, 1.0, 1.0, 0, 1.0, 2.0, 3, 0), 2),      # ranks not a power of two
                       ((128, 16, 32, 1.0, 1.0, 1.0, 0, 1.0, 2.0, 4, 4), 1),      # rank outside [0, n_ranks)
                       ((128, 16, 32, 0.0, 1.0, 1.0, 0, 1.0, 2.0, 4, 0), 1),      # box length
                       ((64, 16, 32, 1.0, 1.0, 1.0, 0, 1.0, 2.0, 2, 0), 2),       # nx below the bulk-copy-fed kernels' minimum
                       ((128, 16, 600, 1.0, 1.0, 1.0, 1, 1.0, 2.0, 2, 0), 2)):    # wall nz beyond the one-pass elimination
        assert not lib.flutas_slab_plan_create(*args)
        assert lib.flutas_last_error_code() == code, (args, lib.flutas_last_error())
    if not torch.cuda.is_available():
        assert not lib.flutas_slab_plan_create(128, 16, 32, 1.0, 1.0, 1.0, 0, 1.0, 2.0, 4, 0)
        assert lib.flutas_last_error_code() == 4 and b"no CPU fallback" in lib.flutas_last_error()


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _all_to_all(dist, send, rank, world):
    """gloo has no all-to-all: every rank gathers every rank's send list and keeps the blocks addressed to it"""
    import torch
    mine = torch.stack(send)
    every = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(every, mine)
    return [every[src][rank] for src in range(world)]


def _worker(rank, world, port, q):
    os.environ.update(WORLD_SIZE=str(world), RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    nz, ny, nxh, periodic = 8, 4, 3, True
    nzl, rpp = nz // world, ny // world
    full = np.random.default_rng(0).standard_normal((nz, ny, nxh))                      # the same on both ranks
    (k0, k1), (j0, j1) = slab.partition(nz, ny, world, rank)
    mine = full[k0:k1]
    # forward: send row block s of my planes to rank s; what arrives must be all planes of my rows
    send = [torch.from_numpy(np.ascontiguousarray(mine[:, s * rpp:(s + 1) * rpp])) for s in range(world)]
    recv = _all_to_all(dist, send, rank, world)
    zloc = np.empty((nz, rpp, nxh))
    for src in range(world):
        for kl in range(nzl):
            for jl in range(rpp):
                r, k, jj = slab.forward_destination(src * nzl + kl, rank * rpp + jl, nz, ny, world)
                assert r == rank
                zloc[k, jj] = recv[src][kl, jl].numpy()
    ok_fwd = np.array_equal(zloc, full[:, j0:j1])
    # backward: every plane of my rows goes to its owner and, at slab boundaries, to the neighbour's halo plane
    out = [np.full((nzl + 2, rpp, nxh), np.nan) for _ in range(world)]
    for k in range(nz):
        for (r, kl, _) in slab.backward_destinations(k, j0, nz, ny, world, periodic):
            out[r][kl] = zloc[k]
    send = [torch.from_numpy(o) for o in out]
    recv = _all_to_all(dist, send, rank, world)
    back = np.concatenate([t.numpy() for t in recv], axis=1)                              # (nzl + 2, ny, nxh)
    want = np.stack([full[(k0 - 1 + i) % nz] for i in range(nzl + 2)])
    q.put((rank, bool(ok_fwd), bool(np.array_equal(back, want))))
    dist.barrier()
    dist.destroy_process_group()


def test_maps_are_the_two_transposes_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=90) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out == [(0, True, True), (1, True, True)]


def test_halo_neighbours():
    assert slab.halo_neighbours(4, 0, True) == (3, 1) and slab.halo_neighbours(4, 3, True) == (2, 0)
    assert slab.halo_neighbours(4, 0, False) == (None, 1) and slab.halo_neighbours(4, 3, False) == (2, None)
    assert slab.halo_neighbours(1, 0, True) == (0, 0) and slab.halo_neighbours(1, 0, False) == (None, None)


def _halo_worker(rank, world, port, q):
    os.environ.update(WORLD_SIZE=str(world), RANK=str(rank), LOCAL_RANK=str(rank), MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    import torch
    import torch.distributed as dist
    import workloads as wl
    dist.init_process_group(backend="gloo", rank=rank, world_size=world)
    nz, ny, nx = 8, 3, 5
    nzl = nz // world
    rng = np.random.default_rng(3)
    w_full, phi_full = rng.standard_normal((nz, ny, nx)), rng.standard_normal((nz, ny, nx))     # the same on every rank
    ok = []
    for periodic in (True, False):
        want_w, want_phi = (wl.slab_split(a, world, periodic)[rank] for a in (w_full, phi_full))
        w, phi = want_w.copy(), want_phi.copy()
        w[0] = w[nzl + 1] = phi[0] = phi[nzl + 1] = -7.0                                        # stale halos
        tw, tp = torch.from_numpy(w), torch.from_numpy(phi)
        slab.exchange_halos(tw, tp, nzl, periodic)
        below, above = slab.halo_neighbours(world, rank, periodic)
        # what a step reads: plane 0 of w, both halo planes of phi; planes beyond a wall stay as they were (never read)
        good = np.array_equal(w[1:nzl + 1], want_w[1:nzl + 1]) and np.array_equal(phi[1:nzl + 1], want_phi[1:nzl + 1])
        good &= np.array_equal(w[0], want_w[0]) and np.array_equal(phi[0], want_phi[0]) if below is not None else bool(np.all(w[0] == -7.0))
        good &= np.array_equal(phi[nzl + 1], want_phi[nzl + 1]) if above is not None else bool(np.all(phi[nzl + 1] == -7.0))
        good &= bool(np.all(w[nzl + 1] == -7.0))                                                # the upper halo of w is never needed
        ok.append(bool(good))
    q.put((rank, *ok))
    dist.barrier()
    dist.destroy_process_group()


@pytest.mark.parametrize("world", [2, 4])
def test_halo_exchange_gloo(world):
    """exchange_halos between processes: with two ranks both messages of a rank go to the same peer (order matters), with
    four every rank has two distinct neighbours; periodic and wall-bounded"""
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_halo_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert out == [(r, True, True) for r in range(world)]
