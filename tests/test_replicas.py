"""N > 1 host logic on CPU: two gloo ranks aggregate their replicas' throughput (sum of units,
max of time), as bench.py does under torchrun."""
import os
import socket

import torch.multiprocessing as mp


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    os.environ.update(WORLD_SIZE=str(world), RANK=str(rank), LOCAL_RANK=str(rank),
                      MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    from paper_2204_08834_b200 import replicas
    r, lr, w = replicas.init_from_env(backend="gloo")
    replicas.barrier()
    units, ms = replicas.aggregate_throughput(1000.0 * (rank + 1), 10.0 + 5.0 * rank)
    q.put((r, w, units, ms, replicas.replica_density_ratio(rank)))
    replicas.barrier()


def test_two_rank_aggregation_gloo():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    out = sorted(q.get(timeout=120) for _ in procs)
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert [o[0] for o in out] == [0, 1] and all(o[1] == 2 for o in out)
    for o in out:
        assert o[2] == 3000.0 and o[3] == 15.0          # SUM of units, MAX of time on every rank
    assert out[0][4] == 50.0 and out[1][4] == 1.0


def test_single_process_aggregation_is_identity():
    from paper_2204_08834_b200 import replicas
    assert replicas.aggregate_throughput(7.0, 3.0) == (7.0, 3.0)
