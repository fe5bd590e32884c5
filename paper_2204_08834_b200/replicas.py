"""Host-side plumbing for running N independent replicas of the projection step, one process per GPU.

The path does not shard without an exchange step and BASELINE.json's north_star excludes a multi-GPU
decomposition, so N GPUs means N independent boxes (ensemble members / parameter sweep): "replicas
only", weak scaling, no data-path collective.  The only communication is the timing protocol:
a barrier before and after the timed region and a MAX over ranks of the device time.
"""
import os

import torch
import torch.distributed as dist


def init_from_env(backend=None):
    """(rank, local_rank, world_size); initialises torch.distributed when WORLD_SIZE > 1."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1 and not dist.is_initialized():
        if backend is None:
            backend = "nccl" if torch.cuda.is_available() else "gloo"
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29500")
        dist.init_process_group(backend=backend, rank=rank, world_size=world)
    return rank, local_rank, world


def barrier():
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def _device_for_collectives():
    if dist.is_initialized() and dist.get_backend() == "nccl":
        return torch.device("cuda", torch.cuda.current_device())
    return torch.device("cpu")


def aggregate_throughput(units_local, ms_local):
    """Whole-job throughput of independent replicas: (sum of units over ranks, max of ms over ranks).

    units_local: work units this rank processed in the timed region (grid points x steps)
    ms_local:    device time of this rank's timed region, milliseconds"""
    if not (dist.is_available() and dist.is_initialized()):
        return float(units_local), float(ms_local)
    dev = _device_for_collectives()
    u = torch.tensor([float(units_local)], dtype=torch.float64, device=dev)
    t = torch.tensor([float(ms_local)], dtype=torch.float64, device=dev)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(u.item()), float(t.item())


def replica_density_ratio(rank, ratios=(50.0, 1.0)):
    """Each replica takes one member of the density-ratio sweep of config 4 (BASELINE.json: {1, 50})."""
    return ratios[rank % len(ratios)]
