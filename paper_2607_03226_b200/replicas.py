"""Host-side plumbing for running N independent replicas of the solver, one process per GPU.

The north_star keeps the hot path on one GPU (nothing spans more than one), so the multi-GPU mode is "replicas only"
(DESIGN.md section 8): every rank solves its own problem instance, there is NO data-path collective, and the only
communication is the timing protocol of the measurement contract -- a barrier on both sides of the timed region and
the MAX over ranks of the device-timed duration.  `torch.distributed` does the plumbing (NCCL on GPUs, gloo in the
CPU tests); this module holds no arithmetic of the method.
"""
from __future__ import annotations

import os


def env_rank():
    """(rank, world_size, local_rank) from the torchrun environment (1-process defaults)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend, device=None):
    """Joins the process group torchrun described (MASTER_ADDR/PORT from the env); returns torch.distributed or None
    for a single process."""
    rank, world, _ = env_rank()
    if world <= 1:
        return None
    import torch.distributed as dist
    if not dist.is_initialized():
        kw = {"device_id": device} if (device is not None and backend == "nccl") else {}
        dist.init_process_group(backend, rank=rank, world_size=world, **kw)
    return dist


def barrier(dist, sync=None):
    """`sync` (e.g. torch.cuda.synchronize) runs before and after the collective barrier."""
    if sync:
        sync()
    if dist is not None:
        dist.barrier()
        if sync:
            sync()


def max_over_ranks(value, dist, device="cpu"):
    """MAX over ranks of a scalar (the slowest replica defines the step time)."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_replica, world, seconds_per_step):
    """Aggregate throughput of `world` replicas that each process `units_per_replica` per step (weak scaling)."""
    return world * units_per_replica / seconds_per_step
