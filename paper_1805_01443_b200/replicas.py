"""Multi-GPU plumbing for the replicas-only scaling of this path.

north_star fixes one GPU per problem: no domain decomposition, no data-path collective.  With N
GPUs, ``bench.py --gpus N`` therefore runs N independent replicas of the workload, one process per
GPU, and only the *measurement* crosses ranks: a barrier on both sides of the timed region, the
maximum of the per-rank device times, the sum of the units processed.  These helpers do exactly
that over ``torch.distributed`` (NCCL on the GPU box, gloo in the CPU tests) and nothing else.
"""
from __future__ import annotations

import os


def world():
    """(rank, local_rank, world_size) from the torchrun environment (1 process when absent)."""
    return (int(os.environ.get("RANK", "0")), int(os.environ.get("LOCAL_RANK", "0")),
            int(os.environ.get("WORLD_SIZE", "1")))


def init(backend: str, device=None):
    """Join the job's process group if there is more than one rank.  Returns True when joined."""
    rank, _local, size = world()
    if size <= 1:
        return False
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    os.environ.setdefault("MASTER_PORT", "29500")
    kw = {}
    if device is not None and backend == "nccl":
        kw["device_id"] = device
    dist.init_process_group(backend=backend, rank=rank, world_size=size, **kw)
    return True


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.barrier()


def aggregate(elapsed_ms: float, units: float, device="cpu"):
    """Whole-job figures of a replicas run: (max over ranks of elapsed_ms, sum over ranks of units)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return float(elapsed_ms), float(units)
    t = torch.tensor([float(elapsed_ms)], dtype=torch.float64, device=device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def throughput(elapsed_ms: float, units: float, device="cpu") -> tuple[float, float]:
    """(units per second of the whole job, the max-over-ranks time in ms)."""
    t, u = aggregate(elapsed_ms, units, device)
    return (u / (t * 1e-3) if t > 0 else 0.0), t


def finish():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized():
        dist.destroy_process_group()
