"""Multi-GPU plumbing of bench.py: the construction path does not shard (replicas only), so N
ranks build N independent networks.  There is no collective on the data path; torch.distributed is used only to
line the ranks up around the timed region and to reduce the device time to its maximum over the ranks."""
from __future__ import annotations

import os


def env_world():
    """(world_size, rank, local_rank) as torchrun exports them; (1, 0, 0) for a plain launch."""
    return (int(os.environ.get("WORLD_SIZE", "1")), int(os.environ.get("RANK", "0")),
            int(os.environ.get("LOCAL_RANK", "0")))


def init(backend: str, device=None):
    """Join the process group when launched with WORLD_SIZE > 1; returns torch.distributed or None."""
    world, _, _ = env_world()
    if world <= 1:
        return None
    import torch.distributed as dist
    kw = {"device_id": device} if (device is not None and backend == "nccl") else {}
    dist.init_process_group(backend, **kw)
    return dist


def barrier(dist, sync=None):
    if dist is not None:
        dist.barrier()
    if sync is not None:
        sync()


def max_over_ranks(dist, value: float, device="cpu") -> float:
    """The slowest rank's time: what the whole job took."""
    if dist is None:
        return float(value)
    import torch
    t = torch.tensor([float(value)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_per_step: int, steps: int, world: int, slowest_ms: float) -> float:
    """Units all ranks processed divided by the time of the slowest rank (weak scaling: per-rank work is fixed)."""
    return world * units_per_rank_per_step * steps / (slowest_ms * 1e-3)
