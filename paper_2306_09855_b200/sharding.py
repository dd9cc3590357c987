"""One shard of a network per rank (include/nc.h: nc_set_shard; multi-GPU construction is the paper's stated
future work; reading S1).  Nodes are partitioned into contiguous ranges, rank r owns range r and keeps, of every connect
call, the connections whose target it owns.  No connection crosses between ranks: a rank draws the random numbers of the
connections it does not own as well and skips them, so the data path has no collective; torch.distributed is used only to
check that the shards add up and (bench.py --sharded) to line the ranks up around the timed region.

Nothing here computes anything of the method: `backend` is a paper_2306_09855_b200.binding.NC context (or, in the CPU
tests, the oracle, which has the same method names)."""
from __future__ import annotations

import numpy as np

from . import workloads as WL


def partition(n_nodes: int, world: int):
    """Contiguous node ranges of near-equal size: rank r owns ids bounds[r] .. bounds[r + 1] - 1."""
    return [n_nodes * r // world for r in range(world + 1)]


def owned_range(n_nodes: int, world: int, rank: int):
    b = partition(n_nodes, world)
    return b[rank], b[rank + 1] - b[rank]


def build_shard(net, backend, world: int, rank: int, finalize: bool = True):
    """Replay the recipe on `backend` as rank `rank` of `world`."""
    return WL.run(net, backend, finalize=finalize, shard=owned_range(net.n_nodes, world, rank))


def shard_sizes(dist, n_local: int, device="cpu"):
    """Connections held by every rank (all_gather of one integer)."""
    if dist is None:
        return [int(n_local)]
    import torch
    mine = torch.tensor([int(n_local)], dtype=torch.int64, device=device)
    out = [torch.zeros_like(mine) for _ in range(dist.get_world_size())]
    dist.all_gather(out, mine)
    return [int(t.item()) for t in out]


def summed_out_degree(dist, out_degree: np.ndarray, device="cpu") -> np.ndarray:
    """Out-degree of every node over all shards (a source's connections are spread over the ranks that own its targets)."""
    if dist is None:
        return out_degree.astype(np.int64)
    import torch
    t = torch.from_numpy(out_degree.astype(np.int64)).to(device)
    dist.all_reduce(t, op=dist.ReduceOp.SUM)
    return t.cpu().numpy()
