"""Batch sharding across ranks: problems are independent, so the only exchange is one
sum-all-reduce of the 2K+1 shared hyper-parameter gradients after the backward pass (CDU_RHO_PER_ITER)."""
from __future__ import annotations

from typing import Dict, List, Sequence


def shard_indices(n_items: int, rank: int, world: int) -> List[int]:
    """Contiguous, balanced split of range(n_items); the first n_items % world ranks get one more."""
    base, rem = divmod(n_items, world)
    start = rank * base + min(rank, rem)
    return list(range(start, start + base + (1 if rank < rem else 0)))


def allreduce_shared_grads(grads: Dict[str, "object"], keys: Sequence[str] = ("g_rho", "g_alpha", "g_sigma"), group=None) -> None:
    """In-place SUM over ranks of the shared-theta gradients; a no-op without an initialised process group."""
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size(group) == 1:
        return
    for k in keys:
        dist.all_reduce(grads[k], op=dist.ReduceOp.SUM, group=group)
