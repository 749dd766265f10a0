"""Host-side logic for running the rollout on several GPUs (one process per GPU).

The path shards BY AGENTS: every agent's rollout depends only on the (replicated) sphere world
(oracle pin P12), so each rank rolls its own block of agents with no communication
during the S steps.  The only exchange is the end-of-cycle selection: every rank contributes its local
winner's key (collided, cost, global index) and all ranks take the lexicographic minimum -- 12 bytes
per rank, done with one all_gather.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import math
from typing import List, Sequence, Tuple


def shard_range(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of `n_items` for `rank` of `world`; sizes differ by at most one."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def local_key(collided: int, cost: float, local_index: int, offset: int) -> Tuple[int, float, int]:
    """Selection key of a rank's local winner, with the index made global.  NaN cost ranks last."""
    if cost != cost:
        return (1, math.inf, local_index + offset)
    return (1 if collided else 0, float(cost), local_index + offset)


def combine_best(keys: Sequence[Tuple[int, float, int]]) -> Tuple[int, float, int]:
    """Lexicographic minimum of (collided, cost, global index) over ranks (reading G24)."""
    return min(keys)


def all_gather_best(key: Tuple[int, float, int], group=None) -> Tuple[int, float, int]:
    """Exchange the per-rank keys with torch.distributed (gloo on CPU, NCCL on GPU) and combine."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    mine = torch.tensor([float(key[0]), float(key[1]), float(key[2])], dtype=torch.float64, device=dev)
    out: List[torch.Tensor] = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine, group=group)
    keys = [(int(t[0].item()), float(t[1].item()), int(t[2].item())) for t in out]
    return combine_best(keys)
