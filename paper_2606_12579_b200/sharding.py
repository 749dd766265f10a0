"""Host-side logic for running the rollout on several GPUs (one process per GPU).

The path shards BY AGENTS: every agent's rollout depends only on the (replicated) sphere world
(oracle pin P12), so each rank rolls its own block of agents with no communication
during the S steps.  The only exchange is the end-of-cycle selection (reading G24): every
rank contributes the key (collided, cost, global index) of its local winner WITHOUT hysteresis and -- the
rank that owns the incumbent -- the incumbent's own key of this cycle; all ranks take the lexicographic
minimum of the winners and then apply the hysteresis rule ONCE, globally.  24 bytes per rank, one
all_gather.  The comparison C_best < alpha * C_prev is taken in FP32, as the selection kernel takes it.
"""
from __future__ import annotations

import math
from typing import List, Optional, Sequence, Tuple

import numpy as np

Key = Tuple[int, float, int]            # (collided, cost, global agent index)


def shard_range(n_items: int, rank: int, world: int) -> Tuple[int, int]:
    """Contiguous block [lo, hi) of `n_items` for `rank` of `world`; sizes differ by at most one."""
    base, rem = divmod(n_items, world)
    lo = rank * base + min(rank, rem)
    return lo, lo + base + (1 if rank < rem else 0)


def local_prev(prev_best: int, lo: int, hi: int) -> int:
    """The global incumbent as a LOCAL index on the rank that owns it, -1 on every other rank."""
    return prev_best - lo if lo <= prev_best < hi else -1


def local_key(collided: int, cost: float, local_index: int, offset: int) -> Key:
    """Selection key of a rank's local winner, with the index made global.  NaN cost ranks last."""
    if cost != cost:
        return (1, math.inf, local_index + offset)
    return (1 if collided else 0, float(cost), local_index + offset)


def combine_best(keys: Sequence[Key], incumbent: Optional[Key] = None, alpha: float = 0.9) -> Key:
    """Lexicographic minimum of the ranks' raw winners, then the hysteresis rule against the incumbent's key
    (collided, cost, global index) -- the same rule as one GPU applies to all agents (reading G24): the incumbent
    keeps its place unless the challenger's flag is better, or the flags are equal and C_best < alpha * C_prev."""
    best = min(keys)
    if incumbent is None or incumbent[2] < 0 or incumbent[2] == best[2]:
        return best
    bc, bC, _ = best
    cp, Cp, _ = incumbent
    improves = (bc < cp) or (bc == cp and np.float32(bC) < np.float32(alpha) * np.float32(Cp))
    return best if improves else incumbent


def selection_keys(rec: dict, lo: int, prev_local: int) -> Tuple[Key, Optional[Key]]:
    """From one rank's selection record (api.Context.select with the LOCAL incumbent or -1): its raw winner's key and,
    on the owning rank, the incumbent's key."""
    raw = local_key(rec["raw_collided"], rec["raw_cost"], rec["raw_index"], lo)
    inc = local_key(rec["prev_collided"], rec["prev_cost"], prev_local, lo) if prev_local >= 0 else None
    return raw, inc


def all_gather_best(raw: Key, incumbent: Optional[Key] = None, alpha: float = 0.9, group=None) -> Key:
    """Exchange the per-rank keys with torch.distributed (gloo on CPU, NCCL on GPU) and combine."""
    import torch
    import torch.distributed as dist
    world = dist.get_world_size(group)
    dev = "cuda" if dist.get_backend(group) == "nccl" else "cpu"
    inc = incumbent if incumbent is not None else (0, 0.0, -1)
    mine = torch.tensor([float(raw[0]), float(raw[1]), float(raw[2]), float(inc[0]), float(inc[1]), float(inc[2])],
                        dtype=torch.float64, device=dev)
    out: List[torch.Tensor] = [torch.empty_like(mine) for _ in range(world)]
    dist.all_gather(out, mine, group=group)
    keys = [(int(t[0].item()), float(t[1].item()), int(t[2].item())) for t in out]
    incs = [(int(t[3].item()), float(t[4].item()), int(t[5].item())) for t in out if int(t[5].item()) >= 0]
    return combine_best(keys, incs[0] if incs else None, alpha)
