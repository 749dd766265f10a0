"""Multi-GPU host logic on CPU (-m "not gpu"): agent sharding and the end-of-cycle winner exchange, with
torch.distributed gloo, world_size 2.  The per-rank rollouts are the oracle's (the CUDA path needs a GPU);
what is tested is that sharding + key exchange reproduces the single-process selection."""
import os
import socket

import numpy as np
import pytest
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2606_12579_b200 import scenes, sharding


def test_shard_range_partitions():
    for n in (1, 2, 7, 1024, 1025):
        for w in (1, 2, 3, 8):
            r = [sharding.shard_range(n, k, w) for k in range(w)]
            assert r[0][0] == 0 and r[-1][1] == n
            assert all(r[k][1] == r[k + 1][0] for k in range(w - 1))
            sizes = [b - a for a, b in r]
            assert max(sizes) - min(sizes) <= 1


def test_combine_best_is_lexicographic():
    assert sharding.combine_best([(1, 0.1, 3), (0, 0.9, 7), (0, 0.9, 5)]) == (0, 0.9, 5)
    assert sharding.local_key(0, float("nan"), 2, 10) == (1, float("inf"), 12)


def test_combine_best_applies_hysteresis_once():
    keys = [(0, 0.50, 3), (0, 0.48, 40)]
    # challenger 40 does not beat alpha * C_prev = 0.45: the incumbent (agent 7) stays; with alpha = 1 it loses
    assert sharding.combine_best(keys, (0, 0.5, 7), alpha=0.9) == (0, 0.5, 7)
    assert sharding.combine_best(keys, (0, 0.5, 7), alpha=1.0) == (0, 0.48, 40)
    assert sharding.combine_best(keys, (1, 0.1, 7), alpha=0.9) == (0, 0.48, 40)      # collided incumbent always loses
    assert sharding.combine_best(keys, (0, 0.48, 40), alpha=0.9) == (0, 0.48, 40)    # the incumbent is the winner
    assert sharding.combine_best(keys, None) == (0, 0.48, 40)
    assert sharding.local_prev(40, 32, 64) == 8 and sharding.local_prev(40, 0, 32) == -1


def _select_like_gpu(orc, cost, collided, alpha, prev_local):
    """A rank's selection record as api.Context.select returns it, built from the oracle's selection."""
    raw, raw_cost = orc.best_agent(cost, collided, alpha, -1)
    idx, c = orc.best_agent(cost, collided, alpha, prev_local)
    rec = dict(index=idx, collided=int(collided[idx]), cost=c, raw_index=raw, raw_collided=int(collided[raw]), raw_cost=raw_cost,
               prev_collided=0, prev_cost=float("nan"))
    if prev_local >= 0:
        rec.update(prev_collided=int(collided[prev_local]), prev_cost=float(cost[prev_local, 0]))
    return rec


def _scene():
    return scenes.fast_clutter(n_agents=37, n_spheres=120, r_lo=0.02, r_hi=0.06, steps=60)


def _worker(rank, world, port, q, cases):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle
    sc = _scene()
    lo, hi = sharding.shard_range(sc.n_agents, rank, world)
    o = oracle.rollout_scene(sc, agent_slice=slice(lo, hi))
    out = []
    for alpha, prev in cases:
        pl = sharding.local_prev(prev, lo, hi)
        rec = _select_like_gpu(oracle, o["cost"], o["collided"], alpha, pl)
        raw, inc = sharding.selection_keys(rec, lo, pl)
        out.append(sharding.all_gather_best(raw, inc, alpha))
    q.put((rank, out))
    dist.destroy_process_group()


def test_two_rank_selection_matches_single_process(orc):
    sc = _scene()
    o = orc.rollout_scene(sc)
    best, _ = orc.best_agent(o["cost"], o["collided"], 0.9, -1)
    order = np.lexsort((o["cost"][:, 0], o["collided"]))          # agents by key
    lo1, _ = sharding.shard_range(sc.n_agents, 1, 2)
    on_rank1 = [int(i) for i in order if i >= lo1 and i != best]
    on_rank0 = [int(i) for i in order if i < lo1 and i != best]
    # no incumbent; incumbents on rank 1 and on rank 0 (a close runner-up that keeps its place at alpha = 0.9 and a
    # poor one that loses it); alpha = 1 (plain comparison); the incumbent IS the winner
    cases = [(0.9, -1), (0.9, on_rank1[0]), (0.9, on_rank0[0]), (0.9, on_rank1[-1]), (0.9, on_rank0[-1]),
             (1.0, on_rank1[0]), (0.5, on_rank1[1]), (0.9, int(best))]
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q, cases)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60); assert p.exitcode == 0
    assert got[0] == got[1]
    kept = 0
    for (alpha, prev), key in zip(cases, got[0]):
        want, cost = orc.best_agent(o["cost"], o["collided"], alpha, prev)
        assert key[2] == want and key[1] == cost and key[0] == int(o["collided"][want]), (alpha, prev, key, want)
        kept += int(prev >= 0 and want == prev and prev != best)
    assert kept >= 1                                               # the hysteresis rule really decided a case
