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


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"; os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    from oracle import oracle
    sc = scenes.fast_clutter(n_agents=37, n_spheres=120, r_lo=0.02, r_hi=0.06, steps=60)
    lo, hi = sharding.shard_range(sc.n_agents, rank, world)
    o = oracle.rollout_scene(sc, agent_slice=slice(lo, hi))
    idx, cost = oracle.best_agent(o["cost"], o["collided"], 0.9, -1)
    key = sharding.all_gather_best(sharding.local_key(int(o["collided"][idx]), cost, idx, lo))
    q.put((rank, key))
    dist.destroy_process_group()


def test_two_rank_selection_matches_single_process(orc):
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = dict(q.get(timeout=120) for _ in range(2))
    for p in procs:
        p.join(60); assert p.exitcode == 0
    sc = scenes.fast_clutter(n_agents=37, n_spheres=120, r_lo=0.02, r_hi=0.06, steps=60)
    o = orc.rollout_scene(sc)
    want, cost = orc.best_agent(o["cost"], o["collided"], 0.9, -1)
    assert got[0] == got[1]
    assert got[0][2] == want and got[0][1] == cost and got[0][0] == int(o["collided"][want])
