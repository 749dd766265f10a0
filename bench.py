#!/usr/bin/env python
"""bench.py -- headline benchmark of the G-MAPP rollout on B200.

A "step" is one planning cycle of the whole hot path: one persistent rollout
launch over all agents x spheres x rollout steps, then the selection kernel and its 8-byte download.
Workload at N=1: BASELINE.json configs[2], "dense depth-derived clutter" = 1024 agents x 4096 spheres x
100 rollout steps, the configuration north_star's target is quoted on.  Synthetic, seeded inputs
(paper_2606_12579_b200/scenes.py) stand in for the paper's scenes, whose geometry the paper does not give.

    python bench.py --gpus 1 --steps 20 --warmup 5
    python -m torch.distributed.run --nproc-per-node N ... bench.py --gpus N ...   (weak scaling by agents)
    python bench.py --impl reference ...     (the FP64 oracle on the host cores, bounded sample)
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "agent-sphere force interactions/s"
UNIT = "interactions/s"
# Algorithmic FP32 work of one agent-sphere pair: distance + gate
# 17 flop, circular-field force 18 flop, an FFMA counted as 2.  Newton-refinement instructions that this
# implementation adds for accuracy are NOT counted.
FLOP_PER_PAIR = 35.0
# FP32 peak from the guide's unit counts and clock: 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz
NOMINAL_SMS, LANES_PER_SM, MAX_GHZ = 148, 128, 1.965
PEAK_TFLOPS = NOMINAL_SMS * LANES_PER_SM * 2 * MAX_GHZ / 1e3
# dram__bytes_read.sum + dram__bytes_write.sum of one rollout launch, from committed `ncu --set full` captures (not
# measurable inside an un-profiled run).  config3: profiles/r01_rollout_x2_full.md, 187.6 KB read + 0 B written
# (algorithmic: 64 KB sphere pairs + 24 KB agents in; 36 KB results out stay in L2).  Workloads without a capture report
# null and say why.
TRAFFIC_BYTES_PER_LAUNCH = {"config3": 187648}
TRAFFIC_SOURCE = {"config3": "profiles/r01_rollout_x2_full.md (ncu --set full, one launch)"}
# every BASELINE.json config and the 3 x 3 stress sweep, plus agent counts between the grid points (launch selection)
ALL_CONFIG_ROWS = (["config1", "config2", "config3", "config4"]
                   + [f"sweep:{a}x{s}" for s in (4096, 16384, 65536) for a in (1024, 4096, 16384)]
                   + ["sweep:1500x4096", "sweep:2048x4096", "sweep:3000x4096"])
# moving spheres (config 4): FP32-pipe lane-operations per pair of the method as SURVEY.md 8(d) counts them (static: 22)
LANE_OPS_PER_PAIR_MOVING = 36.0


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", default="config3", help="config1|config2|config3|config4|sweep:<agents>x<spheres>")
    ap.add_argument("--cull", type=int, default=-1, help="-1 library default, 0 branch-free, 1 warp-vote skip")
    ap.add_argument("--lanes", type=int, default=0)
    ap.add_argument("--agents-per-thread", type=int, default=0)
    ap.add_argument("--stage", type=int, default=-1)
    ap.add_argument("--max-ctas", type=int, default=0)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-all-configs", action="store_true", help="skip the all_configs key (every config + the sweep)")
    ap.add_argument("--rows", default="", help="comma-separated rows for all_configs (default: all of them)")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


def make_scene(name: str, seed: int = 0):
    from paper_2606_12579_b200 import scenes
    if name.startswith("sweep:"):
        a, s = name[6:].split("x")
        return scenes.config5(int(a), int(s), seed=seed)
    return getattr(scenes, name)(seed=seed)


# ------------------------------------------------------------------------------------------ clocks
class ClockSampler:
    """Samples SM clock and throttle reasons through NVML during the timed region."""

    def __init__(self, index: int):
        self.samples, self.reasons, self.max_mhz, self._stop = [], set(), None, threading.Event()
        self.ok = False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
            self.ok = True
        except Exception as e:          # NVML missing: report that, do not fail the bench
            self.err = repr(e)

    def _run(self):
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    r = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:
                    r = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for bit, nm in names.items():
                    if r & bit:
                        self.reasons.add(nm)
            except Exception:
                pass
            self._stop.wait(0.002)

    def __enter__(self):
        if self.ok:
            self.t = threading.Thread(target=self._run, daemon=True)
            self.t.start()
        return self

    def __exit__(self, *a):
        if self.ok:
            self._stop.set()
            self.t.join()

    def summary(self):
        if not self.ok or not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": self.max_mhz, "reasons": [], "note": "NVML unavailable"}
        return {"sm_mhz": float(np.median(self.samples)), "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(self.samples)}


# ------------------------------------------------------------------------------------------ oracle legs
def oracle_rate(scene, target_seconds: float):
    """Time the FP64 oracle, as it stands, on the host cores over a bounded sample of `scene`: a seeded random sample
    of n agents, all spheres, all rollout steps.
    Returns (interactions/s, cores, sample text, seconds)."""
    from oracle import oracle
    cores = oracle.max_threads()
    n_all = scene.n_agents
    order = np.random.default_rng(12579).permutation(n_all)
    probe = min(n_all, cores)
    t0 = time.perf_counter()
    oracle.rollout_scene(scene, threads=cores, agent_slice=np.sort(order[:probe]))
    t_probe = max(time.perf_counter() - t0, 1e-4)
    n = int(min(n_all, max(probe, (target_seconds / t_probe) * probe)))
    n = max(cores, (n // cores) * cores) if n >= cores else n
    # when the whole workload takes less than the target, repeat it so the sample is still ~target seconds of CPU work
    t_est = t_probe * n / probe
    reps = int(max(1, min(50, round(target_seconds / max(t_est, 1e-3))))) if n == n_all else 1
    idx = np.sort(order[:n])
    t0 = time.perf_counter()
    for _ in range(reps):
        oracle.rollout_scene(scene, threads=cores, agent_slice=idx)
    dt = time.perf_counter() - t0
    pairs = float(n) * scene.n_spheres * scene.steps * reps
    sample = (f"random {n} of {n_all} agents (seeded) x {scene.n_spheres} spheres x {scene.steps} steps, OpenMP over agents"
              + (f", repeated {reps}x" if reps > 1 else ""))
    return pairs / dt, cores, sample, dt


def oracle_spot_check(api, scene, g_final, g_collided, n_sample: int = 16):
    """Ties a timed row to a correct result: the GPU's final states / collision flags of `n_sample` randomly chosen
    agents (seeded) against the FP64 oracle run on exactly those agents (agent independence, pin P12).  Agents whose
    ORACLE trajectory moves by more than 1e-5 m under a one-ulp perturbation of the start position are counted as
    ill-conditioned and excluded from the error maximum (0 on every BASELINE config 1-4)."""
    from oracle import oracle
    import copy
    n = scene.n_agents
    idx = np.sort(np.random.default_rng(2606).choice(n, min(n_sample, n), replace=False))
    cores = oracle.max_threads()
    o = oracle.rollout_scene(scene, threads=cores, agent_slice=idx)
    s2 = copy.copy(scene)
    k = np.float32(1.0 + 2.0 ** -23)
    if scene.kind == 0:
        s2.agents = scene.agents.copy(); s2.agents[:, :3] *= k
        o2 = oracle.rollout_scene(s2, threads=cores, agent_slice=idx)
        po, po2 = o["final"][:, :3], o2["final"][:, :3]
        pg = g_final[idx, :3].astype(np.float64)
    else:
        s2.pos = scene.pos * k
        o2 = oracle.rollout_scene(s2, threads=cores, agent_slice=idx)
        po, po2 = o["p"], o2["p"]
        pg = api.state14_to_pose(g_final[idx])[1]
    good = np.abs(po2 - po).max(axis=1) <= 1e-5
    perr = np.abs(pg - po).max(axis=1)
    waive = (o["margins"][:, 2] < 1e-6 * scene.gains["r_influence"]) | ~good
    flags_ok = bool(np.array_equal(g_collided[idx][~waive], o["collided"][~waive]))
    return {"agents": int(idx.size), "max_pos_err_m": float(perr[good].max(initial=0.0)),
            "pos_tol_m": 1e-4, "collision_flags_equal": flags_ok, "ill_conditioned": int((~good).sum()),
            "collided_in_sample": int(o["collided"].sum()), "finite": bool(np.all(np.isfinite(g_final)))}


def measured_hbm_gbs():
    """HBM copy bandwidth of this pool's B200s: MEASURED_PEAKS.json (driver-written) or the profiling guide's fallback."""
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "MEASURED_PEAKS.json hbm_gbs"
    except Exception:
        return 6650.0, "of fallback (B200_PROFILING.md: 6.65 TB/s)"


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    scene = make_scene(args.config)
    per_step = max(2.0, min(args.cpu_seconds, 150.0 / max(1, args.steps + args.warmup)))
    rates, secs, info = [], [], None
    for i in range(args.warmup + args.steps):
        r, cores, sample, dt = oracle_rate(scene, per_step)
        if i >= args.warmup:
            rates.append(r); secs.append(dt)
        info = (cores, sample)
    value = float(np.mean(rates))
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": float(np.mean(secs) * 1e3),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": scene.name, "n_agents": scene.n_agents, "n_spheres": scene.n_spheres,
                   "rollout_steps": scene.steps, "note": "each step times a bounded sample of the workload"},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle", "sample": info[1]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------ our arm
def scaled_scene(name: str, world: int):
    """Weak scaling: the global problem has world x the config's agents; the sphere world is replicated."""
    from paper_2606_12579_b200 import scenes
    if world == 1:
        return make_scene(name)
    if name.startswith("sweep:"):
        a, s = name[6:].split("x")
        return scenes.config5(int(a) * world, int(s))
    base = {"config1": 16, "config2": 64, "config3": 1024, "config4": 256}[name]
    if name == "config1":
        raise SystemExit("config1 is fully specified (16 agents) and is not a multi-GPU workload")
    return getattr(scenes, name)(n_agents=base * world)


def measure_row(api, scenes_mod, name, dev, flush, K, check: bool):
    """One all_configs row: the workload `name` on its own context, default launch selection, branch-free kernel.
    kernel_ms = mean CUDA-event time of the rollout launch; cycle_ms = rollout + selection + result download."""
    import torch
    scene = make_scene(name)
    kind = scene.kind
    if kind == scenes_mod.KIND_POINT3:
        h_agents, goal = np.ascontiguousarray(scene.agents), scene.goal
    else:
        h_agents = api.pose_to_state14(scene.quat, scene.pos, scene.twist)
        goal = api.pose_to_state14(scene.goal_quat, scene.goal, np.zeros(6))[0, :8]
    ctx = api.Context(max_agents=scene.n_agents, max_spheres=max(scene.n_spheres, 1), device=dev.index or 0)
    d_xyzr = torch.from_numpy(scene.xyzr).to(dev)
    d_vel = None if scene.vel is None else torch.from_numpy(scene.vel).to(dev)
    ctx.set_obstacles(d_xyzr, d_vel, n=scene.n_spheres)
    d_agents = torch.from_numpy(h_agents).to(dev)
    d_out = torch.empty_like(d_agents)
    gains = api.make_gains(scene.gains)
    for _ in range(3):
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        ctx.best_agent_ex(scene.alpha, scene.prev_best)
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    torch.cuda.synchronize(dev)
    for i in range(K):                                       # the rollout kernel alone
        flush.zero_()
        ev[i][0].record()
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        ev[i][1].record()
    torch.cuda.synchronize(dev)
    for i in range(K):                                       # the cycle: rollout + selection, nothing recorded in between
        flush.zero_()
        ev[i][2].record()
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        best = ctx.best_agent_ex(scene.alpha, scene.prev_best)
        ev[i][3].record()
    torch.cuda.synchronize(dev)
    kernel_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
    cycle_ms = float(np.mean([e[2].elapsed_time(e[3]) for e in ev]))
    pairs = float(scene.n_agents) * scene.n_spheres * scene.steps
    info = ctx.launch_info()
    row = {"workload": scene.name, "n_agents": scene.n_agents, "n_spheres": scene.n_spheres, "rollout_steps": scene.steps,
           "kernel_ms": kernel_ms, "cycle_ms": cycle_ms, "interactions_per_s": pairs / (cycle_ms * 1e-3),
           "kernel_interactions_per_s": pairs / (kernel_ms * 1e-3),
           "frac": pairs * FLOP_PER_PAIR / (kernel_ms * 1e-3) / 1e12 / PEAK_TFLOPS,
           "us_per_rollout_step": kernel_ms * 1e3 / scene.steps, "best_index": int(best[0]),
           "launch": {k: info[k] for k in ("grid", "block", "lanes_per_agent", "agents_per_thread", "agents_per_cta",
                                           "stage", "tile_spheres", "n_tiles", "smem_bytes", "regs_per_thread", "packed_x2",
                                           "selection_fused")}}
    if scene.vel is not None:
        row["frac_moving_lane_ops"] = (pairs * LANE_OPS_PER_PAIR_MOVING / (kernel_ms * 1e-3)
                                       / (NOMINAL_SMS * LANES_PER_SM * MAX_GHZ * 1e9))
        row["frac_note"] = ("moving spheres: `frac` counts the 35 flop of a STATIC pair; frac_moving_lane_ops counts the 36 "
                            "FP32-pipe lane-operations of a moving pair against 148 x 128 lanes x 1.965 GHz")
    if check:
        col = torch.empty(scene.n_agents, dtype=torch.int32, device=dev)
        ctx.get_results(None, None, col)
        torch.cuda.synchronize(dev)
        row["oracle_check"] = oracle_spot_check(api, scene, d_out.cpu().numpy(), col.cpu().numpy())
    ctx.close()
    del d_xyzr, d_vel, d_agents, d_out
    return row


def run_all_configs(api, scenes_mod, dev, flush, rows, check: bool):
    out = {"note": "every BASELINE.json config and the 3 x 3 stress sweep (config 5) plus three agent counts between the grid "
                   "points; default launch selection, branch-free kernel (cull=0), L2 flushed between timed iterations; "
                   "frac = 35 flop x pairs / kernel time / 74.45 TFLOP/s; oracle_check = FP64 oracle on 16 seeded random agents",
           "rows": {}}
    for name in rows:
        big = name.startswith("sweep:") and int(name[6:].split("x")[0]) * int(name[6:].split("x")[1]) >= (1 << 28)
        out["rows"][name] = measure_row(api, scenes_mod, name, dev, flush, 3 if big else 5, check)
    return out


def run_ours(args):
    import torch
    import torch.distributed as dist
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if world != args.gpus:
        raise SystemExit(f"--gpus {args.gpus} but WORLD_SIZE={world}: launch with torch.distributed.run --nproc-per-node {args.gpus}")
    # GMAPP_BENCH_BACKEND=gloo: smoke test of the multi-rank code path on a box with fewer GPUs than ranks (the ranks'
    # kernels are independent of each other; only the 24-byte winner exchange goes through the backend).  Never a bench number.
    backend = os.environ.get("GMAPP_BENCH_BACKEND", "nccl")
    n_dev = torch.cuda.device_count()
    if backend == "nccl" and local_rank >= n_dev:
        raise SystemExit(f"rank {rank}: LOCAL_RANK {local_rank} but only {n_dev} CUDA devices")
    local_rank = local_rank % max(n_dev, 1)
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    red_dev = dev if backend == "nccl" else torch.device("cpu")     # where the max-over-ranks reductions live
    if world > 1:
        if backend == "nccl":
            dist.init_process_group("nccl", device_id=dev)
        else:
            dist.init_process_group(backend)
    from paper_2606_12579_b200 import api, scenes, sharding

    scene = scaled_scene(args.config, world)
    lo, hi = sharding.shard_range(scene.n_agents, rank, world)
    kind = scene.kind
    if kind == scenes.KIND_POINT3:
        h_agents = np.ascontiguousarray(scene.agents[lo:hi]); goal = scene.goal
    else:
        h_agents = api.pose_to_state14(scene.quat[lo:hi], scene.pos[lo:hi], scene.twist[lo:hi])
        goal = api.pose_to_state14(scene.goal_quat, scene.goal, np.zeros(6))[0, :8]
    n_local = hi - lo
    pairs_local = float(n_local) * scene.n_spheres * scene.steps
    pairs_global = float(scene.n_agents) * scene.n_spheres * scene.steps
    gains = api.make_gains(scene.gains)

    ctx = api.Context(max_agents=n_local, max_spheres=max(scene.n_spheres, 1), device=local_rank)
    tune = dict(lanes_per_agent=args.lanes, agents_per_thread=args.agents_per_thread, cull=args.cull, stage=args.stage,
                max_ctas=args.max_ctas)
    ctx.set_tuning(**tune)
    d_xyzr = torch.from_numpy(scene.xyzr).to(dev)
    d_vel = None if scene.vel is None else torch.from_numpy(scene.vel).to(dev)
    ctx.set_obstacles(d_xyzr, d_vel, n=scene.n_spheres)
    d_agents = torch.from_numpy(h_agents).to(dev)
    d_out = torch.empty_like(d_agents)
    flush = torch.empty(256 * 1024 * 1024, dtype=torch.uint8, device=dev)      # > 126 MB L2

    # the incumbent as a local index on the rank that owns it (-1 elsewhere); the rollout's fused selection tail is armed
    # with it, and with several ranks the hysteresis rule is applied once, after the all_gather (sharding.py)
    prev_local = sharding.local_prev(scene.prev_best, lo, hi)
    ctx.set_selection(scene.alpha, prev_local)

    def select():
        if world == 1:
            idx, cost, _ = ctx.best_agent_ex(scene.alpha, prev_local)
            return idx, cost
        raw, inc = sharding.selection_keys(ctx.select(scene.alpha, prev_local), lo, prev_local)
        key = sharding.all_gather_best(raw, inc, scene.alpha)
        return key[2], key[1]

    def cycle():
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        return select()

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    K, W = args.steps, max(args.warmup, 3)
    for _ in range(W):
        flush.zero_(); cycle()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(K)]
    sampler = ClockSampler(local_rank)
    barrier()
    t_wall0 = time.perf_counter()
    with sampler:
        for i in range(K):
            flush.zero_()                                    # L2 flush between timed iterations (untimed);
            ev[i][0].record()                                # the cycle is queued behind it: no idle-GPU host gap
            ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
            idx, cost = select()                             # selection (dependent launch or fused tail); the host polls its record
            ev[i][2].record()
        barrier()
    wall_ms = (time.perf_counter() - t_wall0) * 1e3
    step_ms = np.array([e[0].elapsed_time(e[2]) for e in ev])
    total_ms = float(step_ms.sum())
    if world > 1:
        t = torch.tensor([total_ms], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        total_ms = float(t.item())
    info = ctx.launch_info()
    launches = K * (info["kernels_launched"] + (0 if info["selection_fused"] else 1))

    # ---- roofline of the dominant kernel (the rollout), branch-free variant: every pair does the full math
    ctx.set_tuning(**{**tune, "cull": 0})
    for _ in range(3):
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
    rev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(K)]
    torch.cuda.synchronize(dev)
    sampler2 = ClockSampler(local_rank)               # clocks under the roofline loop as well
    sampler2.__enter__()
    for i in range(K):
        flush.zero_()
        rev[i][0].record()
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        rev[i][1].record()
    torch.cuda.synchronize(dev)
    bf_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in rev]))
    info_bf = ctx.launch_info()
    achieved = pairs_local * FLOP_PER_PAIR / (bf_ms * 1e-3) / 1e12
    # ---- the warp-vote variant (cull=1: the force math is skipped where no lane's pair is inside r_d; results
    # are bit-identical).  Reported beside the headline, never as the roofline numerator.
    ctx.set_tuning(**{**tune, "cull": 1})
    for _ in range(3):
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
    torch.cuda.synchronize(dev)
    for i in range(K):
        flush.zero_()
        rev[i][0].record()
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        rev[i][1].record()
    torch.cuda.synchronize(dev)
    cull_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in rev]))
    ctx.set_tuning(**tune)
    peak_meas = ctx.measure_fp32_peak(False)
    peak_meas_x2 = ctx.measure_fp32_peak(True)

    # ---- planning-cycle latency distribution: 20 warm-ups, 200 timed cycles, host wall clock of
    # gmapp_rollout + gmapp_best_agent (launch + execution + sync + 12-byte download), spheres resident, no L2 flush
    for _ in range(20):
        cycle()
    lat = []
    for _ in range(200):
        torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        ctx.rollout(kind, d_agents, d_out, goal, gains, scene.dt, scene.steps)
        ctx.best_agent_ex(scene.alpha, prev_local)
        lat.append((time.perf_counter() - t0) * 1e3)
    lat = np.array(lat)
    sampler2.__exit__()
    sampler.samples += sampler2.samples; sampler.reasons |= sampler2.reasons

    # ---- closed-loop re-planning (gmapp_replan): cycles chained on the device, no host synchronisation inside
    n_cyc, exec_steps = 50, max(1, scene.steps // 10)
    d_loop = d_agents.clone()
    ctx.replan(kind, d_loop, goal, gains, scene.dt, scene.steps, exec_steps, 3)
    torch.cuda.synchronize(dev)
    d_loop.copy_(d_agents)
    rp0, rp1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    rp0.record()
    ctx.replan(kind, d_loop, goal, gains, scene.dt, scene.steps, exec_steps, n_cyc)
    rp1.record()
    torch.cuda.synchronize(dev)
    replan_ms = rp0.elapsed_time(rp1) / n_cyc
    # the same 50 cycles captured once as a CUDA graph and replayed
    side = torch.cuda.Stream(device=dev)
    side.wait_stream(torch.cuda.current_stream(dev))
    with torch.cuda.stream(side):
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=side):
            ctx.replan(kind, d_loop, goal, gains, scene.dt, scene.steps, exec_steps, n_cyc)
    torch.cuda.synchronize(dev)
    d_loop.copy_(d_agents)
    graph.replay(); torch.cuda.synchronize(dev)
    d_loop.copy_(d_agents)
    rp0.record(); graph.replay(); rp1.record()
    torch.cuda.synchronize(dev)
    replan_graph_ms = rp0.elapsed_time(rp1) / n_cyc
    del graph

    # ---- sphere-world builder (gmapp_build_sphere_world) on a separate context: 2 x 848 x 480 points (the paper's two
    # depth cameras), 4 cm voxels; HBM-bound (12 B read per point)
    vox = None
    if world == 1:
        pts, lo_w, hi_w = scenes.depth_cloud(seed=0, n_points=2 * 848 * 480)
        d_pts = torch.from_numpy(pts).to(dev)
        vctx = api.Context(max_agents=1, max_spheres=32768, device=local_rank)
        for _ in range(3):
            vctx.build_sphere_world(d_pts, lo_w, hi_w, 0.04, 32768)
        ve = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(20)]
        torch.cuda.synchronize(dev)
        for a, b in ve:
            flush.zero_()
            a.record(); vctx.build_sphere_world(d_pts, lo_w, hi_w, 0.04, 32768); b.record()
        torch.cuda.synchronize(dev)
        vms = float(np.mean([a.elapsed_time(b) for a, b in ve]))
        hbm, hbm_how = measured_hbm_gbs()
        vox = {"points": int(pts.shape[0]), "ms": vms, "GB_per_s": pts.nbytes / (vms * 1e-3) / 1e9,
               "frac_of_hbm": pts.nbytes / (vms * 1e-3) / 1e9 / hbm, "hbm_peak_GB_per_s": hbm, "hbm_peak_how": hbm_how,
               "algorithmic_bytes": int(pts.nbytes),
               "note": "ONE launch (k_vox_build_small: per-block voxel bitmaps in shared memory, 12 B read per point; the block that "
                       "finishes last scans the merged bitmap and emits the spheres in both layouts, the sentinel tail and the count); "
                       "grids beyond 262144 voxels: mark + compact, 2 launches; bit-exact vs oracle/voxel.py"}
        vctx.close()

    # ---- end to end through the C ABI with HOST buffers (sphere + agent upload, 8-byte result download)
    for _ in range(3):
        ctx.plan_cycle_host(kind, h_agents, goal, gains, scene.dt, scene.steps, h_xyzr=scene.xyzr, h_vel=scene.vel,
                            alpha=scene.alpha, prev_best=prev_local)
    barrier()
    e2e_s = 0.0
    for i in range(K):
        flush.zero_(); torch.cuda.synchronize(dev)
        t0 = time.perf_counter()
        idx_e, cost_e = ctx.plan_cycle_host(kind, h_agents, goal, gains, scene.dt, scene.steps, h_xyzr=scene.xyzr,
                                            h_vel=scene.vel, alpha=scene.alpha, prev_best=prev_local)
        if world > 1:
            raw_e, inc_e = sharding.selection_keys(ctx.select(scene.alpha, prev_local), lo, prev_local)
            idx_e = sharding.all_gather_best(raw_e, inc_e, scene.alpha)[2]
        e2e_s += time.perf_counter() - t0
    if world > 1:
        t = torch.tensor([e2e_s], dtype=torch.float64, device=red_dev)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        e2e_s = float(t.item())
    h2d = scene.xyzr.nbytes + (0 if scene.vel is None else scene.vel.nbytes) + h_agents.nbytes
    d2h = 36

    if rank == 0:
        line = {
            "metric": METRIC, "value": pairs_global * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world,
            "steps": K, "warmup": W, "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": scene.name, "n_agents": scene.n_agents, "n_spheres": scene.n_spheres,
                       "rollout_steps": scene.steps, "agents_per_gpu": n_local, "parallelism": f"agents x{world}",
                       "l2": "flushed between timed iterations (256 MB write, untimed)",
                       "step": "one planning cycle: rollout kernel + selection (a dependent launch behind the packed kernels, fused "
                               "into the tail of the wide 6D kernel) + its 36-byte record polled in pinned memory",
                       "launch": info},
            "planning_cycle_latency_ms": {"device_p50": float(np.percentile(step_ms, 50)),
                                          "device_p99": float(np.percentile(step_ms, 99)),
                                          "rollout_kernel_mean": bf_ms,
                                          "host_200_warm": {"p50": float(np.percentile(lat, 50)), "p99": float(np.percentile(lat, 99)),
                                                            "min": float(lat.min()), "runs": 200}},
            "wall_ms_per_step_incl_flush": wall_ms / K,
            "e2e": {"value": pairs_global * K / e2e_s, "unit": UNIT, "h2d_bytes_per_step": int(h2d),
                    "d2h_bytes_per_step": int(d2h), "ms_per_step": e2e_s / K * 1e3,
                    "call": "gmapp_plan_cycle_host (host spheres + agents in, best index out; the packing and rollout kernels read the pinned host buffers over the host link themselves, the rollout's selection tail writes its record to pinned memory)"},
            "gpu_launches": int(launches),
            "roofline": {"bound": "alu", "achieved": achieved, "peak": PEAK_TFLOPS, "unit": "TFLOP/s",
                         "frac": achieved / PEAK_TFLOPS, "traffic": TRAFFIC_BYTES_PER_LAUNCH.get(args.config) if world == 1 else None,
                         "traffic_source": TRAFFIC_SOURCE.get(args.config, "null: no committed ncu --set full capture of this workload "
                                                              "(dram bytes cannot be read outside a profiler)"),
                         "kernel": ("k_rollout_x2" if info_bf["packed_x2"] else "k_rollout / k_rollout_wide")
                                   + " (branch-free variant, cull=0; the persistent rollout kernel, one launch per cycle)",
                         "kernel_ms": bf_ms,
                         "distance_refinement": "two-pass: raw MUFU.RSQ sweep, Newton step only for a warp within R/16 of a surface "
                                                "(neither is part of the 35 flop per pair; DESIGN.md section 6)",
                         "flop_per_pair": FLOP_PER_PAIR, "pairs_per_launch": pairs_local,
                         "peak_how": "148 SMs x 128 FP32 lanes x 2 x 1.965 GHz (guide unit counts, max clock)",
                         "peak_measured_ffma_tflops": peak_meas, "peak_measured_ffma2_tflops": peak_meas_x2,
                         "frac_of_measured_ffma": achieved / peak_meas if peak_meas else None,
                         "launch": info_bf},
            "replan": {"ms_per_cycle": replan_ms, "cycles_per_s": 1e3 / replan_ms, "cuda_graph_ms_per_cycle": replan_graph_ms, "cycles": n_cyc, "exec_steps": exec_steps,
                       "note": "gmapp_replan: rollout + selection + restart chained on the device (the paper's control "
                               "loop runs at ~100 Hz, PAPER.md:47)"},
            "sphere_world_builder": vox,
            "cull_variant": {"kernel_ms": cull_ms, "interactions_per_s": pairs_local / (cull_ms * 1e-3),
                             "note": "same kernel with the warp-vote skip of the force math (tuning cull=1); "
                                     "bit-identical results; not used for the roofline"},
            "clocks": sampler.summary(),
        }
        if world == 1 and not args.no_all_configs:
            rows = [r for r in args.rows.split(",") if r] or ALL_CONFIG_ROWS
            line["all_configs"] = run_all_configs(api, scenes, dev, flush, rows, check=not args.no_cpu_baseline)
            # the headline scene (config 3) keeps every agent > 0.1 m from any surface, so its force sweeps all run on the raw
            # MUFU.RSQ distance: the best case of the two-pass refinement.  The same kernel with most warps in the REFINED
            # mode (the Newton step is not part of the 35 algorithmic flop) is the dense stress scene below.
            dense = line["all_configs"]["rows"].get("sweep:1024x4096")
            if dense:
                line["roofline"]["refined_case"] = {
                    "workload": dense["workload"], "kernel_ms": dense["kernel_ms"], "frac": dense["frac"],
                    "achieved": dense["frac"] * PEAK_TFLOPS, "launch": dense["launch"],
                    "note": "same launch shape and kernel as the headline on the config-5 scene of the same size (spheres fill 6 % of the "
                            "cube, agents start among them: warps switch to the refined sweep while an agent is within R/16 of a surface)"}
        if world == 1 and not args.no_cpu_baseline:
            r, cores, sample, dt = oracle_rate(scene, args.cpu_seconds)
            line["cpu_baseline"] = {"value": r, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample,
                                    "seconds": dt}
        print(json.dumps(line), flush=True)
    ctx.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    args = parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
