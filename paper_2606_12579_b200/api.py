"""Thin ctypes binding of libgmapp.so (include/gmapp.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels behind the C ABI.  PyTorch supplies device memory and streams.

There is NO CPU fallback: if libgmapp.so is missing or fails to load, importing this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_PKG = os.path.dirname(os.path.abspath(__file__))
_CSRC = os.path.join(_PKG, "csrc")
_SO = os.path.join(_PKG, "libgmapp.so")
_INCLUDE = os.path.join(os.path.dirname(_PKG), "include")

GMAPP_OK, GMAPP_EINVAL, GMAPP_ECAPACITY, GMAPP_ESTATE, GMAPP_ECUDA = 0, 1, 2, 3, 4
GMAPP_POINT3, GMAPP_MOTOR6 = 0, 1
STATUS_NAMES = {0: "GMAPP_OK", 1: "GMAPP_EINVAL", 2: "GMAPP_ECAPACITY", 3: "GMAPP_ESTATE", 4: "GMAPP_ECUDA"}

_GAIN_FIELDS = ["k_circ", "k_att", "k_damp", "k_att_rot", "k_damp_rot", "inv_mass", "inv_inertia",
                "vel_factor", "r_influence", "r_agent", "eps_dist", "w_goal", "w_obs", "w_path",
                "w_smooth", "r_cost_goal", "r_cost_obs", "a_max"]


class gmapp_gains(C.Structure):
    _fields_ = [(k, C.c_float) for k in _GAIN_FIELDS] + [("heuristic", C.c_int32)]


class gmapp_tuning(C.Structure):
    _fields_ = [("lanes_per_agent", C.c_int32), ("agents_per_thread", C.c_int32), ("cull", C.c_int32),
                ("stage", C.c_int32), ("max_ctas", C.c_int32), ("scalar_path", C.c_int32), ("reserved", C.c_int32 * 2)]


class gmapp_selection(C.Structure):
    _fields_ = [("index", C.c_int32), ("collided", C.c_int32), ("cost", C.c_float),
                ("raw_index", C.c_int32), ("raw_collided", C.c_int32), ("raw_cost", C.c_float),
                ("prev_collided", C.c_int32), ("prev_cost", C.c_float)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class gmapp_launch_info(C.Structure):
    _fields_ = [(k, C.c_int32) for k in
                ("grid", "block", "lanes_per_agent", "agents_per_thread", "agents_per_cta", "cull", "stage",
                 "tile_spheres", "n_tiles", "smem_bytes", "regs_per_thread", "kernels_launched", "packed_x2", "selection_fused")]

    def as_dict(self):
        return {k: int(getattr(self, k)) for k, _ in self._fields_}


EXPORTS = ["gmapp_default_gains", "gmapp_create", "gmapp_destroy", "gmapp_set_obstacles",
           "gmapp_set_obstacles_host", "gmapp_build_sphere_world", "gmapp_build_sphere_world_static", "gmapp_get_obstacles", "gmapp_set_tuning", "gmapp_set_agent_params", "gmapp_rollout", "gmapp_set_trajectory_output", "gmapp_replan", "gmapp_best_agent", "gmapp_best_agent_ex", "gmapp_select", "gmapp_set_selection",
           "gmapp_forces",
           "gmapp_get_results", "gmapp_plan_cycle_host", "gmapp_get_launch_info", "gmapp_measure_fp32_peak", "gmapp_microbench",
           "gmapp_sm_count", "gmapp_last_error"]


def build(force: bool = False) -> str:
    """Compile libgmapp.so in-tree for sm_100a (paper_2606_12579_b200/build_lib.py; nvcc cross-compiles without a GPU)."""
    from . import build_lib
    return build_lib.build(force=force)


def _load():
    if not os.path.exists(_SO):
        raise ImportError(f"{_SO} is missing: build it with __graft_entry__.build() "
                          "(paper_2606_12579_b200.api.build()); there is no CPU fallback")
    lib = C.CDLL(_SO)
    vp, ip, fp = C.c_void_p, C.POINTER(C.c_int), C.POINTER(C.c_float)
    lib.gmapp_default_gains.argtypes = [C.POINTER(gmapp_gains)]; lib.gmapp_default_gains.restype = None
    lib.gmapp_create.argtypes = [C.POINTER(vp), C.c_int, C.c_int, C.c_int]
    lib.gmapp_destroy.argtypes = [vp]
    lib.gmapp_set_obstacles.argtypes = [vp, vp, vp, C.c_int, vp]
    lib.gmapp_set_obstacles_host.argtypes = [vp, vp, vp, C.c_int, vp]
    lib.gmapp_build_sphere_world.argtypes = [vp, vp, C.c_int, fp, fp, C.c_float, C.c_int, vp, vp]
    lib.gmapp_build_sphere_world_static.argtypes = [C.c_int, vp, C.c_int, fp, fp, C.c_float, C.c_int, vp, vp, vp]
    lib.gmapp_get_obstacles.argtypes = [vp, vp, C.c_int, vp]
    lib.gmapp_set_tuning.argtypes = [vp, C.POINTER(gmapp_tuning)]
    lib.gmapp_set_agent_params.argtypes = [vp, vp, vp, vp, C.c_int, vp]
    lib.gmapp_rollout.argtypes = [vp, C.c_int, vp, vp, C.c_int, fp, C.POINTER(gmapp_gains), C.c_float, C.c_int, vp]
    lib.gmapp_set_trajectory_output.argtypes = [vp, vp]
    lib.gmapp_replan.argtypes = [vp, C.c_int, vp, C.c_int, fp, C.POINTER(gmapp_gains), C.c_float, C.c_int, C.c_int, C.c_float,
                                 C.c_int, C.c_int, vp, vp, vp]
    lib.gmapp_best_agent.argtypes = [vp, C.c_float, C.c_int, ip, fp, vp]
    lib.gmapp_best_agent_ex.argtypes = [vp, C.c_float, C.c_int, ip, fp, ip, vp]
    lib.gmapp_select.argtypes = [vp, C.c_float, C.c_int, C.POINTER(gmapp_selection), vp]
    lib.gmapp_set_selection.argtypes = [vp, C.c_float, C.c_int]
    lib.gmapp_forces.argtypes = [vp, C.c_int, vp, C.c_int, fp, C.POINTER(gmapp_gains), C.c_float, vp, vp, vp]
    lib.gmapp_get_results.argtypes = [vp, vp, vp, vp, vp]
    lib.gmapp_plan_cycle_host.argtypes = [vp, C.c_int, vp, vp, C.c_int, vp, vp, C.c_int, fp, C.POINTER(gmapp_gains),
                                          C.c_float, C.c_int, C.c_float, C.c_int, ip, fp, vp]
    lib.gmapp_get_launch_info.argtypes = [vp, C.POINTER(gmapp_launch_info)]
    lib.gmapp_measure_fp32_peak.argtypes = [vp, C.c_int, fp, vp]
    lib.gmapp_microbench.argtypes = [vp, C.c_int, fp, vp]
    lib.gmapp_sm_count.argtypes = [vp]; lib.gmapp_sm_count.restype = C.c_int
    lib.gmapp_last_error.argtypes = [vp]; lib.gmapp_last_error.restype = C.c_char_p
    for name in EXPORTS:
        getattr(lib, name)          # raises AttributeError if a declared symbol is not exported
    return lib


_lib = _load()


class GmappError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__(f"{STATUS_NAMES.get(status, status)}: {msg}")
        self.status = status


def make_gains(g=None) -> gmapp_gains:
    s = gmapp_gains()
    _lib.gmapp_default_gains(C.byref(s))
    if g:
        for k, v in g.items():
            setattr(s, k, int(v) if k == "heuristic" else float(v))
    return s


def _ptr(t):
    if t is None:
        return None
    return C.c_void_p(t.data_ptr())


def _farr(a, n):
    a = np.ascontiguousarray(a, dtype=np.float32).reshape(-1)
    assert a.size >= n
    return a.ctypes.data_as(C.POINTER(C.c_float)), a     # keep `a` alive in the caller


def _stream(stream):
    if stream is None:
        import torch
        stream = torch.cuda.current_stream().cuda_stream
    return C.c_void_p(int(stream))


def pose_to_state14(quat, pos, twist) -> np.ndarray:
    """Marshalling helper: (unit quaternion w,x,y,z; world position; body twist) -> [n][14] motor + twist,
    the GMAPP_MOTOR6 layout of include/gmapp.h (d = (1/2) t (x) r)."""
    q = np.asarray(quat, np.float64).reshape(-1, 4)
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    t = np.asarray(pos, np.float64).reshape(-1, 3)
    w, v = q[:, 0], q[:, 1:]
    dw = -0.5 * np.einsum("ij,ij->i", t, v)
    dv = 0.5 * (w[:, None] * t + np.cross(t, v))
    out = np.concatenate([q, dw[:, None], dv, np.asarray(twist, np.float64).reshape(-1, 6)], axis=1)
    return np.ascontiguousarray(out.astype(np.float32))


def state14_to_pose(state14):
    """Inverse marshalling helper: [n][14] -> (quat [n,4], pos [n,3], twist [n,6]) in float64."""
    s = np.asarray(state14, np.float64).reshape(-1, 14)
    r, d = s[:, :4], s[:, 4:8]
    rw, rv, dw, dv = r[:, 0], r[:, 1:], d[:, 0], d[:, 1:]
    t = 2.0 * (rw[:, None] * dv - dw[:, None] * rv + np.cross(rv, dv))
    return r.copy(), t, s[:, 8:].copy()


def build_sphere_world_static(d_points, lo, hi, pitch, capacity, d_xyzr_out, d_count_out=None, n_points=None, device=0,
                              stream=None):
    """gmapp_build_sphere_world_static: the allocation-free sphere-world builder (no context; scratch in a static device
    array of the library, at most 262 144 voxels).  d_xyzr_out: caller-owned device tensor [capacity][4]."""
    n = int(d_points.shape[0]) if n_points is None else n_points
    lp, k1 = _farr(lo, 3)
    hp, k2 = _farr(hi, 3)
    st = _lib.gmapp_build_sphere_world_static(int(device), _ptr(d_points), n, lp, hp, C.c_float(pitch), int(capacity),
                                              _ptr(d_xyzr_out), _ptr(d_count_out), _stream(stream))
    if st != GMAPP_OK:
        raise GmappError(st, _lib.gmapp_last_error(None).decode())


class Context:
    """Owns one gmapp_ctx.  Methods mirror the C entry points one to one."""

    def __init__(self, max_agents: int, max_spheres: int, device: int = 0):
        self._h = C.c_void_p()
        st = _lib.gmapp_create(C.byref(self._h), device, max_agents, max_spheres)
        if st != GMAPP_OK:
            raise GmappError(st, _lib.gmapp_last_error(None).decode())
        self.device = device

    def _check(self, st):
        if st != GMAPP_OK:
            raise GmappError(st, _lib.gmapp_last_error(self._h).decode())

    def close(self):
        if self._h:
            _lib.gmapp_destroy(self._h)
            self._h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @property
    def sm_count(self) -> int:
        return int(_lib.gmapp_sm_count(self._h))

    def set_obstacles(self, d_xyzr, d_vel=None, n=None, stream=None):
        n = int(d_xyzr.shape[0]) if n is None else n
        self._check(_lib.gmapp_set_obstacles(self._h, _ptr(d_xyzr), _ptr(d_vel), n, _stream(stream)))

    def set_obstacles_host(self, h_xyzr, h_vel=None, stream=None):
        x = np.ascontiguousarray(h_xyzr, dtype=np.float32)
        v = None if h_vel is None else np.ascontiguousarray(h_vel, dtype=np.float32)
        self._check(_lib.gmapp_set_obstacles_host(self._h, x.ctypes.data_as(C.c_void_p),
                                                  None if v is None else v.ctypes.data_as(C.c_void_p),
                                                  int(x.shape[0]), _stream(stream)))

    def build_sphere_world(self, d_points, lo, hi, pitch, capacity, d_count_out=None, n_points=None, stream=None):
        n = int(d_points.shape[0]) if n_points is None else n_points
        lp, k1 = _farr(lo, 3)
        hp, k2 = _farr(hi, 3)
        self._check(_lib.gmapp_build_sphere_world(self._h, _ptr(d_points), n, lp, hp, C.c_float(pitch), int(capacity),
                                                  _ptr(d_count_out), _stream(stream)))

    def get_obstacles(self, d_xyzr_out, n=None, stream=None):
        n = int(d_xyzr_out.shape[0]) if n is None else n
        self._check(_lib.gmapp_get_obstacles(self._h, _ptr(d_xyzr_out), n, _stream(stream)))

    def set_tuning(self, lanes_per_agent=0, agents_per_thread=0, cull=-1, stage=-1, max_ctas=0, scalar_path=0,
                   reset=False):
        if reset:
            self._check(_lib.gmapp_set_tuning(self._h, None))
            return
        t = gmapp_tuning(lanes_per_agent, agents_per_thread, cull, stage, max_ctas, scalar_path)
        self._check(_lib.gmapp_set_tuning(self._h, C.byref(t)))

    def set_agent_params(self, r_influence=None, k_circ=None, heuristic=None, n=None, stream=None):
        """Per-agent detection radius / gain / heuristic (host arrays, any None); all None or n == 0 clears."""
        arrs = [None if a is None else np.ascontiguousarray(a, dtype=dt)
                for a, dt in ((r_influence, np.float32), (k_circ, np.float32), (heuristic, np.int32))]
        if n is None:
            n = max([a.shape[0] for a in arrs if a is not None], default=0)
        for a in arrs:
            assert a is None or a.shape[0] >= n
        ptrs = [None if a is None else a.ctypes.data_as(C.c_void_p) for a in arrs]
        self._check(_lib.gmapp_set_agent_params(self._h, ptrs[0], ptrs[1], ptrs[2], int(n), _stream(stream)))

    def rollout(self, kind, d_agents, d_agents_out, goal, gains, dt, steps, n_agents=None, stream=None):
        n = int(d_agents.shape[0]) if n_agents is None else n_agents
        gp, keep = _farr(goal, 3 if kind == GMAPP_POINT3 else 8)
        g = gains if isinstance(gains, gmapp_gains) else make_gains(gains)
        self._check(_lib.gmapp_rollout(self._h, kind, _ptr(d_agents), _ptr(d_agents_out), n, gp, C.byref(g),
                                       C.c_float(dt), int(steps), _stream(stream)))

    def set_trajectory_output(self, d_traj=None):
        self._check(_lib.gmapp_set_trajectory_output(self._h, _ptr(d_traj)))

    def replan(self, kind, d_agents, goal, gains, dt, steps, exec_steps, n_cycles, alpha=0.9, prev_best=-1,
               d_path_out=None, d_best_out=None, n_agents=None, stream=None):
        n = int(d_agents.shape[0]) if n_agents is None else n_agents
        gp, keep = _farr(goal, 3 if kind == GMAPP_POINT3 else 8)
        g = gains if isinstance(gains, gmapp_gains) else make_gains(gains)
        self._check(_lib.gmapp_replan(self._h, kind, _ptr(d_agents), n, gp, C.byref(g), C.c_float(dt), int(steps),
                                      int(exec_steps), C.c_float(alpha), int(prev_best), int(n_cycles),
                                      _ptr(d_path_out), _ptr(d_best_out), _stream(stream)))

    def best_agent(self, alpha=0.9, prev_best=-1, stream=None):
        idx, cost = C.c_int(), C.c_float()
        self._check(_lib.gmapp_best_agent(self._h, C.c_float(alpha), int(prev_best), C.byref(idx), C.byref(cost),
                                          _stream(stream)))
        return idx.value, cost.value

    def best_agent_ex(self, alpha=0.9, prev_best=-1, stream=None):
        idx, cost, col = C.c_int(), C.c_float(), C.c_int()
        self._check(_lib.gmapp_best_agent_ex(self._h, C.c_float(alpha), int(prev_best), C.byref(idx), C.byref(cost),
                                             C.byref(col), _stream(stream)))
        return idx.value, cost.value, col.value

    def select(self, alpha=0.9, prev_best=-1, stream=None) -> dict:
        rec = gmapp_selection()
        self._check(_lib.gmapp_select(self._h, C.c_float(alpha), int(prev_best), C.byref(rec), _stream(stream)))
        return rec.as_dict()

    def set_selection(self, alpha=0.9, prev_best=-1):
        self._check(_lib.gmapp_set_selection(self._h, C.c_float(alpha), int(prev_best)))

    def forces(self, kind, d_agents, goal, gains, t_obstacles, d_f_rep, d_f_total, n_agents=None, stream=None):
        n = int(d_agents.shape[0]) if n_agents is None else n_agents
        gp, keep = _farr(goal, 3 if kind == GMAPP_POINT3 else 8)
        g = gains if isinstance(gains, gmapp_gains) else make_gains(gains)
        self._check(_lib.gmapp_forces(self._h, kind, _ptr(d_agents), n, gp, C.byref(g), C.c_float(t_obstacles),
                                      _ptr(d_f_rep), _ptr(d_f_total), _stream(stream)))

    def get_results(self, d_cost=None, d_min_clearance=None, d_collided=None, stream=None):
        self._check(_lib.gmapp_get_results(self._h, _ptr(d_cost), _ptr(d_min_clearance), _ptr(d_collided),
                                           _stream(stream)))

    def plan_cycle_host(self, kind, h_agents, goal, gains, dt, steps, h_xyzr=None, h_vel=None, alpha=0.9,
                        prev_best=-1, h_agents_out=None, stream=None):
        a = np.ascontiguousarray(h_agents, dtype=np.float32)
        x = None if h_xyzr is None else np.ascontiguousarray(h_xyzr, dtype=np.float32)
        v = None if h_vel is None else np.ascontiguousarray(h_vel, dtype=np.float32)
        gp, keep = _farr(goal, 3 if kind == GMAPP_POINT3 else 8)
        g = gains if isinstance(gains, gmapp_gains) else make_gains(gains)
        idx, cost = C.c_int(), C.c_float()
        if h_agents_out is not None:
            assert h_agents_out.dtype == np.float32 and h_agents_out.flags.c_contiguous
        self._check(_lib.gmapp_plan_cycle_host(
            self._h, kind, a.ctypes.data_as(C.c_void_p),
            None if h_agents_out is None else h_agents_out.ctypes.data_as(C.c_void_p), int(a.shape[0]),
            None if x is None else x.ctypes.data_as(C.c_void_p), None if v is None else v.ctypes.data_as(C.c_void_p),
            -1 if x is None else int(x.shape[0]), gp, C.byref(g), C.c_float(dt), int(steps), C.c_float(alpha),
            int(prev_best), C.byref(idx), C.byref(cost), _stream(stream)))
        return idx.value, cost.value

    def launch_info(self) -> dict:
        info = gmapp_launch_info()
        self._check(_lib.gmapp_get_launch_info(self._h, C.byref(info)))
        return info.as_dict()

    def microbench(self, kind: int, stream=None) -> float:
        out = C.c_float()
        self._check(_lib.gmapp_microbench(self._h, int(kind), C.byref(out), _stream(stream)))
        return out.value

    def measure_fp32_peak(self, use_f32x2=False, stream=None) -> float:
        out = C.c_float()
        self._check(_lib.gmapp_measure_fp32_peak(self._h, int(bool(use_f32x2)), C.byref(out), _stream(stream)))
        return out.value


MICROBENCH_KINDS = ["FFMA, three distinct registers", "FFMA2, three distinct register pairs", "FFMA2, two distinct register pairs",
                    "FFMA2, broadcast operand {a,a}", "MUFU.RCP (+ a co-issued FADD)", "MUFU.RCP predicated off on every lane", "FMNMX", "FMNMX3",
                    "FSETP + FSEL (per pair of instructions)", "FFMA2, three distinct register pairs, none shared between chains",
                    "FFMA2 + FMNMX on separate chains (per pair of instructions)", "FFMA2 + 2 FMNMX (per triple)",
                    "FFMA + FMNMX (per pair)",
                    "sweep mix: 16 FFMA2 + 4 MUFU + 5 FMNMX/FMNMX3 + 2 FSETP + 2 FSEL (per group of 29; reported per 8 'instructions' = x 0.5 groups)",
                    "the same mix with 32 scalar FFMA in place of the 16 FFMA2 (x 0.5 groups)"]


def run_scene(ctx: Context, scene, device="cuda:0", tuning=None, steps=None):
    """Convenience used by tests / smoke / bench: upload a scenes.Scene, roll it out, fetch everything.
    Returns a dict of numpy arrays (final states, cost[n,5], min_clearance, collided, best index/cost)."""
    import torch
    dev = torch.device(device)
    xyzr = torch.from_numpy(scene.xyzr).to(dev)
    vel = None if scene.vel is None else torch.from_numpy(scene.vel).to(dev)
    ctx.set_obstacles(xyzr, vel, n=scene.n_spheres)
    if tuning is not None:
        ctx.set_tuning(**tuning)
    if scene.kind == GMAPP_POINT3:
        h_agents, goal = scene.agents, scene.goal
    else:
        h_agents = pose_to_state14(scene.quat, scene.pos, scene.twist)
        goal = pose_to_state14(scene.goal_quat, scene.goal, np.zeros(6))[0, :8]
    agents = torch.from_numpy(h_agents).to(dev)
    out = torch.empty_like(agents)
    n = agents.shape[0]
    S = scene.steps if steps is None else steps
    ctx.rollout(scene.kind, agents, out, goal, scene.gains, scene.dt, S)
    cost = torch.empty((n, 5), dtype=torch.float32, device=dev)
    clr = torch.empty(n, dtype=torch.float32, device=dev)
    col = torch.empty(n, dtype=torch.int32, device=dev)
    ctx.get_results(cost, clr, col)
    idx, c = ctx.best_agent(scene.alpha, scene.prev_best)
    torch.cuda.synchronize(dev)
    return dict(final=out.cpu().numpy(), cost=cost.cpu().numpy(), min_clearance=clr.cpu().numpy(),
                collided=col.cpu().numpy(), best=idx, best_cost=c, info=ctx.launch_info())
