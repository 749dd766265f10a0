"""ctypes wrapper around oracle/gmapp_oracle.c (the FP64 CPU oracle).

TEST INFRASTRUCTURE, NOT THE PRODUCT.  Importable only from tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs.  It imports nothing from the CUDA package except
nothing at all: scenes are passed in as plain numpy arrays / dicts.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "gmapp_oracle.c")
_SO = os.path.join(_HERE, "libgmapp_oracle.so")

_GAIN_FIELDS = ["k_circ", "k_att", "k_damp", "k_att_rot", "k_damp_rot", "inv_mass", "inv_inertia",
                "vel_factor", "r_influence", "r_agent", "eps_dist", "w_goal", "w_obs", "w_path",
                "w_smooth", "r_cost_goal", "r_cost_obs", "a_max"]


class OrcGains(C.Structure):
    _fields_ = [(k, C.c_double) for k in _GAIN_FIELDS] + [("heuristic", C.c_int)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (seconds).  Building the checker is not using it."""
    if force or not os.path.exists(_SO) or os.path.getmtime(_SO) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-std=c99", "-fopenmp", "-fPIC", "-shared", "-Wall", "-Wextra",
               "-fno-fast-math", "-ffp-contract=off", "-o", _SO, _SRC, "-lm"]
        subprocess.check_call(cmd)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_best_agent.restype = C.c_int
        _lib.orc_pair_force.restype = C.c_int
        _lib.orc_max_threads.restype = C.c_int
    return _lib


def gains_struct(g: dict) -> OrcGains:
    """Gains are first rounded to FP32 (what the GPU receives), then promoted to double."""
    s = OrcGains()
    for k in _GAIN_FIELDS:
        setattr(s, k, float(np.float32(g[k])))
    s.heuristic = int(g.get("heuristic", 0))
    return s


def _dp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_double))


def _fp(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_float))


def _ip(a):
    return None if a is None else a.ctypes.data_as(C.POINTER(C.c_int))


def _f32c(a):
    return None if a is None else np.ascontiguousarray(a, dtype=np.float32)


def _f64c(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def max_threads() -> int:
    return int(lib().orc_max_threads())


def pair_force(p, v, c, r, gains: dict, u=None):
    """Single agent-sphere pair (Eq. 2-3).  Inputs taken as double, NOT rounded."""
    g = OrcGains()
    for k in _GAIN_FIELDS:
        setattr(g, k, float(gains[k]))
    g.heuristic = int(gains.get("heuristic", 0))
    p, v, c = _f64c(p), _f64c(v), _f64c(c)
    uu = None if u is None else _f64c(u)
    f = np.zeros(3)
    ds = C.c_double()
    gated = lib().orc_pair_force(_dp(p), _dp(v), _dp(c), C.c_double(float(r)), _dp(uu), C.byref(g),
                                 _dp(f), C.byref(ds))
    return f, ds.value, bool(gated)


def current_vector(p, v, c, u=None):
    p, v, c = _f64c(p), _f64c(v), _f64c(c)
    uu = None if u is None else _f64c(u)
    cur = np.zeros(3)
    lib().orc_current_vector(_dp(p), _dp(v), _dp(c), _dp(uu), _dp(cur))
    return cur


def se3_exp(phi, rho):
    R, t = np.zeros(9), np.zeros(3)
    lib().orc_se3_exp(_dp(_f64c(phi)), _dp(_f64c(rho)), _dp(R), _dp(t))
    return R.reshape(3, 3), t


def se3_log(R, t):
    phi, rho = np.zeros(3), np.zeros(3)
    lib().orc_se3_log(_dp(_f64c(R).reshape(-1)), _dp(_f64c(t)), _dp(phi), _dp(rho))
    return phi, rho


def rollout_point3(agents, xyzr, vel, goal, gains: dict, dt: float, steps: int, threads: int = 1,
                   want_traj: bool = False):
    agents, xyzr, vel, goal = _f32c(agents), _f32c(xyzr), _f32c(vel), _f32c(goal)
    n, m = agents.shape[0], xyzr.shape[0]
    out = dict(final=np.zeros((n, 6)), cost=np.zeros((n, 5)), min_clearance=np.zeros(n),
               collided=np.zeros(n, dtype=np.int32), margins=np.zeros((n, 3)))
    traj = np.zeros((n, steps + 1, 6)) if want_traj else None
    g = gains_struct(gains)
    lib().orc_rollout_point3(C.c_int(n), _fp(agents), C.c_int(m), _fp(xyzr), _fp(vel), _fp(goal),
                             C.byref(g), C.c_double(float(np.float32(dt))), C.c_int(steps), C.c_int(threads),
                             _dp(out["final"]), _dp(out["cost"]), _dp(out["min_clearance"]),
                             _ip(out["collided"]), _dp(out["margins"]), _dp(traj))
    if want_traj:
        out["traj"] = traj
    return out


def forces_point3(states, xyzr, vel, goal, gains: dict, t_obstacles: float = 0.0):
    states = _f64c(states)
    xyzr, vel, goal = _f32c(xyzr), _f32c(vel), _f32c(goal)
    n, m = states.shape[0], xyzr.shape[0]
    out = dict(f_rep=np.zeros((n, 3)), f_total=np.zeros((n, 3)), scale=np.zeros(n),
               margins=np.zeros((n, 2)), kappa=np.zeros(n), dmin=np.zeros(n))
    g = gains_struct(gains)
    lib().orc_forces_point3(C.c_int(n), _dp(states), C.c_int(m), _fp(xyzr), _fp(vel),
                            C.c_double(float(t_obstacles)), _fp(goal), C.byref(g),
                            _dp(out["f_rep"]), _dp(out["f_total"]), _dp(out["scale"]),
                            _dp(out["margins"]), _dp(out["kappa"]), _dp(out["dmin"]))
    return out


def quat_to_R(q):
    """Unit quaternion (w,x,y,z) -> rotation matrix; the oracle's own conversion (textbook formula)."""
    q = _f64c(q).reshape(-1, 4)
    q = q / np.linalg.norm(q, axis=1, keepdims=True)
    w, x, y, z = q[:, 0], q[:, 1], q[:, 2], q[:, 3]
    R = np.empty((q.shape[0], 3, 3))
    R[:, 0, 0] = 1 - 2 * (y * y + z * z); R[:, 0, 1] = 2 * (x * y - w * z); R[:, 0, 2] = 2 * (x * z + w * y)
    R[:, 1, 0] = 2 * (x * y + w * z); R[:, 1, 1] = 1 - 2 * (x * x + z * z); R[:, 1, 2] = 2 * (y * z - w * x)
    R[:, 2, 0] = 2 * (x * z - w * y); R[:, 2, 1] = 2 * (y * z + w * x); R[:, 2, 2] = 1 - 2 * (x * x + y * y)
    return R


def rollout_pose6(quat, pos, twist, xyzr, vel, goal_quat, goal_pos, gains: dict, dt: float, steps: int,
                  threads: int = 1, want_traj: bool = False):
    """6D rollout.  quat/pos/twist are the FP32 scene arrays; the oracle converts them to (R, p)."""
    R0 = np.ascontiguousarray(quat_to_R(_f32c(quat))).reshape(-1, 9)
    p0 = _f64c(_f32c(pos))
    tw0 = _f64c(_f32c(twist))
    Rg = np.ascontiguousarray(quat_to_R(_f32c(goal_quat))).reshape(9)
    pg = _f64c(_f32c(goal_pos))
    xyzr, vel = _f32c(xyzr), _f32c(vel)
    n, m = p0.shape[0], xyzr.shape[0]
    out = dict(R=np.zeros((n, 9)), p=np.zeros((n, 3)), twist=np.zeros((n, 6)), cost=np.zeros((n, 5)),
               min_clearance=np.zeros(n), collided=np.zeros(n, dtype=np.int32), margins=np.zeros((n, 3)))
    traj = np.zeros((n, steps + 1, 18)) if want_traj else None
    g = gains_struct(gains)
    lib().orc_rollout_pose6(C.c_int(n), _dp(R0), _dp(p0), _dp(tw0), C.c_int(m), _fp(xyzr), _fp(vel),
                            _dp(Rg), _dp(pg), C.byref(g), C.c_double(float(np.float32(dt))), C.c_int(steps),
                            C.c_int(threads), _dp(out["R"]), _dp(out["p"]), _dp(out["twist"]),
                            _dp(out["cost"]), _dp(out["min_clearance"]), _ip(out["collided"]),
                            _dp(out["margins"]), _dp(traj))
    out["R"] = out["R"].reshape(n, 3, 3)
    if want_traj:
        out["traj"] = traj
    return out


def rollout_pose6_mat(R0, p0, twist0, xyzr, vel, goal_R, goal_p, gains: dict, dt: float, steps: int,
                      want_traj: bool = False):
    """6D rollout from rotation MATRICES given in double (no quaternion conversion, no FP32 rounding of the
    poses): the same C routine as rollout_pose6, for the pins that need exactly rotated / translated inputs."""
    R0 = _f64c(R0).reshape(-1, 9)
    p0, tw0 = _f64c(p0), _f64c(twist0)
    Rg, pg = _f64c(goal_R).reshape(9), _f64c(goal_p)
    xyzr, vel = _f32c(xyzr), _f32c(vel)
    n, m = p0.shape[0], xyzr.shape[0]
    out = dict(R=np.zeros((n, 9)), p=np.zeros((n, 3)), twist=np.zeros((n, 6)), cost=np.zeros((n, 5)),
               min_clearance=np.zeros(n), collided=np.zeros(n, dtype=np.int32), margins=np.zeros((n, 3)))
    traj = np.zeros((n, steps + 1, 18)) if want_traj else None
    g = gains_struct(gains)
    lib().orc_rollout_pose6(C.c_int(n), _dp(R0), _dp(p0), _dp(tw0), C.c_int(m), _fp(xyzr), _fp(vel),
                            _dp(Rg), _dp(pg), C.byref(g), C.c_double(float(np.float32(dt))), C.c_int(steps),
                            C.c_int(1), _dp(out["R"]), _dp(out["p"]), _dp(out["twist"]),
                            _dp(out["cost"]), _dp(out["min_clearance"]), _ip(out["collided"]),
                            _dp(out["margins"]), _dp(traj))
    out["R"] = out["R"].reshape(n, 3, 3)
    if want_traj:
        out["traj"] = traj
    return out


def forces_pose6(R, p, twist, xyzr, vel, goal_quat, goal_pos, gains: dict, t_obstacles: float = 0.0):
    R = _f64c(R).reshape(-1, 9)
    p, twist = _f64c(p), _f64c(twist)
    Rg = np.ascontiguousarray(quat_to_R(_f32c(goal_quat))).reshape(9)
    pg = _f64c(_f32c(goal_pos))
    xyzr, vel = _f32c(xyzr), _f32c(vel)
    n, m = p.shape[0], xyzr.shape[0]
    out = dict(f_rep=np.zeros((n, 3)), wrench=np.zeros((n, 6)), scale=np.zeros(n),
               margins=np.zeros((n, 2)), err=np.zeros((n, 6)))
    g = gains_struct(gains)
    lib().orc_forces_pose6(C.c_int(n), _dp(R), _dp(p), _dp(twist), C.c_int(m), _fp(xyzr), _fp(vel),
                           C.c_double(float(t_obstacles)), _dp(Rg), _dp(pg), C.byref(g),
                           _dp(out["f_rep"]), _dp(out["wrench"]), _dp(out["scale"]), _dp(out["margins"]),
                           _dp(out["err"]))
    return out


def best_agent(cost, collided, alpha: float = 0.9, prev_best: int = -1):
    cost = _f64c(cost)
    collided = np.ascontiguousarray(collided, dtype=np.int32)
    oc = C.c_double()
    idx = lib().orc_best_agent(C.c_int(cost.shape[0]), _dp(cost), _ip(collided),
                               C.c_double(float(np.float32(alpha))), C.c_int(prev_best), C.byref(oc))
    return int(idx), oc.value


def rollout_scene(scene, threads: int = 1, want_traj: bool = False, agent_slice=None):
    """Run the oracle on a scenes.Scene (duck-typed: only attributes are read)."""
    sl = slice(None) if agent_slice is None else agent_slice
    if scene.kind == 0:
        return rollout_point3(scene.agents[sl], scene.xyzr, scene.vel, scene.goal, scene.gains,
                              scene.dt, scene.steps, threads, want_traj)
    return rollout_pose6(scene.quat[sl], scene.pos[sl], scene.twist[sl], scene.xyzr, scene.vel,
                         scene.goal_quat, scene.goal, scene.gains, scene.dt, scene.steps, threads, want_traj)
