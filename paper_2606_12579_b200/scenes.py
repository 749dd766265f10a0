"""Seeded synthetic scenes for the G-MAPP rollout (BASELINE.json configs 1-5).

This module is the ONE piece shared by the CUDA path, the FP64 oracle, the tests and
bench.py.  It holds no arithmetic of the method (no distances-to-force, no integration,
no costs): it only draws random start states, spheres and parameters, applies the
geometric keep-out filter that makes the scenes meaningful, rounds everything to FP32
once, and returns plain numpy arrays.

The scenes STAND IN for the paper's own simulation scenes (Trap / Opening / Cluttered /
Passage; Table II scenes PAPER.md:326-339), whose geometry and
obstacle counts the paper does not give.  Shapes and distributions follow BASELINE.json
`configs` as restated in SURVEY.md section 8(d); items BASELINE.json leaves open are
fixed there and repeated in DESIGN.md ("Input recipe").

Draw order (numpy.random.default_rng(seed), PCG64, FP64 draws cast to FP32 once):
agents first (positions, then velocities / orientations / twists), then spheres
(centres, radii, velocities).  Keep-out redraws continue the same stream.
"""
from __future__ import annotations

import dataclasses
from typing import Optional

import numpy as np

# Workspace cube W of SURVEY.md 8(d): [-0.5,0.5] x [-0.5,0.5] x [0,1] m.
_W_LO = np.array([-0.5, -0.5, 0.0])
_W_HI = np.array([0.5, 0.5, 1.0])
_START_MEAN = np.array([0.3, 0.0, 0.5])
_GOAL_ARM = np.array([-0.3, 0.0, 0.5])

KIND_POINT3 = 0
KIND_MOTOR6 = 1


def default_gains() -> dict:
    """Gain defaults (values the paper leaves open are reading G23)."""
    return dict(
        k_circ=1.0, k_att=2.0, k_damp=0.5, k_att_rot=2.0, k_damp_rot=0.5,
        inv_mass=1.0, inv_inertia=1.0, vel_factor=0.5,
        r_influence=0.15, r_agent=0.0, eps_dist=1e-3,
        w_goal=1.0, w_obs=1.0, w_path=1.0, w_smooth=1.0,
        r_cost_goal=0.0, r_cost_obs=0.0, a_max=10.0, heuristic=0,
    )


@dataclasses.dataclass
class Scene:
    """One rollout problem.  All arrays are float32 and C-contiguous.

    kind == KIND_POINT3: ``agents`` is [n,6] = (p, v).
    kind == KIND_MOTOR6: ``quat`` [n,4] (w,x,y,z; unit), ``pos`` [n,3], ``twist`` [n,6]
    = (omega, nu) body frame, ``goal_quat`` [4]; ``agents`` is None (each side builds its
    own state representation from quat/pos/twist).
    """
    name: str
    kind: int
    xyzr: np.ndarray                      # [n_spheres,4]
    vel: Optional[np.ndarray]             # [n_spheres,3] or None (static)
    goal: np.ndarray                      # [3] goal position
    gains: dict
    dt: float
    steps: int
    agents: Optional[np.ndarray] = None   # POINT3
    quat: Optional[np.ndarray] = None     # MOTOR6
    pos: Optional[np.ndarray] = None
    twist: Optional[np.ndarray] = None
    goal_quat: Optional[np.ndarray] = None
    alpha: float = 0.9
    prev_best: int = -1

    @property
    def n_agents(self) -> int:
        return int((self.agents if self.kind == KIND_POINT3 else self.pos).shape[0])

    @property
    def n_spheres(self) -> int:
        return int(self.xyzr.shape[0])

    @property
    def interactions(self) -> int:
        """Force-evaluating pair interactions per cycle, N_a * N_O * S."""
        return self.n_agents * self.n_spheres * self.steps


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64).astype(np.float32))


def _keepout_ok(c: np.ndarray, r: np.ndarray, goal: np.ndarray) -> np.ndarray:
    """True where a sphere's SURFACE is >= 0.25 m from the start mean and >= 0.10 m from the goal."""
    d_start = np.linalg.norm(c - _START_MEAN, axis=-1) - r
    d_goal = np.linalg.norm(c - goal, axis=-1) - r
    return (d_start >= 0.25) & (d_goal >= 0.10)


def _draw_spheres_W(rng, n, r_lo, r_hi, keepout, goal):
    c = rng.uniform(_W_LO, _W_HI, size=(n, 3))
    r = rng.uniform(r_lo, r_hi, size=n)
    if keepout:
        bad = ~_keepout_ok(c, r, goal)
        while bad.any():
            k = int(bad.sum())
            c[bad] = rng.uniform(_W_LO, _W_HI, size=(k, 3))
            r[bad] = rng.uniform(r_lo, r_hi, size=k)
            bad = ~_keepout_ok(c, r, goal)
    return c, r


def _arm_agents(rng, n):
    p = _START_MEAN + rng.normal(0.0, 0.05, size=(n, 3))
    v = rng.normal(0.0, 0.1, size=(n, 3))
    return p, v


def config1(seed: int = 0) -> Scene:
    """Tiny 3D point-agent rollout: 16 agents x 8 spheres x 100 steps (BASELINE.json configs[0])."""
    rng = np.random.default_rng(seed)
    p = rng.uniform(-0.5, 0.5, size=(16, 3))
    v = np.zeros((16, 3))
    c = rng.uniform(-0.3, 0.3, size=(8, 3))
    r = rng.uniform(0.03, 0.08, size=8)
    g = default_gains()
    return Scene("config1_tiny", KIND_POINT3, _f32(np.c_[c, r]), None, _f32([0.4, 0.4, 0.4]),
                 g, 1e-3, 100, agents=_f32(np.c_[p, v]))


def config2(seed: int = 0, keepout: bool = True, n_agents: int = 64, n_spheres: int = 256,
            steps: int = 500) -> Scene:
    """Single-arm-scale scene: 64 agents x 256 static spheres x 500 steps (configs[1])."""
    rng = np.random.default_rng(seed)
    p, v = _arm_agents(rng, n_agents)
    c, r = _draw_spheres_W(rng, n_spheres, 0.02, 0.1, keepout, _GOAL_ARM)
    g = default_gains()
    return Scene("config2_single_arm", KIND_POINT3, _f32(np.c_[c, r]), None, _f32(_GOAL_ARM),
                 g, 1e-3, steps, agents=_f32(np.c_[p, v]))


def config3(seed: int = 0, keepout: bool = True, n_agents: int = 1024, n_blobs: int = 32,
            per_blob: int = 128, steps: int = 100) -> Scene:
    """Dense depth-derived clutter: 1024 agents x 4096 spheres (32 Gaussian blobs) x 100 steps (configs[2])."""
    rng = np.random.default_rng(seed)
    p, v = _arm_agents(rng, n_agents)
    sigma = 0.05
    centres = rng.uniform(_W_LO, _W_HI, size=(n_blobs, 3))
    if keepout:
        rr = np.full(n_blobs, 3.0 * sigma)
        bad = ~_keepout_ok(centres, rr, _GOAL_ARM)
        while bad.any():
            centres[bad] = rng.uniform(_W_LO, _W_HI, size=(int(bad.sum()), 3))
            bad = ~_keepout_ok(centres, rr, _GOAL_ARM)
    c = np.repeat(centres, per_blob, axis=0) + rng.normal(0.0, sigma, size=(n_blobs * per_blob, 3))
    r = np.full(n_blobs * per_blob, 0.02)
    g = default_gains()
    g["r_influence"] = 0.2
    return Scene("config3_dense_clutter", KIND_POINT3, _f32(np.c_[c, r]), None, _f32(_GOAL_ARM),
                 g, 1e-3, steps, agents=_f32(np.c_[p, v]))


def config4(seed: int = 0, keepout: bool = True, n_agents: int = 256, n_spheres: int = 2048,
            steps: int = 300) -> Scene:
    """6D pose agents (motor state) x 2048 moving spheres x 300 steps (configs[3])."""
    rng = np.random.default_rng(seed)
    p = _START_MEAN + rng.normal(0.0, 0.05, size=(n_agents, 3))
    q = rng.normal(0.0, 1.0, size=(n_agents, 4))
    q /= np.linalg.norm(q, axis=1, keepdims=True)
    q[q[:, 0] < 0] *= -1.0
    nu = rng.normal(0.0, 0.1, size=(n_agents, 3))
    twist = np.c_[np.zeros((n_agents, 3)), nu]
    c, r = _draw_spheres_W(rng, n_spheres, 0.02, 0.05, keepout, _GOAL_ARM)
    u = rng.uniform(-0.3, 0.3, size=(n_spheres, 3))
    g = default_gains()
    # re-normalise AFTER the float32 cast so both sides start from the same unit quaternion
    q32 = _f32(q)
    return Scene("config4_pose6_moving", KIND_MOTOR6, _f32(np.c_[c, r]), _f32(u), _f32(_GOAL_ARM),
                 g, 1e-3, steps, quat=q32, pos=_f32(p), twist=_f32(twist),
                 goal_quat=_f32([1.0, 0.0, 0.0, 0.0]))


SWEEP_AGENTS = (1024, 4096, 16384)
SWEEP_SPHERES = (4096, 16384, 65536)


def config5(n_agents: int, n_spheres: int, seed: int = 0, steps: int = 200) -> Scene:
    """Stress sweep point: uniform spheres in a 2 m cube, 3D point agents (configs[4])."""
    rng = np.random.default_rng(seed)
    p = rng.uniform(-1.0, 1.0, size=(n_agents, 3))
    v = rng.normal(0.0, 0.1, size=(n_agents, 3))
    c = rng.uniform(-1.0, 1.0, size=(n_spheres, 3))
    r = rng.uniform(0.01, 0.05, size=n_spheres)
    g = default_gains()
    return Scene(f"config5_sweep_{n_agents}x{n_spheres}", KIND_POINT3, _f32(np.c_[c, r]), None,
                 _f32([0.8, 0.8, 0.8]), g, 1e-3, steps, agents=_f32(np.c_[p, v]))


def fast_clutter(seed: int = 0, n_agents: int = 96, n_spheres: int = 333, steps: int = 100,
                 moving: bool = False, r_lo: float = 0.01, r_hi: float = 0.04) -> Scene:
    """Parity-only scene (not a benchmark config, SURVEY.md 8(c) 'Observation for the harness'):
    agents fly at ~1 m/s through clutter so the circular-field force is actually exercised.
    Sizes are deliberately ragged (not multiples of 32)."""
    rng = np.random.default_rng(seed + 1000)
    p = np.array([0.45, 0.0, 0.5]) + rng.normal(0.0, 0.08, size=(n_agents, 3))
    aim = _GOAL_ARM - p
    aim /= np.linalg.norm(aim, axis=1, keepdims=True)
    v = aim * rng.uniform(0.7, 1.3, size=(n_agents, 1)) + rng.normal(0.0, 0.15, size=(n_agents, 3))
    c = rng.uniform(_W_LO * np.array([0.6, 0.6, 1.0]) + np.array([0, 0, 0.2]),
                    _W_HI * np.array([0.6, 0.6, 1.0]) - np.array([0, 0, 0.2]), size=(n_spheres, 3))
    r = rng.uniform(r_lo, r_hi, size=n_spheres)
    u = rng.uniform(-0.3, 0.3, size=(n_spheres, 3)) if moving else None
    g = default_gains()
    g["k_att"] = 1.0
    g["k_damp"] = 0.1
    return Scene("fast_clutter" + ("_moving" if moving else ""), KIND_POINT3, _f32(np.c_[c, r]),
                 None if u is None else _f32(u), _f32(_GOAL_ARM), g, 1e-3, steps,
                 agents=_f32(np.c_[p, v]))


def grazing(seed: int = 0, n_agents: int = 40, n_extra: int = 70, steps: int = 100, moving: bool = False) -> Scene:
    """Parity-only scene: agents fly at ~1 m/s tangentially past one large sphere (R = 0.1 m) at surface distances of
    0.3 - 8 mm, i.e. through and around the band eps <= d_O < R/16 where the force is most sensitive to the distance
    (exercises the two-pass distance refinement of the packed kernels: raw -> refined -> raw again), with a ragged
    number of small far-away spheres around."""
    rng = np.random.default_rng(seed + 2000)
    R, c0 = 0.1, np.array([0.0, 0.0, 0.5])
    off = np.linspace(3e-4, 8e-3, n_agents)
    ang = rng.uniform(0.0, 2.0 * np.pi, size=n_agents)                 # where on the sphere's equator-circle the agent passes
    up = np.c_[np.zeros(n_agents), np.sin(ang), np.cos(ang)]
    p = c0 + up * (R + off)[:, None] + np.array([-0.004, 0.0, 0.0])    # 4 mm before the closest point
    v = np.array([1.0, 0.0, 0.0]) + rng.normal(0.0, 0.02, size=(n_agents, 3))
    c = rng.uniform([-0.5, -0.5, 0.0], [0.5, 0.5, 1.0], size=(4 * n_extra, 3))
    c = c[np.linalg.norm(c - c0, axis=1) > 0.32][:n_extra]
    r = rng.uniform(0.01, 0.03, size=len(c))
    xyzr = np.r_[np.c_[c0[None], [[R]]], np.c_[c, r]]
    order = rng.permutation(len(xyzr))                                 # the big sphere lands on an arbitrary lane
    u = None
    if moving:
        u = rng.uniform(-0.3, 0.3, size=(len(xyzr), 3)); u[0] = [0.02, 0.0, 0.0]
        u = u[order]
    g = default_gains()
    g["k_att"] = 1.0
    g["k_damp"] = 0.1
    return Scene("grazing" + ("_moving" if moving else ""), KIND_POINT3, _f32(xyzr[order]), None if u is None else _f32(u),
                 _f32(np.array([0.4, 0.0, 0.6])), g, 1e-3, steps, agents=_f32(np.c_[p, v]))


def by_name(name: str, **kw) -> Scene:
    table = {"config1": config1, "config2": config2, "config3": config3, "config4": config4,
             "fast_clutter": fast_clutter}
    if name.startswith("config5"):
        return config5(**kw)
    return table[name](**kw)


def depth_cloud(seed: int = 0, n_points: int = 200_000, n_objects: int = 12):
    """Synthetic fused depth cloud (stands in for the paper's two 848x480 depth cameras; its frames are
    not available): points on the camera-facing surfaces of a few objects and a table plane inside the workspace W,
    sensor noise, a share of far outliers and of NaN dropouts.  Returns (points [n,3] float32, lo [3], hi [3]).
    No arithmetic of the method: only random draws."""
    rng = np.random.default_rng(seed)
    n_obj = int(0.6 * n_points); n_tab = int(0.3 * n_points); n_out = n_points - n_obj - n_tab
    centres = rng.uniform(_W_LO + 0.15, _W_HI - 0.15, size=(n_objects, 3))
    radii = rng.uniform(0.04, 0.12, size=n_objects)
    which = rng.integers(0, n_objects, size=n_obj)
    dirs = rng.normal(size=(n_obj, 3)); dirs /= np.linalg.norm(dirs, axis=1, keepdims=True)
    dirs[:, 0] = -np.abs(dirs[:, 0])                                  # the half facing the cameras at -x
    obj = centres[which] + radii[which, None] * dirs + rng.normal(0.0, 0.002, size=(n_obj, 3))
    tab = np.c_[rng.uniform(_W_LO[0], _W_HI[0], n_tab), rng.uniform(_W_LO[1], _W_HI[1], n_tab),
                0.05 + rng.normal(0.0, 0.002, n_tab)]
    out = rng.uniform(-3.0, 3.0, size=(n_out, 3))
    pts = np.concatenate([obj, tab, out], axis=0)
    pts = pts[rng.permutation(pts.shape[0])]
    pts[rng.random(pts.shape[0]) < 0.02] = np.nan                     # depth dropouts
    return _f32(pts), _f32(_W_LO), _f32(_W_HI)
