"""Pins for the FP64 oracle (run with -m "not gpu"; no CUDA involved).

Each test checks oracle/gmapp_oracle.c against something other than itself: hand-computed values
(tests/golden/, with citations), closed forms derived from PAPER.md Eq. 2-3 and Eq. 7-11,
invariants the paper states, scipy's expm/logm, a matrix power, or an
independently written numpy restatement that uses a different algebraic form.
"""
import os

import numpy as np
import pytest
import scipy.linalg

from paper_2606_12579_b200 import scenes

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def G(**kw):
    g = scenes.default_gains()
    g.update(kw)
    return g


def _rows(name):
    out = []
    for line in open(os.path.join(GOLD, name)):
        line = line.strip()
        if line and not line.startswith("#"):
            out.append(line.split())
    return out


# ---------------------------------------------------------------------------------- P5
@pytest.mark.parametrize("row", _rows("p5_single_sphere.txt"), ids=lambda r: r[0])
def test_P5_hand_computed_single_sphere(orc, row):
    v = np.array(row[1:4], float); c = np.array(row[4:7], float); r = float(row[7])
    want = np.array(row[8:11], float)
    f, ds, gated = orc.pair_force(np.zeros(3), v, c, r, G())
    assert np.allclose(f, want, rtol=2e-9, atol=1e-9), (f, want)
    if row[0] == "D":
        assert not gated and np.all(f == 0.0)       # exactly zero outside r_d
    if row[0] == "C":
        assert gated and np.allclose(f, 0, atol=1e-15)


# ---------------------------------------------------------------------------------- P1, P2, P4, P7
def _random_pairs(n, seed=1):
    rng = np.random.default_rng(seed)
    p = rng.uniform(-0.5, 0.5, (n, 3)); v = rng.normal(0, 1, (n, 3))
    dirn = rng.normal(0, 1, (n, 3)); dirn /= np.linalg.norm(dirn, axis=1, keepdims=True)
    r = rng.uniform(0.02, 0.1, n)
    ds = rng.uniform(2e-3, 0.149, n)
    c = p + dirn * (r + ds)[:, None]
    u = rng.uniform(-0.3, 0.3, (n, 3))
    return p, v, c, r, u, ds


def test_P1_force_orthogonal_to_relative_velocity(orc):
    p, v, c, r, u, _ = _random_pairs(300)
    for i in range(300):
        f, ds, gated = orc.pair_force(p[i], v[i], c[i], r[i], G(), u=u[i])
        assert gated
        vr = v[i] - u[i]
        assert abs(f @ vr) <= 1e-12 * np.linalg.norm(f) * np.linalg.norm(vr) + 1e-300
        assert np.linalg.norm(f) > 0


def test_P2_current_orthogonal_to_surface_normal(orc):
    p, v, c, r, u, _ = _random_pairs(200, seed=2)
    for i in range(200):
        cur = orc.current_vector(p[i], v[i], c[i], u=u[i])
        n = (c[i] - p[i]) / np.linalg.norm(c[i] - p[i])
        assert abs(cur @ n) <= 1e-13 * np.linalg.norm(v[i] - u[i])


def test_P4_closed_form_magnitude_and_direction(orc):
    # |F| = k_f/(2 dO) |v|^2 |sin 2 theta|,  F = (k_f/dO)|v|^2 cos(theta) (vhat cos(theta) - n)
    p, v, c, r, _, ds = _random_pairs(300, seed=3)
    for i in range(300):
        f, ds_o, _ = orc.pair_force(p[i], v[i], c[i], r[i], G(k_circ=1.7))
        d = c[i] - p[i]; n = d / np.linalg.norm(d); nv = np.linalg.norm(v[i]); vh = v[i] / nv
        ct = n @ vh; th = np.arccos(np.clip(ct, -1, 1))
        assert np.isclose(ds_o, ds[i], rtol=1e-9, atol=1e-13)
        assert np.isclose(np.linalg.norm(f), 1.7 / (2 * ds[i]) * nv**2 * abs(np.sin(2 * th)), rtol=1e-7)
        assert np.allclose(f, 1.7 / ds[i] * nv**2 * ct * (vh * ct - n), rtol=1e-8, atol=1e-10)


def test_P4_clamp_below_eps(orc):
    # inside the eps shell and inside the sphere the denominator is eps (Alg. 1 line 6)
    g = G()
    v = np.array([0.0, 1.0, 0.0])
    for ds in (5e-4, 0.0, -0.01):
        r = 0.05
        c = np.array([np.cos(0.4), np.sin(0.4), 0.0]) * (r + ds)
        dist = np.linalg.norm(c); dsv = dist - r
        f, ds_o, gated = orc.pair_force(np.zeros(3), v, c, r, g)
        n = c / dist; ct = n @ v
        want = 1.0 / 1e-3 * ct * (v * ct - n)
        assert gated and np.isclose(ds_o, dsv) and dsv < 1e-3
        assert np.allclose(f, want, rtol=1e-9)


def test_P7_galilean(orc):
    p, v, c, r, u, _ = _random_pairs(100, seed=4)
    for i in range(100):
        f_m, _, _ = orc.pair_force(p[i], v[i], c[i], r[i], G(), u=u[i])
        f_s, _, _ = orc.pair_force(p[i], v[i] - u[i], c[i], r[i], G())
        assert np.allclose(f_m, f_s, rtol=1e-12, atol=1e-14)


def test_G5_avoidance_direction(orc):
    # approaching a sphere slightly to the +y side: the force must push towards -y (away), G5
    f, _, _ = orc.pair_force(np.zeros(3), [1, 0, 0], [0.1, 0.05, 0], 0.03, G())
    assert f[1] < 0
    # moving obstacle approaching a resting agent from +x, offset +y: relative velocity is +x
    f2, _, _ = orc.pair_force(np.zeros(3), [0, 0, 0], [0.1, 0.05, 0], 0.03, G(), u=[-1, 0, 0])
    assert np.allclose(f2, f)


def test_G7_degenerate_zero_velocity_and_centre(orc):
    f, ds, gated = orc.pair_force(np.zeros(3), np.zeros(3), [0.1, 0.0, 0], 0.03, G())
    assert gated and np.all(f == 0)
    f, ds, gated = orc.pair_force(np.zeros(3), [1, 0, 0], np.zeros(3), 0.03, G())
    assert gated and np.all(f == 0) and ds == -0.03


# ---------------------------------------------------------------------------------- P3
def test_P3_zero_outside_influence_bitwise(orc):
    sc = scenes.config1()
    far = sc.xyzr.copy()
    far[:, :3] += 10.0
    a = orc.rollout_point3(sc.agents, far, None, sc.goal, sc.gains, sc.dt, sc.steps)
    b = orc.rollout_point3(sc.agents, np.zeros((0, 4), np.float32), None, sc.goal, sc.gains, sc.dt, sc.steps)
    assert np.array_equal(a["final"], b["final"])
    assert np.array_equal(a["cost"][:, [1, 3, 4]], b["cost"][:, [1, 3, 4]])
    assert np.all(a["cost"][:, 2] == 0) and not a["collided"].any()
    assert np.all(np.isinf(b["min_clearance"]))


# ---------------------------------------------------------------------------------- P6
def _run3(orc, agents, xyzr, vel, goal, g, steps=60):
    return orc.rollout_point3(agents, xyzr, vel, goal, g, 1e-3, steps)


def test_P6_mirror_rotation_permutation(orc):
    sc = scenes.fast_clutter(n_agents=12, n_spheres=40, moving=True)
    base = _run3(orc, sc.agents, sc.xyzr, sc.vel, sc.goal, sc.gains)
    assert np.abs(base["cost"][:, 2]).max() > 0           # the field is actually exercised
    # mirror in the plane x = 0 (exact in floating point: sign flips only)
    ag = sc.agents.copy(); ag[:, [0, 3]] *= -1
    sp = sc.xyzr.copy(); sp[:, 0] *= -1
    ve = sc.vel.copy(); ve[:, 0] *= -1
    go = sc.goal.copy(); go[0] *= -1
    m = _run3(orc, ag, sp, ve, go, sc.gains)
    fm = m["final"].copy(); fm[:, [0, 3]] *= -1
    assert np.allclose(fm, base["final"], rtol=0, atol=1e-12)
    assert np.allclose(m["cost"], base["cost"], rtol=0, atol=1e-12)
    # permutation of spheres: same sum up to round-off
    perm = np.random.default_rng(0).permutation(sc.n_spheres)
    pr = _run3(orc, sc.agents, sc.xyzr[perm], sc.vel[perm], sc.goal, sc.gains)
    assert np.allclose(pr["final"], base["final"], rtol=0, atol=1e-10)
    # rotation by 90 deg about z, (x,y) -> (-y,x): exact permutation of float32 coordinates
    def rot(a, cols):
        b = a.copy(); b[:, cols[0]] = -a[:, cols[1]]; b[:, cols[1]] = a[:, cols[0]]; return b
    ag = rot(rot(sc.agents, (0, 1)), (3, 4))
    r_ = _run3(orc, ag, rot(sc.xyzr, (0, 1)), rot(sc.vel, (0, 1)),
               np.array([-sc.goal[1], sc.goal[0], sc.goal[2]], np.float32), sc.gains)
    back = r_["final"].copy()
    back[:, 0] = r_["final"][:, 1]; back[:, 1] = -r_["final"][:, 0]
    back[:, 3] = r_["final"][:, 4]; back[:, 4] = -r_["final"][:, 3]
    assert np.allclose(back, base["final"], rtol=0, atol=1e-12)
    assert np.allclose(r_["cost"], base["cost"], rtol=0, atol=1e-12)


def test_P6_superposition(orc):
    sc = scenes.fast_clutter(n_agents=6, n_spheres=120)
    st = orc.rollout_scene(sc, want_traj=True)["traj"][:, 60]      # mid-flight states, inside the clutter
    tot = orc.forces_point3(st, sc.xyzr, None, sc.goal, sc.gains)["f_rep"]
    acc = np.zeros_like(tot)
    for j in range(sc.n_spheres):
        acc += orc.forces_point3(st, sc.xyzr[j:j + 1], None, sc.goal, sc.gains)["f_rep"]
    assert np.abs(tot).max() > 0
    assert np.allclose(acc, tot, rtol=1e-12, atol=1e-12)


# ---------------------------------------------------------------------------------- P1 (rollout)
def test_P1_speed_drift_scales_with_dt(orc):
    # With attraction and damping off the CF force does no work; the explicit update of
    # Eq. 10-11 gains |v|^2 by (vel_factor dt |a|)^2 per step, so the drift over a FIXED time is O(dt).
    g = G(k_att=0.0, k_damp=0.0)
    ag = np.array([[0, 0, 0, 1.0, 0, 0]], np.float32)
    sp = np.array([[0.12, 0.06, 0.0, 0.03], [0.2, -0.07, 0.02, 0.03]], np.float32)
    drift = []
    for dt, steps in ((1e-3, 128), (5e-4, 256), (2.5e-4, 512)):
        out = orc.rollout_point3(ag, sp, None, np.zeros(3, np.float32), g, dt, steps)
        drift.append(np.linalg.norm(out["final"][0, 3:]) - 1.0)
    assert 0 < drift[2] < drift[1] < drift[0] < 1e-2
    assert 1.7 < drift[0] / drift[1] < 2.3 and 1.7 < drift[1] / drift[2] < 2.3
    # and the direction really turned (the force acted)
    assert abs(out["final"][0, 4]) > 1e-3


# ---------------------------------------------------------------------------------- P8
def test_P8_no_obstacle_closed_form_matrix_power(orc):
    k, D, dt, S = 2.0, 0.5, 1e-3, 400
    ag = np.array([[0.1, -0.2, 0.7, 0.05, 0.0, -0.3]], np.float32)
    goal = np.array([0.4, 0.4, 0.0], np.float32)
    out = orc.rollout_point3(ag, np.zeros((0, 4), np.float32), None, goal, G(k_att=k, k_damp=D), dt, S)
    dtf = float(np.float32(dt))
    M = np.array([[1 - 0.5 * dtf * dtf * k, dtf * (1 - 0.5 * dtf * D)],
                  [-0.5 * dtf * k, 1 - 0.5 * dtf * D]])
    Mp = np.linalg.matrix_power(M, S)
    for a in range(3):
        e0 = float(ag[0, a]) - float(goal[a]); v0 = float(ag[0, 3 + a])
        e, v = Mp @ np.array([e0, v0])
        assert np.isclose(out["final"][0, a] - float(goal[a]), e, rtol=1e-10, atol=1e-13)
        assert np.isclose(out["final"][0, 3 + a], v, rtol=1e-10, atol=1e-13)
    assert np.all(np.abs(np.linalg.eigvals(M)) < 1.0)          # converges to the goal


def test_P8_long_horizon_goal_convergence(orc):
    ag = np.array([[0.4 - 0.7, 0.4, 0.4, 0, 0, 0]], np.float32)
    goal = np.array([0.4, 0.4, 0.4], np.float32)
    out = orc.rollout_point3(ag, np.zeros((0, 4), np.float32), None, goal, G(), 1e-3, 60000)
    assert np.linalg.norm(out["final"][0, :3] - goal) < 1e-3
    assert np.linalg.norm(out["final"][0, 3:]) < 1e-3


# ---------------------------------------------------------------------------------- P9
def test_P9_three_step_golden(orc):
    ag = np.array([[0, 0, 0, 1, 0, 0]], np.float32)
    sp = np.array([[0.1, 0.05, 0.0, 0.03]], np.float32)
    goal = np.array([1, 0, 0], np.float32)
    for row in _rows("p9_three_steps.txt"):
        steps = int(row[0]); want = np.array(row[1:7], float)
        out = orc.rollout_point3(ag, sp, None, goal, G(), 1e-3, steps)
        # inputs are FP32-rounded (0.1f, 0.05f, 0.03f, 1e-3f): allow that rounding, ~1e-7 relative
        assert np.allclose(out["final"][0], want, rtol=3e-7, atol=1e-12), (steps, out["final"][0], want)


# ---------------------------------------------------------------------------------- P10
def _twist_mat(phi, rho):
    X = np.zeros((4, 4))
    X[:3, :3] = np.array([[0, -phi[2], phi[1]], [phi[2], 0, -phi[0]], [-phi[1], phi[0], 0]])
    X[:3, 3] = rho
    return X


def test_P10_se3_exp_log_vs_scipy(orc):
    rng = np.random.default_rng(5)
    for scale in (1e-9, 1e-5, 1e-3, 9e-3, 1.1e-2, 0.3, 1.0, 2.5, 3.1):
        for _ in range(8):
            phi = rng.normal(0, 1, 3); phi *= scale / np.linalg.norm(phi)
            rho = rng.normal(0, 1, 3)
            R, t = orc.se3_exp(phi, rho)
            E = scipy.linalg.expm(_twist_mat(phi, rho))
            assert np.allclose(R, E[:3, :3], rtol=0, atol=2e-14)
            assert np.allclose(t, E[:3, 3], rtol=0, atol=2e-14)
            assert np.allclose(R @ R.T, np.eye(3), atol=1e-14)
            phi2, rho2 = orc.se3_log(R, t)
            assert np.allclose(phi2, phi, rtol=0, atol=5e-13 + 1e-9 * (scale > 3))
            assert np.allclose(rho2, rho, rtol=0, atol=5e-12 + 1e-8 * (scale > 3))
            if 1e-3 <= scale <= 2.5:
                Lm = scipy.linalg.logm(E).real
                assert np.allclose(phi2, [Lm[2, 1], Lm[0, 2], Lm[1, 0]], atol=1e-10)
                assert np.allclose(rho2, Lm[:3, 3], atol=1e-10)


def test_P10_se3_log_golden_and_pi(orc):
    want = np.array(_rows("p10_se3_log.txt")[0], float)
    Rz = np.array([[0, -1, 0], [1, 0, 0], [0, 0, 1.0]])
    phi, rho = orc.se3_log(Rz, [1, 0, 0])
    assert np.allclose(np.r_[phi, rho], want, atol=1e-15)
    # rotation by exactly pi and just below pi about a random axis
    rng = np.random.default_rng(6)
    for th in (np.pi, np.pi - 1e-7, np.pi - 1e-4):
        n = rng.normal(0, 1, 3); n /= np.linalg.norm(n)
        R, t = orc.se3_exp(th * n, [0.3, -0.2, 0.5])
        phi, rho = orc.se3_log(R, t)
        R2, t2 = orc.se3_exp(phi, rho)
        assert np.isclose(np.linalg.norm(phi), th, atol=1e-7)
        assert np.allclose(R2, R, atol=1e-9) and np.allclose(t2, t, atol=1e-8)


def test_P10_pose6_reduces_to_point3(orc):
    # R = I, omega = 0, goal orientation I: the 6D rollout is the 3D rollout (moving spheres included)
    sc = scenes.fast_clutter(n_agents=7, n_spheres=30, moving=True, steps=80)
    n = sc.n_agents
    quat = np.tile(np.array([1, 0, 0, 0], np.float32), (n, 1))
    twist = np.c_[np.zeros((n, 3), np.float32), sc.agents[:, 3:]]
    a = orc.rollout_point3(sc.agents, sc.xyzr, sc.vel, sc.goal, sc.gains, sc.dt, sc.steps)
    b = orc.rollout_pose6(quat, sc.agents[:, :3], twist, sc.xyzr, sc.vel, [1, 0, 0, 0], sc.goal,
                          sc.gains, sc.dt, sc.steps)
    assert np.allclose(b["p"], a["final"][:, :3], rtol=0, atol=1e-13)
    assert np.allclose(b["twist"][:, 3:], a["final"][:, 3:], rtol=0, atol=1e-12)
    assert np.allclose(b["twist"][:, :3], 0, atol=1e-15)
    assert np.allclose(b["R"], np.eye(3), atol=1e-15)
    assert np.allclose(b["cost"], a["cost"], rtol=0, atol=1e-9)
    assert np.array_equal(b["collided"], a["collided"])


def test_P10_pose6_pure_rotation_attractor(orc):
    # no spheres, agent at the goal position, rotated by theta about z: the error is pure rotation,
    # omega obeys the scalar recurrence of P8 with (k_att_rot, k_damp_rot); position stays put.
    th = 0.8
    quat = np.array([[np.cos(th / 2), 0, 0, np.sin(th / 2)]], np.float32)
    pos = np.array([[0.1, 0.2, 0.3]], np.float32)
    out = orc.rollout_pose6(quat, pos, np.zeros((1, 6), np.float32), np.zeros((0, 4), np.float32), None,
                            [1, 0, 0, 0], pos[0], G(k_att_rot=3.0, k_damp_rot=0.7), 1e-3, 250)
    q64 = quat[0].astype(np.float64); th0 = 2 * np.arctan2(q64[3], q64[0])
    dt = float(np.float32(1e-3)); k = float(np.float32(3.0)); D = float(np.float32(0.7))
    M = np.array([[1 - 0.5 * dt * dt * k, dt * (1 - 0.5 * dt * D)], [-0.5 * dt * k, 1 - 0.5 * dt * D]])
    # x = rotation angle about z: x' = x + dt w', w' = w + (dt/2)(-k x - D w)  (Eq. 7-11 on a pure rotation)
    x, w = np.linalg.matrix_power(M, 250) @ np.array([th0, 0.0])
    ang = np.arctan2(out["R"][0][1, 0], out["R"][0][0, 0])
    assert np.isclose(ang, x, atol=1e-12) and 0 < x < th0
    assert np.isclose(out["twist"][0, 2], w, atol=1e-12) and w < 0
    assert np.allclose(out["twist"][0, [0, 1, 3, 4, 5]], 0, atol=1e-15)
    assert np.allclose(out["p"][0], pos[0].astype(np.float64), atol=1e-15)


# ---------------------------------------------------------------------------------- P11
def test_P11_cost_closed_forms_straight_line(orc):
    # constant velocity straight at the goal, no forces: J = 0, L = S dt |v|, Eq. 17-20 by hand
    g = G(k_att=0.0, k_damp=0.0)
    v = np.array([0.3, 0.0, 0.4])                     # |v| = 0.5
    ag = np.array([[0, 0, 0, *v]], np.float32)
    goal = np.array([0.6, 0.0, 0.8], np.float32)      # d1 = 1.0
    S, dt = 200, 1e-3
    out = orc.rollout_point3(ag, np.zeros((0, 4), np.float32), None, goal, g, dt, S)
    dtf = float(np.float32(dt)); vf = ag[0, 3:].astype(np.float64); gf = goal.astype(np.float64)
    L = S * dtf * np.linalg.norm(vf); d1 = np.linalg.norm(gf)
    C, Cg, Co, Cp, Cs = out["cost"][0]
    assert np.isclose(Cp, 1 - L / d1, rtol=1e-12)     # L < d1 branch of Eq. 19
    assert Cs < 1e-20 and Co == 0.0 and Cg == 1.0     # farther than r_d the whole way (Eq. 17 saturates)
    assert np.isclose(C, Cg + Co + Cp + Cs)
    # overshoot branch: start close, L > d1
    goal2 = (vf * 0.02).astype(np.float32)            # d1 = 0.01 < L = 0.1
    out2 = orc.rollout_point3(ag, np.zeros((0, 4), np.float32), None, goal2, g, dt, S)
    d1b = np.linalg.norm(goal2.astype(np.float64))
    assert np.isclose(out2["cost"][0, 3], 1 - d1b / L, rtol=1e-12)
    # C_goal inside r_cost_goal: mean over the S+1 poses of min(d, r)/r, by numpy
    ks = np.arange(S + 1)
    dists = np.linalg.norm(gf[None] * 0 + goal2.astype(np.float64)[None] - ks[:, None] * dtf * vf[None], axis=1)
    assert np.isclose(out2["cost"][0, 1], np.mean(np.minimum(dists, 0.15 * 1.0) / float(np.float32(0.15))), rtol=1e-9)


def test_P11_cost_obstacle_and_weights_static_agent(orc):
    # agent at rest, no gains: it never moves; C_obs = 1 - ds/r_d with ds by hand; weights multiply
    g = G(k_att=0.0, k_damp=0.0, w_goal=0.5, w_obs=2.0, w_path=3.0, w_smooth=4.0)
    ag = np.array([[0, 0, 0, 0, 0, 0]], np.float32)
    sp = np.array([[0.1, 0.0, 0.0, 0.04], [0.5, 0.5, 0.5, 0.01]], np.float32)
    out = orc.rollout_point3(ag, sp, None, np.array([0.05, 0, 0], np.float32), g, 1e-3, 10)
    ds = float(np.float32(0.1)) - float(np.float32(0.04)); rd = float(np.float32(0.15))
    Cg = float(np.float32(0.05)) / rd
    assert np.isclose(out["cost"][0, 2], 1 - ds / rd, rtol=1e-12)
    assert np.isclose(out["cost"][0, 1], Cg, rtol=1e-12)
    assert np.isclose(out["cost"][0, 3], 1.0) and out["cost"][0, 4] == 0          # L = 0 < d1 -> 1 - 0
    assert np.isclose(out["cost"][0, 0], 0.5 * Cg + 2.0 * (1 - ds / rd) + 3.0 * 1.0)
    assert np.isclose(out["min_clearance"][0], ds) and out["collided"][0] == 0
    # inside a sphere: collided, clearance negative, C_obs clamps to 1
    sp2 = np.array([[0.01, 0.0, 0.0, 0.04]], np.float32)
    out2 = orc.rollout_point3(ag, sp2, None, np.zeros(3, np.float32), g, 1e-3, 5)
    assert out2["collided"][0] == 1 and out2["min_clearance"][0] < 0 and out2["cost"][0, 2] == 1.0
    # L = d1 = 0 -> C_path = 0 (G22)
    assert out2["cost"][0, 3] == 0.0


def test_P11_jerk_normalisation(orc):
    # constant acceleration (k_att=0, k_damp=0 is force-free; use a far goal so f_a ~ const):
    # with constant a the third difference vanishes; with linearly growing a it is vf dt^3 jdot.
    g = G(k_att=1.0, k_damp=0.0, a_max=0.05)
    ag = np.array([[0, 0, 0, 0, 0, 0]], np.float32)
    goal = np.array([1000.0, 0, 0], np.float32)       # a ~ 1000 - x, x stays ~ 1e-2: nearly constant
    S, dt = 100, float(np.float32(1e-3))
    out = orc.rollout_point3(ag, np.zeros((0, 4), np.float32), None, goal, g, 1e-3, S)
    # closed form: a_k = k (g - x_k); third difference = vf dt^2 (a_k - a_{k-1}) = -vf dt^2 k dt v_{k-1}
    x, v, J, a_prev, k = 0.0, 0.0, 0.0, None, 0
    for k in range(1, S + 1):
        a = 1.0 * (1000.0 - x)
        if k >= 3:
            J += (0.5 * dt * dt * (a - a_prev)) ** 2
        v += 0.5 * dt * a; x += dt * v; a_prev = a
    want = min(1.0, J / ((S + 1) * dt**4 * float(np.float32(0.05)) ** 2))
    assert 0 < want < 1
    # the oracle differences positions ~0.5e-2 in FP64: relative accuracy of J ~ 1e-16*x/|t3| ~ 1e-6
    assert np.isclose(out["cost"][0, 4], want, rtol=1e-4)


# ---------------------------------------------------------------------------------- P12
def test_P12_agent_independence(orc):
    sc = scenes.fast_clutter(n_agents=20, n_spheres=60)
    full = orc.rollout_scene(sc)
    idx = [17, 3, 9]
    sub = orc.rollout_point3(sc.agents[idx], sc.xyzr, sc.vel, sc.goal, sc.gains, sc.dt, sc.steps)
    assert np.array_equal(sub["final"], full["final"][idx])
    assert np.array_equal(sub["cost"], full["cost"][idx])
    par = orc.rollout_scene(sc, threads=4)
    assert np.array_equal(par["final"], full["final"]) and np.array_equal(par["cost"], full["cost"])


# ---------------------------------------------------------------------------------- P13
def _numpy_rollout_point3(sc):
    """Independent restatement: vectorised over agents and spheres, BAC-CAB closed form of Eq. 2-3
    (F = (k/dO)(s/|d|^2)[(s/|v|) v - |v| d]) instead of the oracle's literal cross products, path
    length from velocities and jerk from acceleration differences instead of position differences."""
    g = {k: (float(np.float32(v)) if k != "heuristic" else v) for k, v in sc.gains.items()}
    dt = float(np.float32(sc.dt)); S = sc.steps
    p = sc.agents[:, :3].astype(np.float64); v = sc.agents[:, 3:].astype(np.float64)
    c0 = sc.xyzr[:, :3].astype(np.float64); r = sc.xyzr[:, 3].astype(np.float64)
    u = np.zeros_like(c0) if sc.vel is None else sc.vel.astype(np.float64)
    pg = sc.goal.astype(np.float64)
    n = p.shape[0]
    rd, eps = g["r_influence"], g["eps_dist"]
    sumG = np.zeros(n); sumO = np.zeros(n); L = np.zeros(n); J = np.zeros(n)
    minclr = np.full(n, np.inf); coll = np.zeros(n, bool)
    d1 = np.linalg.norm(pg - p, axis=1); a_prev = None

    def pose_terms(p, k):
        c = c0 + (k * dt) * u
        d = c[None] - p[:, None]
        dist = np.linalg.norm(d, axis=2)
        ds = dist - (g["r_agent"] + r)[None]
        return d, dist, ds

    for k in range(S + 1):
        d, dist, ds = pose_terms(p, k)
        dmin = ds.min(axis=1) if ds.shape[1] else np.full(n, np.inf)
        sumG += np.minimum(np.linalg.norm(pg - p, axis=1), rd) / rd
        sumO += 1 - np.clip(dmin, 0, rd) / rd
        minclr = np.minimum(minclr, dmin); coll |= dmin < 0
        if k == S:
            break
        vr = v[:, None] - u[None]
        nv = np.linalg.norm(vr, axis=2)
        s = (d * vr).sum(axis=2)
        dO = np.maximum(ds, eps)
        with np.errstate(divide="ignore", invalid="ignore"):
            w = np.where((ds <= rd) & (nv > 0) & (dist > 0), s / (dO * dist**2), 0.0)
            F = w[..., None] * (np.where(nv > 0, s / nv, 0.0)[..., None] * vr - nv[..., None] * d)
        f = g["k_circ"] * F.sum(axis=1) + g["k_att"] * (pg - p) - g["k_damp"] * v
        a = g["inv_mass"] * f
        v = v + g["vel_factor"] * dt * a
        L += dt * np.linalg.norm(v, axis=1)
        if k >= 2:
            J += ((g["vel_factor"] * dt * dt * (a - a_prev)) ** 2).sum(axis=1)
        a_prev = a
        p = p + dt * v
    Nk = S + 1
    Cp = np.where(L >= d1, 1 - d1 / np.where(L > 0, L, 1), 1 - L / np.where(d1 > 0, d1, 1))
    Cs = np.minimum(1, J / (Nk * dt**4 * g["a_max"] ** 2))
    cost = np.c_[sumG / Nk + sumO / Nk + Cp + Cs, sumG / Nk, sumO / Nk, Cp, Cs]
    return p, v, cost, minclr, coll


@pytest.mark.parametrize("make", [scenes.config1,
                                  lambda: scenes.fast_clutter(n_agents=24, n_spheres=77),
                                  lambda: scenes.fast_clutter(n_agents=16, n_spheres=50, moving=True)],
                         ids=["config1", "fast", "fast_moving"])
def test_P13_numpy_restatement(orc, make):
    sc = make()
    o = orc.rollout_scene(sc)
    p, v, cost, minclr, coll = _numpy_rollout_point3(sc)
    assert np.allclose(o["final"][:, :3], p, rtol=0, atol=1e-11)
    assert np.allclose(o["final"][:, 3:], v, rtol=0, atol=1e-10)
    assert np.allclose(o["cost"][:, :4], cost[:, :4], rtol=0, atol=1e-9)
    # Eq. 20 from positions (oracle) vs from accelerations (here): FP64 cancellation ~1e-6 relative
    assert np.allclose(o["cost"][:, 4], cost[:, 4], rtol=2e-4, atol=1e-12)
    assert np.allclose(o["min_clearance"], minclr, rtol=0, atol=1e-12)
    assert np.array_equal(o["collided"].astype(bool), coll)


# ---------------------------------------------------------------------------------- selection
def test_best_agent_key_and_hysteresis(orc):
    cost = np.zeros((5, 5)); cost[:, 0] = [0.5, 0.3, 0.3, 0.1, 0.4]
    coll = np.array([0, 0, 0, 1, 0], np.int32)
    assert orc.best_agent(cost, coll, 0.9, -1) == (1, 0.3)             # collided agent 3 loses; tie -> lowest index
    assert orc.best_agent(cost, coll, 0.9, 4)[0] == 1                  # 0.3 < 0.9*0.4
    assert orc.best_agent(cost, coll, 0.9, 2)[0] == 2                  # 0.3 !< 0.9*0.3: incumbent stays
    assert orc.best_agent(cost, coll, 0.7, 4)[0] == 4                  # 0.3 !< 0.7*0.4 = 0.28
    assert orc.best_agent(cost, coll, 0.9, 3)[0] == 1                  # incumbent collided: any free agent wins
    allc = np.ones(5, np.int32)
    assert orc.best_agent(cost, allc, 0.9, -1)[0] == 3                 # all collided: plain cost order
    cost[1, 0] = np.nan
    assert orc.best_agent(cost, coll, 0.9, -1)[0] == 2                 # NaN ranks last
    assert orc.best_agent(np.zeros((0, 5)), np.zeros(0, np.int32), 0.9, -1)[0] == -1


# ---------------------------------------------------------------------------------- scenes
def test_scenes_are_seeded_and_shaped():
    a, b = scenes.config3(), scenes.config3()
    assert np.array_equal(a.agents, b.agents) and np.array_equal(a.xyzr, b.xyzr)
    assert a.agents.shape == (1024, 6) and a.xyzr.shape == (4096, 4) and a.steps == 100
    assert a.agents.dtype == np.float32 and a.interactions == 1024 * 4096 * 100
    assert not np.array_equal(scenes.config3(seed=1).xyzr, a.xyzr)
    c2 = scenes.config2()
    d = np.linalg.norm(c2.xyzr[:, :3] - np.array([0.3, 0, 0.5]), axis=1) - c2.xyzr[:, 3]
    assert d.min() >= 0.25 - 1e-6 and c2.agents.shape == (64, 6) and c2.steps == 500
    c4 = scenes.config4()
    assert c4.quat.shape == (256, 4) and c4.vel.shape == (2048, 3) and c4.steps == 300
    assert np.allclose(np.linalg.norm(c4.quat.astype(np.float64), axis=1), 1, atol=1e-6)
    c1 = scenes.config1()
    assert c1.agents.shape == (16, 6) and c1.xyzr.shape == (8, 4) and np.all(c1.agents[:, 3:] == 0)
    c5 = scenes.config5(1024, 4096)
    assert c5.agents.shape == (1024, 6) and c5.steps == 200


# ---------------------------------------------------------------------------------- P14: APF (Eq. 1, reading N1)
def _p14_rows():
    rows = []
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "p14_apf_single_sphere.txt")):
        if line.strip() and not line.startswith("#"):
            t = line.split()
            rows.append((t[0], [float(x) for x in t[1:4]], float(t[4]), [float(x) for x in t[5:8]]))
    return rows


@pytest.mark.parametrize("row", _p14_rows(), ids=lambda r: r[0])
def test_P14_apf_hand_computed_single_sphere(orc, row):
    name, c, r, want = row
    g = dict(scenes.default_gains(), heuristic=1)
    for v in ([1.0, 0.0, 0.0], [0.0, 0.0, 0.0], [-0.3, 0.4, 2.0]):        # Eq. 1 has no velocity in it
        f, ds, gated = orc.pair_force([0, 0, 0], v, c, r, g)
        assert np.allclose(f, want, rtol=2e-9, atol=1e-9), (name, f, want)
    assert gated == (name != "C")


def test_P14_apf_is_minus_gradient_of_khatib_potential(orc):
    """Textbook check: F = -grad U with U = (k_f/2)(1/dO - 1/r_d)^2 inside r_d (central differences in FP64)."""
    g = dict(scenes.default_gains(), heuristic=1, k_circ=0.7)
    rng = np.random.default_rng(5)
    c, r = np.array([0.05, -0.02, 0.1]), 0.04
    def U(p):
        ds = np.linalg.norm(c - p) - r
        return 0.0 if ds > g["r_influence"] else 0.5 * g["k_circ"] * (1.0 / max(ds, g["eps_dist"]) - 1.0 / g["r_influence"]) ** 2
    n_in = 0
    for _ in range(50):
        p = c + rng.normal(size=3) * 0.08
        ds = np.linalg.norm(c - p) - r
        if not (2e-3 < ds < g["r_influence"] - 1e-3):
            continue
        n_in += 1
        h = 1e-7
        grad = np.array([(U(p + h * e) - U(p - h * e)) / (2 * h) for e in np.eye(3)])
        f, _, gated = orc.pair_force(p, [0.2, 0.1, 0.0], c, r, g)
        assert gated and np.allclose(f, -grad, rtol=1e-5, atol=1e-6)
        assert np.dot(f, c - p) < 0                                   # repulsion: away from the obstacle
    assert n_in >= 10


def test_P14_apf_rollout_superposition_and_mirror(orc):
    """APF forces superpose over spheres and mirror with the scene (same O(3) argument as P6)."""
    sc = scenes.fast_clutter(n_agents=6, n_spheres=40, steps=20)
    g = dict(sc.gains, heuristic=1)
    st = sc.agents.astype(np.float64)
    tot = orc.forces_point3(st, sc.xyzr, None, sc.goal, g)["f_rep"]
    acc = np.zeros_like(tot)
    for j in range(sc.n_spheres):
        acc += orc.forces_point3(st, sc.xyzr[j:j + 1], None, sc.goal, g)["f_rep"]
    assert np.allclose(tot, acc, rtol=1e-12, atol=1e-12)
    M = np.diag([1.0, -1.0, 1.0])
    stm = np.concatenate([st[:, :3] @ M, st[:, 3:] @ M], axis=1)
    xm = sc.xyzr.astype(np.float64).copy(); xm[:, :3] = xm[:, :3] @ M
    totm = orc.forces_point3(stm, xm.astype(np.float32), None, (sc.goal @ M).astype(np.float32), g)["f_rep"]
    assert np.allclose(totm, tot @ M, rtol=1e-12, atol=1e-12)


# ---------------------------------------------------------------------------------- P15: sphere-world builder (N3)
def test_P15_voxel_oracle_brute_force_and_invariants():
    from oracle import voxel
    rng = np.random.default_rng(3)
    lo, hi, pitch = np.float32([-0.5, -0.5, 0.0]), np.float32([0.5, 0.5, 1.0]), np.float32(0.04)
    pts = rng.uniform(-0.7, 1.2, size=(400, 3)).astype(np.float32)
    pts[::37] = np.nan
    xyzr, dims, lin = voxel.sphere_world_from_points(pts, lo, hi, pitch)
    # float32(0.04) is a hair below 0.04, so 1 m holds 25 full voxels and a sliver of a 26th
    assert list(dims) == [26, 26, 26]
    D = 26
    # brute force with a Python set, one point at a time
    want = set()
    for p in pts:
        if np.any(np.isnan(p)) or not (np.all(p >= lo) and np.all(p < hi)):
            continue
        i = [int(np.floor(np.float32(np.float32(p[a] - lo[a]) / pitch))) for a in range(3)]
        if all(i[a] < dims[a] for a in range(3)):
            want.add((i[2] * D + i[1]) * D + i[0])
    assert sorted(want) == lin.tolist() and 0 < len(want) <= 400
    assert np.all(np.diff(lin) > 0) and np.all(xyzr[:, 3] == np.float32(0.02))
    # every kept point lies in the cube of half-width pitch/2 (+ rounding) around one emitted centre
    inside = ~np.isnan(pts).any(axis=1) & np.all((pts >= lo) & (pts < hi), axis=1)
    d = np.abs(pts[inside][:, None, :].astype(np.float64) - xyzr[None, :, :3].astype(np.float64)).max(axis=2).min(axis=1)
    assert d.max() <= 0.02 + 1e-6
    # hand case: one point in the first voxel, one in the last
    x2, _, l2 = voxel.sphere_world_from_points(np.float32([[-0.49, -0.49, 0.01], [0.49, 0.49, 0.99]]), lo, hi, pitch)
    assert l2.tolist() == [0, (24 * D + 24) * D + 24]
    assert np.allclose(x2[0], [-0.48, -0.48, 0.02, 0.02], atol=1e-7) and np.allclose(x2[1], [0.48, 0.48, 0.98, 0.02], atol=1e-6)
    # idempotence: voxelising the emitted centres gives the same spheres
    x3, _, l3 = voxel.sphere_world_from_points(xyzr[:, :3], lo, hi, pitch)
    assert np.array_equal(l3, lin) and np.array_equal(x3, xyzr)


def test_depth_cloud_is_seeded_and_shaped():
    a, lo, hi = scenes.depth_cloud(seed=1, n_points=5000)
    b, _, _ = scenes.depth_cloud(seed=1, n_points=5000)
    assert a.shape == (5000, 3) and a.dtype == np.float32 and np.array_equal(a, b, equal_nan=True)
    assert 0 < np.isnan(a).any(axis=1).sum() < 500


def test_grazing_scene_is_seeded_and_skims_the_band(orc):
    """The parity-only `grazing` scene: start surface distances to the 0.1 m sphere span 0.3-8 mm (below, inside and
    above R/16 = 6.25 mm), nothing else within the influence radius of the start cloud, and the oracle keeps every
    agent out of collision while the closest ones stay under 1 mm."""
    a, b = scenes.grazing(), scenes.grazing()
    assert np.array_equal(a.agents, b.agents) and np.array_equal(a.xyzr, b.xyzr) and a.vel is None
    big = int(np.argmax(a.xyzr[:, 3]))
    assert a.xyzr[big, 3] == np.float32(0.1) and (a.xyzr[:, 3] > 0.05).sum() == 1
    d0 = np.linalg.norm(a.agents[:, :3].astype(np.float64) - a.xyzr[big, :3], axis=1) - 0.1
    assert 2e-4 < d0.min() < 5e-4 and 7e-3 < d0.max() < 9e-3
    others = np.delete(np.arange(a.n_spheres), big)
    dd = np.linalg.norm(a.agents[:, None, :3].astype(np.float64) - a.xyzr[None, others, :3], axis=2) - a.xyzr[None, others, 3]
    assert dd.min() > a.gains["r_influence"]
    o = orc.rollout_scene(a)
    assert not o["collided"].any() and o["min_clearance"].min() < 1e-3 and o["min_clearance"].max() > 6.25e-3
    m = scenes.grazing(moving=True)
    assert m.vel is not None and m.vel.shape == (m.n_spheres, 3) and np.array_equal(m.xyzr, a.xyzr)
