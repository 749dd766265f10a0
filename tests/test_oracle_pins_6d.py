"""Pins for the parts of the FP64 oracle that round 1 left unpinned (run with -m "not gpu"; no CUDA involved).

P16  the 6D rollout (oracle/gmapp_oracle.c: pose6_wrench, orc_rollout_pose6) against a restatement on 4 x 4
     homogeneous matrices that uses only library routines for the group operations:
         T <- T @ expm(dt * hat(twist))              Eq. 11, PAPER.md:141 (right multiplication, body twist)
         e  = vee(logm(inv(T) @ T_g))                Eq. 8,
         wrench = (K e - D twist) + (0, R^T f_r)     Eq. 6-7, reading G18
     and the closed form of the circular-field force (P4: F = (k_f/d_O) |v|^2 cos(th) (v^ cos(th) - n^)) instead of the
     oracle's literal double cross product.  Random orientations, translation errors AND repulsive forces at the same
     time, so R vs R^T, Rt Rg vs Rg Rt, R Rd vs Rd R and p + R td vs p + td all change the result.
P17  equivariance of the 6D rollout under a rigid motion of the world (the 6D counterpart of P6): spheres, start poses
     and goal moved by (Q, t0) => positions move with it, BODY twists and every cost are unchanged.  Q and t0 are exact
     in FP32 (a signed axis permutation, dyadic offsets) so the FP32 sphere inputs of the oracle stay exact.
P18  quat_to_R: hand cases (90 degree turns about x, y, z) and scipy's Rotation.
P19  the per-state diagnostics that are the denominators / waiver masks of the GPU force parity (readings G10, G29):
     scale = |f_a| + sum_j |f_j|, gate margin, clamp margin, kappa -- hand-computed from P5-A (tests/golden/p5_single_sphere.txt).
"""
import numpy as np
import scipy.linalg
from scipy.spatial.transform import Rotation

from paper_2606_12579_b200 import scenes


def _f32(x):
    return float(np.float32(x))


def _hat6(tw):
    X = np.zeros((4, 4))
    w = tw[:3]
    X[:3, :3] = np.array([[0, -w[2], w[1]], [w[2], 0, -w[0]], [-w[1], w[0], 0]])
    X[:3, 3] = tw[3:]
    return X


def _vee6(X):
    return np.array([X[2, 1], X[0, 2], X[1, 0], X[0, 3], X[1, 3], X[2, 3]])


def _cf_sum_closed_form(p, v, xyzr, vel, t, g):
    """Sphere sum with the closed form of Eq. 2-3 (pin P4), not the cross products."""
    f = np.zeros(3)
    for j in range(xyzr.shape[0]):
        u = vel[j] if vel is not None else np.zeros(3)
        c = xyzr[j, :3] + t * u
        d = c - p
        dist = np.linalg.norm(d)
        ds = dist - (g["r_agent"] + xyzr[j, 3])
        if not ds <= g["r_influence"]:
            continue
        dO = max(ds, g["eps_dist"])
        vr = v - u
        nv = np.linalg.norm(vr)
        if nv == 0.0 or dist == 0.0:
            continue
        n, vh = d / dist, vr / nv
        cth = n @ vh
        f += (g["k_circ"] / dO) * nv * nv * cth * (vh * cth - n)
    return f


def _rollout_4x4(R0, p0, tw0, xyzr, vel, Rg, pg, gains, dt, steps):
    g = {k: (_f32(v) if k != "heuristic" else v) for k, v in gains.items()}
    dt = _f32(dt)
    xyzr = np.asarray(xyzr, np.float32).astype(np.float64)
    vel = None if vel is None else np.asarray(vel, np.float32).astype(np.float64)
    Tg = np.eye(4); Tg[:3, :3] = Rg; Tg[:3, 3] = pg
    out_p, out_R, out_tw = [], [], []
    for i in range(len(p0)):
        T = np.eye(4); T[:3, :3] = R0[i]; T[:3, 3] = p0[i]
        tw = np.array(tw0[i], float)
        for k in range(steps):
            R, p = T[:3, :3], T[:3, 3]
            f_r = _cf_sum_closed_form(p, R @ tw[3:], xyzr, vel, k * dt, g)
            e = _vee6(scipy.linalg.logm(np.linalg.inv(T) @ Tg).real)
            tau = g["k_att_rot"] * e[:3] - g["k_damp_rot"] * tw[:3]
            f = g["k_att"] * e[3:] - g["k_damp"] * tw[3:] + R.T @ f_r
            tw = tw + g["vel_factor"] * dt * np.r_[g["inv_inertia"] * tau, g["inv_mass"] * f]
            T = T @ scipy.linalg.expm(dt * _hat6(tw))
        out_p.append(T[:3, 3].copy()); out_R.append(T[:3, :3].copy()); out_tw.append(tw)
    return np.array(out_R), np.array(out_p), np.array(out_tw)


def _pose_scene(n_agents, n_spheres, moving, seed):
    """Poses with random orientations, a translation error, fast body velocities aimed through clutter."""
    sc = scenes.fast_clutter(seed=seed, n_agents=n_agents, n_spheres=n_spheres, moving=moving, steps=50)
    rng = np.random.default_rng(seed + 77)
    R0 = Rotation.random(n_agents, random_state=seed + 5).as_matrix()
    p0 = sc.agents[:, :3].astype(np.float64)
    nu = np.einsum("nji,nj->ni", R0, sc.agents[:, 3:].astype(np.float64))        # body-frame linear velocity R^T v
    om = rng.normal(0.0, 0.8, size=(n_agents, 3))
    Rg = Rotation.from_rotvec([0.4, -0.7, 0.5]).as_matrix()
    return sc, R0, p0, np.c_[om, nu], Rg


def test_P16_pose6_rollout_vs_4x4_expm_logm(orc):
    gains = dict(scenes.default_gains(), k_att=1.5, k_damp=0.3, k_att_rot=2.5, k_damp_rot=0.4, inv_mass=0.8,
                 inv_inertia=1.3)
    for n_sph, moving in ((0, False), (20, False), (20, True)):
        sc, R0, p0, tw0, Rg = _pose_scene(5, max(n_sph, 1), moving, seed=3)
        xyzr = sc.xyzr[:n_sph]
        vel = sc.vel[:n_sph] if moving else None
        pg = sc.goal.astype(np.float64)
        got = orc.rollout_pose6_mat(R0, p0, tw0, xyzr, vel, Rg, pg, gains, 1e-3, 50)
        Rw, pw, tww = _rollout_4x4(R0, p0, tw0, xyzr, vel, Rg, pg, gains, 1e-3, 50)
        assert np.allclose(got["p"], pw, rtol=0, atol=1e-10), np.abs(got["p"] - pw).max()
        assert np.allclose(got["R"], Rw, rtol=0, atol=1e-10)
        assert np.allclose(got["twist"], tww, rtol=0, atol=1e-9), np.abs(got["twist"] - tww).max()
        if n_sph:
            # the repulsion really acted (otherwise the frame of f_r would not be exercised)
            free = orc.rollout_pose6_mat(R0, p0, tw0, xyzr[:0], None, Rg, pg, gains, 1e-3, 50)
            assert np.abs(free["p"] - got["p"]).max() > 1e-4


def test_P16_detects_frame_mistakes():
    """The restatement itself distinguishes the orderings the pin is meant to catch (left vs right multiplication)."""
    sc, R0, p0, tw0, Rg = _pose_scene(2, 20, False, seed=3)
    T = np.eye(4); T[:3, :3] = R0[0]; T[:3, 3] = p0[0]
    E = scipy.linalg.expm(1e-3 * _hat6(tw0[0]))
    assert np.abs(T @ E - E @ T).max() > 1e-5


def test_P17_pose6_rigid_motion_equivariance(orc):
    gains = dict(scenes.default_gains(), k_att=1.0, k_damp=0.1, k_att_rot=2.0, k_damp_rot=0.5)
    sc, R0, p0, tw0, Rg = _pose_scene(6, 40, True, seed=4)
    # dyadic rounding keeps every moved coordinate exactly representable in FP32
    grid = 2.0 ** -12
    xyzr = np.round(sc.xyzr.astype(np.float64) / grid) * grid
    vel = np.round(sc.vel.astype(np.float64) / grid) * grid
    pg = np.round(sc.goal.astype(np.float64) / grid) * grid
    Q = np.array([[0, 0, -1.0], [1.0, 0, 0], [0, -1.0, 0]])          # proper rotation (det +1), Q != Q^T
    assert np.isclose(np.linalg.det(Q), 1.0) and np.abs(Q - Q.T).max() == 1.0
    t0 = np.array([0.25, -0.5, 0.125])
    a = orc.rollout_pose6_mat(R0, p0, tw0, xyzr, vel, Rg, pg, gains, 1e-3, 60, want_traj=True)
    xyzr_m = np.c_[xyzr[:, :3] @ Q.T + t0, xyzr[:, 3]]
    assert np.array_equal(xyzr_m.astype(np.float32).astype(np.float64), xyzr_m)
    b = orc.rollout_pose6_mat(np.einsum("ij,njk->nik", Q, R0), p0 @ Q.T + t0, tw0, xyzr_m, vel @ Q.T,
                              Q @ Rg, Q @ pg + t0, gains, 1e-3, 60, want_traj=True)
    assert np.allclose(b["p"], a["p"] @ Q.T + t0, rtol=0, atol=1e-12)
    assert np.allclose(b["R"], np.einsum("ij,njk->nik", Q, a["R"]), rtol=0, atol=1e-12)
    assert np.allclose(b["twist"], a["twist"], rtol=0, atol=1e-11)        # body twists do not see the world frame
    assert np.allclose(b["cost"], a["cost"], rtol=0, atol=1e-10)
    assert np.allclose(b["min_clearance"], a["min_clearance"], rtol=0, atol=1e-12)
    assert np.array_equal(b["collided"], a["collided"])
    # every intermediate pose as well
    assert np.allclose(b["traj"][:, :, 12:], a["traj"][:, :, 12:], rtol=0, atol=1e-11)
    assert np.abs(a["twist"][:, :3]).max() > 0.1 and np.abs(a["p"] - p0).max() > 1e-2


def test_P18_quat_to_R_hand_cases_and_scipy(orc):
    h = np.sqrt(0.5)
    Rz = [[0, -1, 0], [1, 0, 0], [0, 0, 1]]
    Rx = [[1, 0, 0], [0, 0, -1], [0, 1, 0]]
    Ry = [[0, 0, 1], [0, 1, 0], [-1, 0, 0]]
    for q, want in (((h, 0, 0, h), Rz), ((h, h, 0, 0), Rx), ((h, 0, h, 0), Ry), ((1, 0, 0, 0), np.eye(3))):
        assert np.allclose(orc.quat_to_R(q)[0], want, atol=1e-15), q
    assert np.allclose(orc.quat_to_R((0.5, 0.5, 0.5, 0.5))[0], [[0, 0, 1], [1, 0, 0], [0, 1, 0]], atol=1e-15)   # 120 deg about (1,1,1)
    rng = np.random.default_rng(9)
    q = rng.normal(0, 1, (50, 4))
    want = Rotation.from_quat(q[:, [1, 2, 3, 0]]).as_matrix()           # scipy is scalar-last and normalises
    assert np.allclose(orc.quat_to_R(q), want, atol=1e-14)
    assert np.allclose(orc.quat_to_R(3.0 * q), want, atol=1e-14)        # not unit: normalised, not scaled


def test_P19_force_diagnostics_hand_case(orc):
    # P5-A (tests/golden/p5_single_sphere.txt): p = 0, v = (1,0,0), sphere c = (0.1, 0.05, 0), r = 0.03, k_f = 1, r_d = 0.15,
    # eps = 1e-3  =>  dist = sqrt(0.0125), d_O = dist - 0.03, |f_j| = 4.88977237.  With p_g = (1,0,0), k_att = 2, k_damp = 0.5:
    # f_a = 2 (1,0,0) - 0.5 (1,0,0) = (1.5, 0, 0).
    g = scenes.default_gains()
    c = np.array([0.1, 0.05, 0.0], np.float32).astype(np.float64); r = float(np.float32(0.03))
    dist = np.linalg.norm(c); dO = dist - r
    fmag = (1.0 / dO) * (c[0] / dist) * (c[1] / dist)                  # (k_f/d_O) |v|^2 |cos th sin th|
    assert abs(fmag - 4.88977237) < 2e-6
    st = np.array([[0, 0, 0, 1.0, 0, 0]])
    xyzr = np.array([[0.1, 0.05, 0.0, 0.03]], np.float32)
    o = orc.forces_point3(st, xyzr, None, [1, 0, 0], g)
    rd, eps = _f32(0.15), _f32(1e-3)
    assert np.isclose(o["scale"][0], 1.5 + fmag, rtol=1e-12) and abs(o["scale"][0] - 6.38977237) < 2e-6
    assert np.isclose(o["margins"][0, 0], abs(dO - rd) / rd, rtol=1e-12) and abs(o["margins"][0, 0] - 0.45464) < 1e-5
    assert np.isclose(o["margins"][0, 1], abs(dO - eps) / eps, rtol=1e-12) and abs(o["margins"][0, 1] - 80.8034) < 1e-3
    assert np.isclose(o["kappa"][0], dist / dO, rtol=1e-12) and abs(o["kappa"][0] - 1.366733) < 1e-5
    assert np.isclose(o["dmin"][0], dO, rtol=1e-12)
    # two mirrored spheres: the forces cancel, the SCALE does not (sum of magnitudes, not magnitude of the sum)
    xyzr2 = np.array([[0.1, 0.05, 0.0, 0.03], [0.1, -0.05, 0.0, 0.03]], np.float32)
    o2 = orc.forces_point3(st, xyzr2, None, [1, 0, 0], g)
    assert np.allclose(o2["f_rep"][0], 0, atol=1e-12)
    assert np.isclose(o2["scale"][0], 1.5 + 2 * fmag, rtol=1e-12)
    # a sphere outside r_d adds nothing to the scale but sets the gate margin when it is the closest to the gate
    xyzr3 = np.array([[0.1, 0.05, 0.0, 0.03], [0.0, 0.0, 0.2, 0.04]], np.float32)     # ds = 0.16: 0.01 outside r_d
    o3 = orc.forces_point3(st, xyzr3, None, [1, 0, 0], g)
    ds3 = _f32(0.2) - _f32(0.04)
    assert np.isclose(o3["scale"][0], 1.5 + fmag, rtol=1e-12)
    assert np.isclose(o3["margins"][0, 0], abs(ds3 - rd) / rd, rtol=1e-9) and abs(o3["margins"][0, 0] - 0.0666667) < 1e-5
    # 6D: scale = |K e - D v| (6-norm) + sum |f_j|; identity pose at the origin, goal (1,0,0) with identity orientation:
    # e = (0, (1,0,0)), twist = (0.2,0,0 ; 1,0,0): K e - D v = (-0.1,0,0 ; 1.5,0,0)
    o6 = orc.forces_pose6(np.eye(3)[None], np.zeros((1, 3)), np.array([[0.2, 0, 0, 1.0, 0, 0]]), xyzr, None,
                          [1, 0, 0, 0], [1, 0, 0], g)
    assert np.isclose(o6["scale"][0], np.hypot(0.1, 1.5) + fmag, rtol=1e-12)
    assert np.allclose(o6["err"][0], [0, 0, 0, 1, 0, 0], atol=1e-15)


def test_P19_rollout_margins_static_agent(orc):
    # an agent at rest with no attractor never moves (the circular field vanishes at v = 0, reading G7): the rollout's
    # margins are those of its start pose, by hand from the two surface distances 0.07 (inside r_d) and 0.16 (outside)
    g = dict(scenes.default_gains(), k_att=0.0, k_damp=0.0)
    ag = np.zeros((1, 6), np.float32)
    xyzr = np.array([[0.1, 0.0, 0.0, 0.03], [0.0, 0.0, 0.2, 0.04]], np.float32)
    o = orc.rollout_point3(ag, xyzr, None, [0, 0, 0], g, 1e-3, 7)
    d0 = _f32(0.1) - _f32(0.03); d1 = _f32(0.2) - _f32(0.04); rd, eps = _f32(0.15), _f32(1e-3)
    want_gate = min(abs(d0 - rd), abs(d1 - rd)) / rd
    want_clamp = min(abs(d0 - eps), abs(d1 - eps)) / eps
    assert np.allclose(o["margins"][0], [want_gate, want_clamp, d0], rtol=1e-9)
    assert abs(want_gate - 0.0666667) < 1e-5 and abs(want_clamp - 69.0) < 1e-3
    assert np.isclose(o["min_clearance"][0], d0, rtol=1e-12) and o["collided"][0] == 0
