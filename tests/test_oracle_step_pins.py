"""Pins for the three parts of the oracle's substep that round 1 left unpinned ("What's weak" 1):

  A9  time-parallel transport of the frames INSIDE the step (which tangents, which direction, after the commit),
  A6  the self-contact friction law: sign, magnitude min(mu_s D_p / h, |v_t|), D_p = sum over the iterations,
  A7  finger capsule geometry p + R(+-gap/2, 0, 0..len) and the body-point velocity.

Every expected value below comes from something other than the oracle: scipy's Rotation for minimal rotations and poses,
the closed-form holonomy of parallel transport along a circle of latitude, and hand-derived closed forms of Eq.13 +
friction on strands that cross at right angles.  Each mistake named in the verdict was injected into oracle/rod_step.hpp by
hand once and seen to fail its pin here (listed in DESIGN.md section 3a)."""
import numpy as np
import pytest
from scipy.spatial.transform import Rotation as Rot

from helpers import rope_problem


def min_rotation(a, b):
    """scipy rotation taking unit vector a to unit vector b about a x b (the rotation-minimising one)"""
    w = np.cross(a, b)
    s, c = np.linalg.norm(w), np.dot(a, b)
    if s < 1e-300:
        return Rot.identity()
    return Rot.from_rotvec(w / s * np.arctan2(s, c))


def gripper_rope(N, actions, x, grasp=(0, 1), **kw):
    """one rope held at `grasp` by one gripper whose initial pose is at vertex grasp[0] with zero rotation"""
    P = rope_problem(x, horizon=len(actions), n_grippers=1, n_grasp_max=len(grasp), **kw)
    P["grasp_verts"] = np.array([[list(grasp)]], dtype=np.int32)
    pose0 = np.zeros((1, 1, 6))
    pose0[0, 0, :3] = x[grasp[0]]
    P["init_pose"] = pose0
    P["finger_geom"] = np.array([[[1.0, 0.01, 1e-3, 0.0]]])          # fingers far from the rope: no contact
    act = np.zeros((len(actions), 1, 1, 6))
    act[:, 0, 0, :3] = x[grasp[0]]
    act[:, 0, 0, 3:] = actions
    P["actions"] = act
    return P


# ---- A9 -----------------------------------------------------------------------------------------------------------
def test_frame_transport_one_large_step_matches_minimal_rotation(orc):
    """An edge carried by the gripper through 0.6 rad in ONE substep: its director must be the minimal rotation
    t_old -> t_new applied to the old director (reading R-4), with t_new the tangent AFTER the commit.  Swapping the
    arguments of the transport, or transporting with the tangents before the commit, moves d1 by O(angle^2)."""
    x = np.array([[0.0, 0, 0], [0.05, 0, 0], [0.1, 0, 0.0]])
    axis = np.array([1.0, 2.0, 3.0]) / np.sqrt(14.0)
    P = gripper_rope(3, [0.6 * axis], x, n_substeps=1, gravity=(0, 0, 0), material=dict(l0=0.05, alpha=1e-3))
    sim = orc.OracleSim(P)
    d1_0 = sim.state()["d1"][0, :, 0].copy()
    st = sim.rollout(1, 0)
    R = Rot.from_rotvec(0.6 * axis)
    t_old, t_new = np.array([1.0, 0, 0]), R.apply([1.0, 0, 0])
    assert np.allclose(st["x"][0, :, 1], R.apply(x[1]), atol=1e-14)              # the grasped vertex is where the pose puts it
    want = min_rotation(t_old, t_new).apply(d1_0)
    got = st["d1"][0, :, 0]
    assert np.allclose(got, want, atol=1e-13), (got, want)
    assert abs(np.dot(got, t_new)) < 1e-14 and abs(np.linalg.norm(got) - 1) < 1e-14
    # the rigidly co-rotated director is a DIFFERENT vector (the frame is not carried rigidly: no twist DoF, R-4 / B-24)
    assert np.linalg.norm(R.apply(d1_0) - want) > 1e-2


def test_frame_transport_holonomy_on_a_circle_of_latitude(orc):
    """Closed form.  An edge whose tangent makes the angle phi with a fixed axis is turned about that axis by theta in
    many small substeps.  Parallel transport along a circle of latitude lags the rigidly co-rotated frame by theta cos(phi)
    about the tangent (the Foucault-pendulum angle): psi = -theta cos(phi).  A transport in the wrong direction or with
    stale tangents is only first-order accurate per substep and misses this by ~1e-3."""
    phi, theta, H = np.deg2rad(60.0), 0.5 * np.pi, 200
    axis = np.array([np.cos(phi), np.sin(phi), 0.0])
    x = np.array([[0.0, 0, 0], [0.05, 0, 0], [0.1, 0, 0.0]])
    acts = [axis * theta * (t + 1) / H for t in range(H)]
    P = gripper_rope(3, acts, x, gravity=(0, 0, 0), material=dict(l0=0.05, alpha=1e-3))
    sim = orc.OracleSim(P)
    d1_0 = sim.state()["d1"][0, :, 0].copy()
    st = sim.rollout(H, 0)
    R = Rot.from_rotvec(axis * theta)
    t_T, rigid, got = R.apply([1.0, 0, 0]), R.apply(d1_0), st["d1"][0, :, 0]
    psi = np.arctan2(np.dot(np.cross(rigid, got), t_T), np.dot(rigid, got))
    assert abs(psi - (-theta * np.cos(phi))) < 2e-6, psi


def test_frame_transport_in_a_moving_rope_with_rest_curvature(orc):
    """A non-planar rope with kappa_bar = kappa(x0) swinging under gravity, one substep per frame: between consecutive
    recorded states every director is the scipy minimal rotation (old tangent -> new tangent, both from the RECORDED
    positions, i.e. after the commit) of the previous one."""
    N = 12
    s = np.linspace(0, 1.5 * np.pi, N)
    x = np.stack([0.04 * np.cos(s), 0.04 * np.sin(s), 0.015 * s], 1)
    P = rope_problem(x, dt=2e-4, horizon=60, n_substeps=1, kappa_bar_from_x0=1, pins=(0,), material=dict(alpha=2e-4, gamma=0.5))
    sim = orc.OracleSim(P)
    sim.rollout(60, 0, record=True)
    worst, moved = 0.0, 0.0
    for t in range(60):
        a, b = sim.record(t), sim.record(t + 1)
        xa, xb = a["x"][0].T, b["x"][0].T
        for j in range(N - 1):
            to = (xa[j + 1] - xa[j]) / np.linalg.norm(xa[j + 1] - xa[j])
            tn = (xb[j + 1] - xb[j]) / np.linalg.norm(xb[j + 1] - xb[j])
            want = min_rotation(to, tn).apply(a["d1"][0, :, j])
            worst = max(worst, np.linalg.norm(b["d1"][0, :, j] - want))
            moved = max(moved, np.linalg.norm(b["d1"][0, :, j] - a["d1"][0, :, j]))
    assert moved > 1e-4          # the frames did move
    assert worst < 1e-13, worst
    # and the rest curvature keeps the moving rope near its helix: the elastic curvature stays small against kappa_bar
    end = sim.record(60)
    kap = orc.material_curvature(end["x"][0].T, end["d1"][0].T[: N - 1])
    kb = end["kappa_bar"][0].T
    assert np.linalg.norm(kb[1:-1], axis=1).min() > 0.05
    assert np.linalg.norm((kap - kb)[1:-1], axis=1).max() < 0.5 * np.linalg.norm(kb[1:-1], axis=1).min()


# ---- A6 -----------------------------------------------------------------------------------------------------------
R_ROPE, DEPTH, H_SUB, MU_S = 2.5e-3, 1e-4, 1e-3, 0.3


def strands_problem(strands, vel, N_C=10):
    """free particles (no stretch, no bending, no gravity) joined into one rope; `strands` = list of (p, q) end points
    of the straight strands, connected by far-away detours; vel = velocity of each strand's two vertices"""
    pts, v = [], []
    for k, (p, q) in enumerate(strands):
        pts += [p, q]
        v += [vel[k], vel[k]]
        if k + 1 < len(strands):
            pts += [[0.3 + 0.1 * k, 0.0, 0.2 + 0.1 * k], [0.3 + 0.1 * k, -0.3, 0.2 + 0.1 * k]]
            v += [[0, 0, 0], [0, 0, 0]]
    P = rope_problem(np.array(pts, float), np.array(v, float), dt=H_SUB, horizon=1, n_substeps=1, n_proj_iters=N_C, stretch_mode=0,
                     enable_self_contact=1, gravity=(0, 0, 0), rope_radius=R_ROPE, material=dict(stretch=0.0, alpha=0.0, mu_s=MU_S))
    return P


@pytest.mark.parametrize("vA,label", [(0.5, "sliding"), (0.01, "sticking")])
def test_self_friction_two_crossing_strands(orc, vA, label):
    """Strand A (along x, moving along x with vA) under strand B (along y, at rest), DEPTH inside each other, placed so that
    the PREDICTED positions cross at both mid points (t = u = 1/2, equal masses).  Eq.13 resolves an isolated pair in its
    first iteration, so D_p = DEPTH; then (L410, R-16) the relative tangential velocity at the contact drops by exactly
    m = min(mu_s D_p / h, |v_t|), never grows, and is shared equally by the four vertices."""
    z, off = 2 * R_ROPE - DEPTH, -H_SUB * vA
    P = strands_problem([([-0.05 + off, 0, 0], [0.05 + off, 0, 0]), ([0, -0.05, z], [0, 0.05, z])], [[vA, 0, 0], [0, 0, 0]])
    st = orc.OracleSim(P).rollout(1, 0)
    v = st["v"][0].T                                    # [N][3]; A = vertices 0,1; B = vertices 4,5
    m = min(MU_S * DEPTH / H_SUB, vA)
    assert (label == "sticking") == (m == vA)
    assert np.allclose(v[[0, 1, 4, 5], 0], [vA - m / 2, vA - m / 2, m / 2, m / 2], rtol=0, atol=1e-13), v[[0, 1, 4, 5], 0]
    assert np.allclose(v[[0, 1, 4, 5], 2], np.array([-1, -1, 1, 1]) * DEPTH / (2 * H_SUB), rtol=0, atol=1e-12)
    assert np.allclose(v[:, 1], 0, atol=1e-15) and np.allclose(v[[2, 3]], 0, atol=1e-15)
    rel = 0.5 * (v[0, 0] + v[1, 0]) - 0.5 * (v[4, 0] + v[5, 0])               # relative tangential velocity at the contact
    assert abs(rel - (vA - m)) < 1e-13
    assert 0.0 <= rel < vA                                                      # friction never accelerates the sliding
    if label == "sticking":
        assert abs(rel) < 1e-15
    assert np.allclose(v.sum(axis=0), [2 * vA, 0, 0], atol=1e-13)               # momentum


def test_self_friction_depth_sum_over_iterations(orc):
    """Three strands piled A / B / C, A and C sliding in opposite directions over B (t = u = 1/2 at the predicted
    positions).  B is pushed equally from both sides, so every Jacobi iteration closes only half of each gap:
    d_k = DEPTH / 2^k, D_p = DEPTH (2 - 2^(1 - N_C)).  `D_p` of the last iteration only, of the first only, or without the
    1/h, all give another friction impulse."""
    z, vA, N_C = 2 * R_ROPE - DEPTH, 0.5, 10
    off = H_SUB * vA
    P = strands_problem([([-0.05 - off, 0, z], [0.05 - off, 0, z]), ([0, -0.05, 0], [0, 0.05, 0]), ([-0.05 + off, 0, -z], [0.05 + off, 0, -z])],
                        [[vA, 0, 0], [0, 0, 0], [-vA, 0, 0]], N_C=N_C)
    st = orc.OracleSim(P).rollout(1, 0)
    v = st["v"][0].T                                    # A = 0,1; B = 4,5; C = 8,9
    Dp = DEPTH * (2.0 - 2.0 ** (1 - N_C))
    m = min(MU_S * Dp / H_SUB, vA)
    assert m < vA and Dp > 1.9 * DEPTH
    assert np.allclose(v[[0, 1], 0], vA - m / 2, rtol=0, atol=1e-12), v[[0, 1], 0]
    assert np.allclose(v[[8, 9], 0], -vA + m / 2, rtol=0, atol=1e-12)
    assert np.allclose(v[[4, 5]], 0, atol=1e-13)                                # B: the two impulses cancel
    assert np.allclose(v[[0, 1], 2], DEPTH * (1.0 - 2.0 ** -N_C) / H_SUB, rtol=0, atol=1e-11)     # sum of A's normal corrections / h
    assert np.allclose(v[[8, 9], 2], -DEPTH * (1.0 - 2.0 ** -N_C) / H_SUB, rtol=0, atol=1e-11)


# ---- A7 fingers ------------------------------------------------------------------------------------------------------
GAP, LEN, RF, EPS = 0.03, 0.05, 0.01, 1e-3


def finger_probe(orc, probes, pose0, pose1, h=1e-3):
    """free particles (vertex 1 of a 3-vertex 'rope' without forces) at `probes`, at rest; one gripper moves pose0 -> pose1
    in one substep.  Returns the particles' velocities after the substep."""
    B = len(probes)
    x = np.zeros((B, 3, 3))
    x[:, 0], x[:, 2] = [5.0, 5.0, 5.0], [5.0, 5.0, 6.0]
    x[:, 1] = probes
    P = rope_problem(x, dt=h, horizon=1, n_substeps=1, stretch_mode=0, gravity=(0, 0, 0), n_grippers=1, n_grasp_max=1, rope_radius=R_ROPE,
                     contact_softness=EPS, material=dict(stretch=0.0, alpha=0.0, mu_r=0.0, l0=1.0))
    P["grasp_verts"] = -np.ones((B, 1, 1), dtype=np.int32)
    P["init_pose"] = np.repeat(np.asarray(pose0, float)[None, None], B, axis=0)
    P["finger_geom"] = np.repeat(np.array([[[GAP, LEN, RF, 0.0]]]), B, axis=0)
    P["actions"] = np.repeat(np.asarray(pose1, float)[None, None, None], B, axis=1)
    return orc.OracleSim(P).rollout(1, 0)["v"][:, :, 1]


def finger_expected(c, pose0, pose1, h):
    """v' = f (v_b . n) n for a particle at rest touched by an approaching finger (e = 0, mu = 0, R-17), with the
    finger capsules at p + R(+-gap/2, 0, 0..len) of the END pose and v_b the finite difference of the body point over h"""
    p0, R0 = np.asarray(pose0[:3]), Rot.from_rotvec(pose0[3:])
    p1, R1 = np.asarray(pose1[:3]), Rot.from_rotvec(pose1[3:])
    v = np.zeros(3)
    for sx in (0.5 * GAP, -0.5 * GAP):                               # finger 0, then finger 1 (sequential, like the step)
        A, Bq = p1 + R1.apply([sx, 0, 0]), p1 + R1.apply([sx, 0, LEN])
        ab = Bq - A
        s = np.clip(np.dot(c - A, ab) / np.dot(ab, ab), 0, 1)
        dv = c - (A + s * ab)
        dist = np.linalg.norm(dv)
        n = dv / dist
        f = min(np.exp((R_ROPE - (dist - RF)) / EPS), 1.0)
        if not f > 0.1:
            continue
        vb = (c - (p0 + R0.apply(R1.inv().apply(c - p1)))) / h
        u = v - vb
        if np.dot(u, n) < 0:
            v = v + f * (-np.dot(u, n)) * n
    return v


def test_finger_capsules_sit_at_the_paper_offsets_and_carry_the_body_velocity(orc):
    h = 1e-3
    rho = np.array([0.0, 0.5 * np.pi, 0.0])                           # 90 degrees about y: local z -> world x, local x -> world -z
    p = np.array([0.2, -0.1, 0.3])
    R = Rot.from_rotvec(rho)
    assert np.allclose(R.apply([0, 0, 1]), [1, 0, 0]) and np.allclose(R.apply([1, 0, 0]), [0, 0, -1])
    reach = RF + R_ROPE
    # probes in local coordinates: beside finger 0 at mid length (outside and between the fingers), off its tip cap, off its
    # base cap, beside finger 1, and one out of reach; distances chosen so that f spans (0.1, 1]
    local = np.array([[0.5 * GAP + reach + 0.5e-3, 0.0, 0.5 * LEN], [0.5 * GAP, reach - 0.2e-3, 0.3 * LEN],
                      [0.5 * GAP + 0.004, 0.003, LEN + reach + 0.001], [0.5 * GAP + 0.002, -0.001, -reach - 0.0015],
                      [-0.5 * GAP - reach - 1e-3, 0.002, 0.7 * LEN], [0.5 * GAP + reach + 0.004, 0.0, 0.5 * LEN]])
    probes = p + R.apply(local)
    # (1) pure translation towards +x_local ... every touched probe sees v_b = dp / h
    for dp_local in ([-2e-4, 1e-4, 0.5e-4], [1.5e-4, -2e-4, -1e-4], [0.5e-4, 1e-4, 2e-4]):
        dp = R.apply(dp_local)
        pose0, pose1 = np.r_[p - dp, rho], np.r_[p, rho]
        got = finger_probe(orc, probes, pose0, pose1, h)
        want = np.array([finger_expected(c, pose0, pose1, h) for c in probes])
        assert np.allclose(got, want, rtol=0, atol=1e-12), (dp_local, got, want)
        assert np.allclose(got[-1], 0)                                  # out of reach: f < 0.1, untouched
    assert np.abs(want).max() > 1e-3
    # (2) pure rotation about the gripper's own axis direction: v_b -> omega x r
    for axis_local, dth in (([0, 1, 0], 4e-3), ([0, 1, 0], -4e-3)):
        rho0 = rho * (1 - dth / (0.5 * np.pi))                          # same axis: rotation vectors add
        pose0, pose1 = np.r_[p, rho0], np.r_[p, rho]
        got = finger_probe(orc, probes, pose0, pose1, h)
        want = np.array([finger_expected(c, pose0, pose1, h) for c in probes])
        assert np.allclose(got, want, rtol=0, atol=1e-12)
        omega = np.array([0.0, 1.0, 0.0]) * dth / h
        touched = np.linalg.norm(got, axis=1) > 0
        assert touched.sum() >= 2
        for c, g in zip(probes[touched], got[touched]):                 # the response is along n with size f (omega x r) . n
            n = g / np.linalg.norm(g)
            vb_n = np.dot(np.cross(omega, c - p), n)
            # f <= 1 and v_b . n differs from (omega x r) . n by O(dth) relative
            assert np.linalg.norm(g) <= vb_n * (1 + 5 * abs(dth)) + 1e-12
    # (3) the geometry alone: read the distance to the capsule back from f = exp(d / eps) of a translating finger
    dp = R.apply([-1e-4, 0, 0])                                         # finger 0 moves towards -x_local ... probe 0 is on its +x side
    dp = -dp
    pose0, pose1 = np.r_[p - dp, rho], np.r_[p, rho]
    got = finger_probe(orc, probes[:1], pose0, pose1, h)[0]
    n = got / np.linalg.norm(got)
    assert np.allclose(n, R.apply([1, 0, 0]), atol=1e-12)               # pushed straight away from the finger axis
    f = np.linalg.norm(got) / np.dot(dp / h, n)
    d = EPS * np.log(f)
    assert abs(d - (-0.5e-3)) < 1e-12                                   # the probe was placed 0.5 mm outside the contact distance
