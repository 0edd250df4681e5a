"""Pins of the oracle's reverse pass (tape AD + checkpoint replay): closed form, central finite
differences of the oracle's own forward rollout on tiny ropes, stride independence (C-14)."""
import copy

import numpy as np
import pytest

from helpers import rope_problem
from workloads import make_problem


def loss_seeds(rng, B, N):
    return rng.normal(size=(B, 3, N)), rng.normal(size=(B, 3, N)) * 1e-2


def forward_loss(orc, P, cx, cv, frozen=None):
    st = orc.OracleSim(P, frozen_init=frozen).rollout(stride=0)
    return float((cx * st["x"]).sum() + (cv * st["v"]).sum())


def perturbed(P, key, delta, eps):
    Q = copy.deepcopy(P)
    if key.startswith("mat:"):
        Q["material"][key[4:]] = Q["material"][key[4:]] + eps * delta
    else:
        Q[key] = Q[key] + eps * delta
    return Q


GRAD_OF = {"x0": "g_x0", "v0": "g_v0", "actions": "g_actions", "kappa_bar0": "g_kappa_bar0"}
MAT_COL = {"stretch": 0, "bend_stiffness": 1, "damping": 2, "yield_curv": 3, "creep_rate": 4}


def check_fd(orc, P, keys, rtol=2e-6, seed=0, scale=None):
    rng = np.random.default_rng(seed)
    B, N = P["config"]["batch"], P["config"]["n_verts"]
    cx, cv = loss_seeds(rng, B, N)
    sim = orc.OracleSim(P)
    frozen = sim.init_products()          # the reverse pass treats the A0 products as independent inputs
    sim.rollout(stride=max(1, P["horizon"] // 3))
    g = sim.backward(cx, cv)
    for key in keys:
        if key.startswith("mat:"):
            base = P["material"][key[4:]]
            delta = rng.uniform(0.5, 1.0, base.shape) * np.maximum(np.abs(base), 1e-12)
            analytic = float((g["g_material"][:, MAT_COL[key[4:]]] * delta).sum())
            eps = 3e-4
        else:
            delta = rng.normal(size=P[key].shape)
            analytic = float((g[GRAD_OF[key]] * delta).sum())
            eps = (scale or {}).get(key, 1e-7)
        fd = (forward_loss(orc, perturbed(P, key, delta, eps), cx, cv, frozen)
              - forward_loss(orc, perturbed(P, key, delta, -eps), cx, cv, frozen)) / (2 * eps)
        assert abs(fd - analytic) <= rtol * max(abs(fd), abs(analytic)) + 1e-12, (key, fd, analytic)
    return g


def wiggly(rng, n, l, amp=0.3):
    x = np.zeros((n, 3))
    d = np.array([1.0, 0, 0])
    for i in range(1, n):
        d = d + amp * rng.normal(size=3)
        d /= np.linalg.norm(d)
        x[i] = x[i - 1] + l * d
    return x


# --- closed form: ballistic ------------------------------------------------------------------------------
def test_ballistic_closed_form(orc):
    rng = np.random.default_rng(1)
    N, H, dt = 5, 12, 1e-3
    P = rope_problem(wiggly(rng, N, 0.1), rng.normal(size=(N, 3)), dt=dt, horizon=H, stretch_mode=0, stride=5,
                     material=dict(stretch=0.0, alpha=0.0))
    cx, cv = loss_seeds(rng, 1, N)
    sim = orc.OracleSim(P)
    sim.rollout()
    g = sim.backward(cx, cv)
    assert np.abs(g["g_x0"] - cx).max() < 1e-13                       # dx_T/dx_0 = I
    assert np.abs(g["g_v0"] - (H * dt * cx + cv)).max() < 1e-13        # dx_T/dv_0 = T I, dv_T/dv_0 = I
    assert np.all(g["g_material"][:, 3:] == 0.0)                       # no plasticity: yield / creep do not enter


# --- C-13: every feature, every input class ---------------------------------------------------------------------
def test_fd_bending_projection_pinned(orc):
    rng = np.random.default_rng(2)
    N = 7
    x = wiggly(rng, N, 0.05, 0.2)
    P = rope_problem(x, 0.1 * rng.normal(size=(N, 3)), horizon=12, pins=[0], material=dict(l0=0.05, alpha=2e-3))
    P["kappa_bar0"] = 0.05 * rng.normal(size=(1, 2, N))
    check_fd(orc, P, ["x0", "v0", "kappa_bar0", "mat:bend_stiffness"])


def test_fd_compliance_damping(orc):
    rng = np.random.default_rng(3)
    N = 6
    P = rope_problem(wiggly(rng, N, 0.05, 0.2) * 1.03, 0.1 * rng.normal(size=(N, 3)), horizon=10,
                     material=dict(l0=0.05, alpha=1e-3, stretch=3e-6, gamma=0.8))
    check_fd(orc, P, ["x0", "v0", "mat:stretch", "mat:damping", "mat:bend_stiffness"])


def test_fd_stretch_energy_mode(orc):
    rng = np.random.default_rng(4)
    N = 6
    P = rope_problem(wiggly(rng, N, 0.05, 0.2) * 1.02, 0.1 * rng.normal(size=(N, 3)), horizon=10, stretch_mode=0,
                     material=dict(l0=0.05, alpha=1e-3, stretch=40.0, gamma=0.3))
    check_fd(orc, P, ["x0", "v0", "mat:stretch", "mat:damping"])


def gripper_plastic_problem(H=10, B=2):
    P = make_problem(3, batch=B, n_verts=8, horizon=H, stride=4)
    rng = np.random.default_rng(5)
    P["actions"] = P["init_pose"][None] + np.cumsum(rng.normal(0, 1, (H, B, 1, 6)) * np.array([2e-3] * 3 + [2e-2] * 3), axis=0)
    P["material"]["yield_curv"][:] = 0.05                         # low yield: plastic flow is active
    P["material"]["creep_rate"][:] = (0.3, 0.7)[:B]
    return P


def test_fd_gripper_actions_plasticity(orc):
    P = gripper_plastic_problem()
    g = check_fd(orc, P, ["actions", "x0", "v0", "mat:yield_curv", "mat:creep_rate", "mat:bend_stiffness"], rtol=5e-6)
    assert np.abs(g["g_material"][:, 3]).min() > 0               # the yield branch really was active
    assert np.abs(g["g_actions"][..., 3:]).max() > 0             # rotations matter (two grasped vertices)


def test_fd_ring_posts_self_contact(orc):
    P = make_problem(4, batch=2, n_verts=24, horizon=10, stride=5)
    rng = np.random.default_rng(6)
    # pull hard so that strands cross within the short horizon
    P["actions"] = np.repeat(P["init_pose"][None], 10, axis=0)
    P["actions"][:, :, 0, 1] -= np.linspace(0.007, 0.07, 10)[:, None]
    P["v0"] = 0.05 * rng.normal(size=P["v0"].shape)
    Q = copy.deepcopy(P)
    Q["config"]["enable_self_contact"] = 0
    assert np.abs(orc.OracleSim(Q).rollout(stride=0)["x"] - orc.OracleSim(P).rollout(stride=0)["x"]).max() > 1e-4
    # the band rests on the posts (u_n = 0 is exactly the branch point of the coupling) and exp(d/eps_s) has a
    # curvature of 1/eps_s^2 = 1e6: central differences only converge for tiny steps and to ~1e-4, hence the tolerance.
    g = check_fd(orc, P, ["x0", "v0", "actions"], rtol=1e-3, scale={"x0": 1e-10, "v0": 1e-8, "actions": 1e-10})
    assert np.isfinite(g["g_x0"]).all()


def test_fd_self_contact_hairpin_with_friction(orc):
    from test_oracle_dynamics import hairpin
    x = hairpin(6, 0.01, 0.012)
    N = len(x)
    v = np.zeros((N, 3))
    v[:6, 1], v[-6:, 1] = -0.8, 0.8
    v[:6, 0], v[-6:, 0] = 0.3, -0.3
    v[:, 2] = 0.03 * np.cos(np.arange(N))
    P = rope_problem(x, v, horizon=8, gravity=(0, 0, 0), enable_self_contact=1,
                     material=dict(l0=0.01, alpha=1e-4, stretch=1e-6, mu_s=0.3))
    sim = orc.OracleSim(P)
    st0 = sim.rollout(stride=0)
    Q = copy.deepcopy(P)
    Q["config"]["enable_self_contact"] = 0
    assert np.abs(orc.OracleSim(Q).rollout(stride=0)["x"] - st0["x"]).max() > 1e-4      # contact really engaged
    check_fd(orc, P, ["x0", "v0"], rtol=2e-5, scale={"x0": 1e-8, "v0": 1e-7})


def test_fd_rigid_primitives(orc):
    rng = np.random.default_rng(7)
    N = 8
    x = wiggly(rng, N, 0.03, 0.25) + [0, 0, 0.004]
    v = 0.3 * rng.normal(size=(N, 3)) + [0.3, 0, -0.5]
    P = rope_problem(x, v, horizon=8, n_primitives=4, restitution=0.2, material=dict(l0=0.03, alpha=5e-4, mu_r=0.4, gamma=0.2))
    P["prim_types"] = np.array([0, 3, 2, 1], dtype=np.int32)
    pp = np.zeros((1, 4, 10))
    pp[0, 0, :4] = [0, 0, 1, 0]
    pp[0, 1, :9] = [0.06, 0.0, 0.0, 0.02, 0.03, 0.012, 0.1, -0.2, 0.4]       # box under part of the rope
    pp[0, 2, :8] = [0.13, 0.01, 0.0, 0, 0, 1, 0.02, 0.012]                   # short cylinder
    pp[0, 3, :7] = [0.0, -0.05, 0.006, 0.2, 0.05, 0.006, 0.006]              # capsule lying across
    P["prim_params"] = pp
    sim = orc.OracleSim(P)
    st = sim.rollout(stride=0)
    Q = copy.deepcopy(P)
    Q["config"]["n_primitives"] = 0
    assert np.abs(orc.OracleSim(Q).rollout(stride=0)["x"] - st["x"]).max() > 1e-4       # contact really engaged
    check_fd(orc, P, ["x0", "v0", "mat:damping"], rtol=2e-5, scale={"x0": 1e-8, "v0": 1e-7})


def test_fd_finger_contact_actions(orc):
    """rope vertices swept by a moving finger capsule: the action gradient flows through the SDF and v_b"""
    N = 8
    x = np.zeros((N, 3))
    x[:, 0] = np.arange(N) * 0.02
    P = rope_problem(x, horizon=8, gravity=(0, 0, 0), n_grippers=1, n_grasp_max=1, material=dict(l0=0.02, alpha=1e-3, mu_r=0.3))
    P["grasp_verts"] = np.array([[[-1]]], dtype=np.int32)                  # nothing grasped: fingers only push
    P["init_pose"] = np.array([[[0.07, -0.02, -0.02, 0.0, 0.0, 0.0]]])
    P["finger_geom"] = np.array([[[0.03, 0.04, 0.01, 0.0]]])
    act = np.repeat(P["init_pose"][None], 8, axis=0)
    act[:, 0, 0, 1] += np.linspace(0.002, 0.016, 8)
    act[:, 0, 0, 5] += np.linspace(0.01, 0.08, 8)
    P["actions"] = act
    sim = orc.OracleSim(P)
    st = sim.rollout(stride=0)
    assert np.abs(st["x"][0, 1]).max() > 1e-3                              # the fingers pushed the rope
    g = check_fd(orc, P, ["actions", "x0"], rtol=2e-5, scale={"x0": 1e-8, "actions": 1e-8})
    assert np.abs(g["g_actions"]).max() > 0


# --- C-14: checkpointing does not change the gradient ---------------------------------------------------------------
def test_gradient_independent_of_checkpoint_stride(orc):
    P = gripper_plastic_problem(H=12)
    rng = np.random.default_rng(8)
    cx, cv = loss_seeds(rng, 2, 8)
    ref = None
    for stride in (1, 5, 12, 100):
        sim = orc.OracleSim(P)
        sim.rollout(stride=stride)
        g = sim.backward(cx, cv)
        if ref is None:
            ref = g
        for k in g:
            assert np.array_equal(g[k], ref[k]), (stride, k)             # bitwise ("replay reproduces the forward")


def test_backward_requires_checkpoints(orc):
    P = gripper_plastic_problem(H=4)
    sim = orc.OracleSim(P)
    sim.rollout(stride=0)
    with pytest.raises(RuntimeError):
        sim.backward(np.zeros((2, 3, 8)), None)
