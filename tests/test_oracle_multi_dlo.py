"""Pins of the oracle's multi-DLO scenes: several ropes laid back
to back in one env, `cuts` marking the edges that do not exist.

What fixes the expected values (none of it is the cut code itself):
  * ropes that never touch must evolve exactly like the same ropes simulated ALONE, each in an env of its own (the
    single-rope oracle, pinned elsewhere), values and gradients, and no gradient may cross from one rope to the other;
  * two one-edge ropes crossing at right angles, pressed DEPTH into each other at their midpoints: Eq.13 in closed form
    (t = u = 1/2, equal masses: every vertex moves by DEPTH / 2 along the normal, the velocities by that over h);
  * A0: every rope gets the frame chain the single-rope A0 gives it, the absent edge has no frame, rope ends no rest curvature."""
import numpy as np

from helpers import rope_problem


def helix(n, phase, centre, pitch=0.01, rad=0.03, l=0.01):
    s = phase + np.arange(n) * l / np.hypot(rad, pitch)
    return np.asarray(centre) + np.stack([rad * np.cos(s), rad * np.sin(s), pitch * s], 1)


def two_ropes(n1, n2):
    a, b = helix(n1, 0.3, (0.0, 0.0, 0.0)), helix(n2, 1.1, (0.5, 0.2, 0.1))
    va = 0.2 * np.stack([np.sin(5 * a[:, 2]), np.cos(3 * a[:, 0]), a[:, 1]], 1)
    vb = 0.2 * np.stack([np.cos(4 * b[:, 1]), b[:, 2], np.sin(2 * b[:, 0])], 1)
    return a, b, va, vb


KW = dict(dt=1e-3, kappa_bar_from_x0=1, enable_plasticity=1, material=dict(alpha=3e-4, gamma=0.3, l0=0.01, sigma_y=2.0, r_c=0.2))


def test_separate_ropes_in_one_env_equal_the_ropes_alone(orc):
    n1, n2, H, S = 10, 12, 12, 5      # n1 even: the red / black order of Eq.10 goes by edge index, so rope 2 keeps the colours it has alone
    a, b, va, vb = two_ropes(n1, n2)
    both = rope_problem(np.concatenate([a, b]), np.concatenate([va, vb]), horizon=H, stride=S, cuts=[n1 - 1], pins=(0, n1), **KW)
    sim = orc.OracleSim(both)
    st = sim.rollout(H, S)
    rng = np.random.default_rng(5)
    seed = rng.standard_normal((1, 3, n1 + n2))
    g = sim.backward(seed, None)
    gm_sum = np.zeros(5)
    for lo, hi, x, v in ((0, n1, a, va), (n1, n1 + n2, b, vb)):
        alone = rope_problem(x, v, horizon=H, stride=S, pins=(0,), **KW)
        so = orc.OracleSim(alone)
        ref = so.rollout(H, S)
        assert np.abs(ref["x"][0] - x.T).max() > 1e-4                       # the ropes did move
        for key in ("x", "v", "kappa_bar"):
            assert np.allclose(st[key][0][:, lo:hi], ref[key][0], rtol=0, atol=1e-13), key
        assert np.allclose(st["d1"][0][:, lo:hi - 1], ref["d1"][0][:, : hi - lo - 1], rtol=0, atol=1e-13)
        gr = so.backward(seed[:, :, lo:hi], None)
        for key in ("g_x0", "g_v0"):
            assert np.allclose(g[key][0][:, lo:hi], gr[key][0], rtol=1e-10, atol=1e-12), key
        gm_sum += gr["g_material"][0]
    assert np.all(st["d1"][0][:, n1 - 1] == 0.0)                            # the absent edge carries no frame
    # no gradient crosses the cut: a loss on rope 2 alone leaves rope 1's inputs without gradient
    seed2 = seed.copy()
    seed2[:, :, :n1] = 0.0
    g2 = sim.backward(seed2, None)
    assert np.all(g2["g_x0"][0][:, :n1] == 0.0) and np.all(g2["g_v0"][0][:, :n1] == 0.0)
    assert np.abs(g2["g_x0"][0][:, n1:]).max() > 1e-3
    # and the material gradient of the env is the sum over its ropes (they share the material, the loss is a sum)
    assert np.allclose(g["g_material"][0], gm_sum, rtol=1e-9, atol=1e-12 * np.abs(gm_sum).max())


def test_rope_on_rope_contact_closed_form(orc):
    """Ropes A = (0, 1) along x and B = (2, 3) along y cross at their midpoints, DEPTH inside each other; rope C = (4, 5)
    is far from both, but the ABSENT edge (3, 4) between B's end and C's start runs straight through A's centre line."""
    R_ROPE, DEPTH, H_SUB = 2.5e-3, 2e-4, 1e-3
    z = R_ROPE - 0.5 * DEPTH                                                # centre lines 2 R - DEPTH apart
    pts = np.array([[-0.02, 0, -z], [0.02, 0, -z], [0, -0.02, z], [0, 0.02, z], [0.01, -0.0195, -3 * z], [0.01, -0.06, -3 * z]])   # (not exactly THROUGH the centre line: Eq.13 has no normal at distance 0)
    kw = dict(dt=H_SUB, horizon=1, n_substeps=1, n_proj_iters=1, stretch_mode=0, enable_self_contact=1, gravity=(0, 0, 0),
              rope_radius=R_ROPE, material=dict(stretch=0.0, alpha=0.0, mu_s=0.0, l0=0.04))
    st = orc.OracleSim(rope_problem(pts, cuts=[1, 3], **kw)).rollout(1, 0)
    want = pts.copy()
    want[:2, 2] -= 0.5 * DEPTH
    want[2:4, 2] += 0.5 * DEPTH
    assert np.allclose(st["x"][0].T, want, rtol=0, atol=1e-15)
    assert np.allclose(st["v"][0][2], np.array([-1, -1, 1, 1, 0, 0]) * 0.5 * DEPTH / H_SUB, rtol=1e-12, atol=0)
    assert np.all(st["v"][0][:2] == 0.0)
    # control: with the edge (3, 4) present it is a segment inside rope A, and Eq.13 pushes on it
    st2 = orc.OracleSim(rope_problem(pts, cuts=[1], **kw)).rollout(1, 0)
    assert np.abs(st2["x"][0].T - want).max() > 1e-4


def test_a0_frames_per_rope_and_rope_ends(orc):
    n1, n2 = 7, 6
    a, b, _, _ = two_ropes(n1, n2)
    both = rope_problem(np.concatenate([a, b]), horizon=1, cuts=[n1 - 1], **KW)
    st = orc.OracleSim(both).state()
    d1 = st["d1"][0]
    da, db = orc.frames_init(a)[0], orc.frames_init(b)[0]
    assert np.allclose(d1[:, : n1 - 1].T, da[: n1 - 1], atol=1e-15) and np.allclose(d1[:, n1: n1 + n2 - 1].T, db[: n2 - 1], atol=1e-15)
    assert np.all(d1[:, n1 - 1] == 0.0)
    kb = st["kappa_bar"][0]
    assert np.all(kb[:, [0, n1 - 1, n1, n1 + n2 - 1]] == 0.0)               # rope ends: no bending element
    ka, kbb = orc.material_curvature(a, da[: n1 - 1]), orc.material_curvature(b, db[: n2 - 1])
    assert np.allclose(kb[:, 1: n1 - 1].T, ka[1: n1 - 1], atol=1e-13) and np.allclose(kb[:, n1 + 1: n1 + n2 - 1].T, kbb[1: n2 - 1], atol=1e-13)
    assert np.abs(kb[:, 1: n1 - 1]).max() > 1e-3
