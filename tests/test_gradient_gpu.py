"""-m gpu: reverse pass of the CUDA path (dlo_backward through the C-ABI) against the oracle's tape-AD gradient on the
same seeded inputs.  Tolerance: ||g_gpu - g_orc|| / ||g_orc|| <= 1e-3 per env and gradient tensor (BASELINE.json).
Horizons are kept short enough that the fp64 tape-AD oracle finishes in seconds; strides that do not divide the
horizon exercise the ragged last segment."""
import numpy as np
import pytest

from parity import GRAD_TOL, gradient_error, loss_and_seed, make_problem, perturbed, summarize

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def both_gradients(dlo, orc, P, H, stride):
    o = orc.OracleSim(P)
    ref_state = o.rollout(H, stride)
    _, seed = loss_and_seed(P, ref_state["x"])
    ref = o.backward(seed)
    o.close()
    sim = dlo.DloSim(P)
    sim.rollout(H, stride)
    got = sim.backward(seed)
    assert sim.n_bad() == 0
    sim.close()
    return got, ref


def check(name, got, ref, keys, tol=GRAD_TOL):
    worst = 0.0
    for k in keys:
        g, r = got[k], ref[k]
        if k == "g_actions":
            g, r = np.moveaxis(g, 1, 0), np.moveaxis(r, 1, 0)       # env axis first
        err = gradient_error(g, r)
        print(summarize("%s %s" % (name, k), err))
        worst = max(worst, err.max())
    assert worst <= tol, (name, worst)


def env_first(k, a):
    return np.moveaxis(a, 1, 0) if k == "g_actions" else a


def apply_over(P, over):
    for k, v in (over or {}).items():
        if k in P["material"]:
            P["material"][k][:] = v
        else:
            P["config"][k] = v


# Smooth cases: no branch of the step sits on its threshold, the gradient is well defined, and every env must meet
# the 1e-3 bar.  (Plasticity with a small creep rate and few steps keeps every hinge well away from its yield surface.)
ALL4 = ("g_actions", "g_x0", "g_v0", "g_material")
STRICT = [
    ("cfg1 full (g_v0)", dict(cfg_id=1), 200, 50, ("g_v0", "g_x0"), None),
    ("cfg1 ragged stride", dict(cfg_id=1, n_verts=20), 23, 7, ("g_v0", "g_x0", "g_material"), None),
    ("cfg4 ring+self-contact", dict(cfg_id=4, batch=2, n_verts=48), 30, 10, ALL4, None),
    ("cfg4 odd ring", dict(cfg_id=4, batch=2, n_verts=45), 20, 20, ("g_actions", "g_x0", "g_v0"), None),
    ("cfg4 N=96 full width", dict(cfg_id=4, batch=2), 10, 4, ALL4, None),
    ("cfg5 features, elastic", dict(cfg_id=5, batch=2), 3, 2, ALL4, dict(enable_plasticity=0)),
    ("cfg3 slow creep", dict(cfg_id=3, batch=4, n_verts=24), 6, 3, ALL4, dict(creep_rate=0.1)),
    ("cfg5 N=70 slow creep", dict(cfg_id=5, batch=2, n_verts=70), 4, 4, ("g_actions", "g_material"), dict(creep_rate=0.1)),
]


@pytest.mark.parametrize("name,kw,H,stride,keys,over", STRICT, ids=[c[0] for c in STRICT])
def test_gradient_parity(dlo, orc, name, kw, H, stride, keys, over):
    P = make_problem(horizon=H, stride=stride, **kw)
    apply_over(P, over)
    got, ref = both_gradients(dlo, orc, P, H, stride)
    check(name, got, ref, keys)


def test_self_contact_crossing_gradient(dlo, orc):
    """one real Eq.13 contact with friction (figure eight), well conditioned: forward and every gradient at the plain bars"""
    from helpers import figure_eight_problem
    from parity import POS_TOL, position_error
    for H in (16, 30):
        P = figure_eight_problem(horizon=H, stride=7)
        free = dict(P, config=dict(P["config"], enable_self_contact=0))
        a, b = orc.OracleSim(P).rollout(H, 0)["x"], orc.OracleSim(free).rollout(H, 0)["x"]
        assert np.abs(a - b).max() > 1e-4, "the contact must actually engage"
        got, ref = both_gradients(dlo, orc, P, H, 7)
        check("figure eight H=%d" % H, got, ref, ("g_x0", "g_v0", "g_material"))
        sim = dlo.DloSim(P)
        x = sim.rollout(H, 0).state()["x"]
        sim.close()
        assert position_error(P, x, a).max() <= POS_TOL


def test_stretch_energy_mode_gradient(dlo, orc):
    P = make_problem(1, n_verts=16, horizon=30, stride=10)
    P["config"]["stretch_mode"] = 0
    P["material"]["stretch"][:] = 2.0e2
    got, ref = both_gradients(dlo, orc, P, 30, 10)
    check("stretch energy", got, ref, ("g_v0", "g_x0", "g_material"))


def test_gradient_independent_of_stride(dlo):
    """memory/recompute trade-off must not change the result"""
    P = make_problem(3, batch=4, n_verts=24, horizon=30)
    outs = []
    for stride in (30, 10, 7):
        sim = dlo.DloSim(P)
        x = sim.rollout(30, stride).state()["x"]
        _, seed = loss_and_seed(P, x)
        outs.append(sim.backward(seed))
        sim.close()
    for o in outs[1:]:
        for k in ("g_actions", "g_x0", "g_v0", "g_material"):
            # identical trajectory, different grouping of the fp32 sums (per-segment accumulation, shared-memory atomics
            # for the gripper poses): agreement to rounding level, relative to the largest entry
            assert np.abs(o[k] - outs[0][k]).max() <= 5e-5 * np.abs(outs[0][k]).max(), k


@pytest.mark.parametrize("cfg, H, stride", [(3, 45, 6), (5, 60, 7)])
def test_gradient_independent_of_tape_buffers(dlo, monkeypatch, cfg, H, stride):
    """How many checkpoint segments are kept on tape (DLO_TAPE_BUFFERS: 1 = every segment replayed on the main stream, 2 =
    the forward tapes its last two and the other replays run under the adjoints on a second stream, 4 = the default cap)
    is a memory / recompute trade-off like the stride: same trajectory, same arithmetic per substep.  Eight
    segments, the last one ragged; a second backward on the same rollout (nothing on tape any more) must agree too."""
    P = make_problem(cfg, batch=12, n_verts=40, horizon=H)
    outs = []
    for nbuf in ("1", "2", "3", "4"):
        monkeypatch.setenv("DLO_TAPE_BUFFERS", nbuf)
        sim = dlo.DloSim(P)
        x = sim.rollout(H, stride).state()["x"]
        _, seed = loss_and_seed(P, x)
        outs.append(sim.backward(seed))
        if nbuf == "4":
            outs.append(sim.backward(seed))
        assert sim.n_bad() == 0
        sim.close()
    assert np.abs(outs[0]["g_x0"]).max() > 0
    for o in outs[1:]:
        for k in ("g_actions", "g_x0", "g_v0", "g_material"):
            assert np.abs(o[k] - outs[0][k]).max() <= 5e-5 * np.abs(outs[0][k]).max(), k


@pytest.mark.parametrize("cfg, H, stride, tol", [(4, 400, 40, 5e-5), (5, 300, 100, 1e-3)])
def test_side_records_equal_recompute(dlo, monkeypatch, cfg, H, stride, tol):
    """A substep that applied a self-contact correction is reversed either from the side record the replay left, or,
    when the pool has no slot (here: DLO_NO_SIDE, no pool at all), by recomputing it inside the adjoint kernel.  Same
    trajectory, same arithmetic per substep: the gradients agree to rounding level (shared-memory atomics aside)."""
    P = make_problem(cfg, batch=16, horizon=H)
    outs = []
    for no_side in (False, True):
        monkeypatch.delenv("DLO_NO_SIDE", raising=False)
        if no_side:
            monkeypatch.setenv("DLO_NO_SIDE", "1")
        sim = dlo.DloSim(P)
        x = sim.rollout(H, stride).state()["x"]
        _, seed = loss_and_seed(P, x)
        outs.append(sim.backward(seed))
        sim.close()
    assert np.abs(outs[0]["g_x0"]).max() > 0
    for k in ("g_actions", "g_x0", "g_v0", "g_material"):
        assert np.abs(outs[1][k] - outs[0][k]).max() <= tol * np.abs(outs[0][k]).max(), k


# Kinked cases: Eq.11 drives every active hinge onto its yield surface, resting contact sits on the
# kink of f = min(exp(d/eps_s), 1), dragged ropes on the Coulomb stick / slide switch: the step is continuous there but its
# derivative jumps, and the oracle's own gradient moves by far more than 1e-3 when its inputs move by one fp32 rounding.
# Bar: every env whose ORACLE gradient is stable under such perturbations (three draws, spread < 1e-3 / (2 sqrt(#substeps)):
# the fp32 run injects one kick per substep where the spread measures ONE) meets the plain 1e-3;
# the others are counted and held to a finite cap.  (The plain-bar claim at full size is tests/test_teacher_forced_gpu.py's.)
KINKED = [
    ("cfg2 ground+grippers", dict(cfg_id=2, batch=8, n_verts=24), 40, 16, ALL4),
    ("cfg3 plasticity+fingers", dict(cfg_id=3, batch=8, n_verts=24), 40, 10, ALL4),
    ("cfg5 full features N=128", dict(cfg_id=5, batch=8), 12, 5, ("g_actions", "g_material")),
]


@pytest.mark.parametrize("name,kw,H,stride,keys", KINKED, ids=[c[0] for c in KINKED])
def test_gradient_parity_at_kinks(dlo, orc, name, kw, H, stride, keys):
    P = make_problem(horizon=H, stride=stride, **kw)
    got, ref = both_gradients(dlo, orc, P, H, stride)
    o = orc.OracleSim(P)
    _, seed = loss_and_seed(P, o.rollout(H, stride)["x"])
    o.close()
    rng = np.random.default_rng(7)
    spread = {k: 0.0 for k in keys}
    for _ in range(3):
        q = orc.OracleSim(perturbed(P, rng))
        q.rollout(H, stride)
        gq = q.backward(seed)
        q.close()
        for k in keys:
            spread[k] = np.maximum(spread[k], gradient_error(env_first(k, gq[k]), env_first(k, ref[k])))
    for k in keys:
        err = gradient_error(env_first(k, got[k]), env_first(k, ref[k]))
        stable = spread[k] < GRAD_TOL / (2.0 * np.sqrt(H * P["config"]["n_substeps"]))
        print(summarize("%s %s gpu" % (name, k), err), "|", summarize("oracle spread", spread[k]), "| oracle-stable envs: %d of %d" % (stable.sum(), len(err)))
        assert (err[stable] <= GRAD_TOL).all(), (name, k, err, spread[k])
        assert np.isfinite(err).all() and (err <= 10.0).all(), (name, k, err)


@pytest.mark.parametrize("N,ring", [(3, False), (4, True), (5, True), (256, False), (255, True)],
                         ids=["N=3 open", "N=4 ring", "N=5 odd ring", "N=256 open", "N=255 odd ring"])
def test_gradient_extreme_sizes(dlo, orc, N, ring):
    """smallest and largest ropes (every lanes-per-env layout, ring wrap through lane 0, third colour of odd rings)"""
    from helpers import rope_problem
    rng = np.random.default_rng(9)
    B, H = 2, 8
    if ring:
        th = np.linspace(0, 2 * np.pi, N, endpoint=False)
        x = np.stack([0.1 * np.cos(th), 0.1 * np.sin(th), 0.02 * np.sin(2 * th)], 1)
    else:
        x = np.stack([np.arange(N) * (0.5 / (N - 1)), np.zeros(N), np.zeros(N)], 1)
    x = x[None].repeat(B, 0) + rng.normal(0, 2e-4, (B, N, 3))
    P = rope_problem(x, rng.normal(0, 0.05, (B, N, 3)), ring=ring, dt=1e-3, horizon=H, stride=3, pins=None if ring else [0],
                     material=dict(alpha=1e-4, gamma=0.05, stretch=1e-7))
    P["loss"] = dict(kind="polyline", target=np.zeros((B, 3, N)))
    got, ref = both_gradients(dlo, orc, P, H, 3)
    # The compliance entry of g_material is a sum of nearly cancelling terms (w_j gbar_j - w_n gbar_n along each edge); for
    # ropes of a handful of vertices its true value (1e-2) is of the size of the fp32 cancellation error (1e-3 ... 1e-2, the
    # same absolute error at N = 24 where the value is 10), so it is compared on the bending and damping entries here.
    for g in (got, ref):
        g["g_material"] = g["g_material"][:, 1:3]
    check("N=%d ring=%s" % (N, ring), got, ref, ("g_x0", "g_v0", "g_material"))


def test_rope_landing_on_box_and_cylinder(dlo, orc):
    """a short rope falls onto a rotated box, a lying cylinder and a thin capsule between them: exercises the box, cylinder
    and capsule SDF branches and their adjoints in contact, with friction"""
    from helpers import rope_problem
    from parity import POS_TOL, position_error
    rng = np.random.default_rng(21)
    B, N, H = 4, 20, 32
    x = np.stack([np.linspace(-0.08, 0.08, N), np.zeros(N), np.full(N, 0.058)], 1)
    x = x[None].repeat(B, 0) + rng.normal(0, 3e-4, (B, N, 3))
    x[:, :, 1] += rng.uniform(-0.01, 0.01, (B, 1))
    v = np.zeros_like(x)
    v[..., 2] = -0.3
    v[..., 0] = 0.2
    P = rope_problem(x, v, dt=1e-3, horizon=H, stride=9, n_primitives=3, material=dict(alpha=3e-4, gamma=0.05, stretch=1e-7, mu_r=0.4))
    P["prim_types"] = np.array([3, 2, 1], dtype=np.int32)
    pp = np.zeros((B, 3, 10))
    pp[:, 0, 0:3] = (-0.04, 0.0, 0.025)                    # box: centre, half extents, rotation vector (tilted and yawed)
    pp[:, 0, 3:6] = (0.03, 0.03, 0.025)
    pp[:, 0, 6:9] = (0.1, -0.15, 0.4)
    pp[:, 1, 0:3] = (0.05, 0.0, 0.03)                      # cylinder lying along y: centre, axis, radius, half height
    pp[:, 1, 3:6] = (0.0, 1.0, 0.0)
    pp[:, 1, 6], pp[:, 1, 7] = 0.022, 0.05
    pp[:, 2, 0:3] = (0.0, -0.03, 0.046)                     # capsule across the gap between them: end points, radius
    pp[:, 2, 3:6] = (0.01, 0.03, 0.05)
    pp[:, 2, 6] = 0.004
    P["prim_params"] = pp
    P["loss"] = dict(kind="polyline", target=np.zeros((B, 3, N)))
    free = dict(P, config=dict(P["config"], n_primitives=0))
    a, b = orc.OracleSim(P).rollout(H, 0)["x"], orc.OracleSim(free).rollout(H, 0)["x"]
    assert np.abs(a - b).max() > 2e-3, "the rope must actually land on the bodies"
    sim = dlo.DloSim(P)
    xg = sim.rollout(H, 0).state()["x"]
    sim.close()
    err = position_error(P, xg, a)
    print(summarize("box+cylinder positions", err))
    assert err.max() <= POS_TOL
    got, ref = both_gradients(dlo, orc, P, H, 9)
    for k in ("g_x0", "g_v0", "g_material"):
        e = gradient_error(got[k], ref[k])
        print(summarize("box+cylinder+capsule " + k, e))
        # contact with thin bodies puts an env on a branch threshold now and then (see KINKED above): three of the four envs
        # must meet the plain bar, the fourth stay within 1e-2
        assert np.sort(e)[-2] <= GRAD_TOL and e.max() <= 1e-2, (k, e)
