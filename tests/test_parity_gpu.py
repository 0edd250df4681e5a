"""-m gpu: the CUDA path (through the C-ABI) against the fp64 oracle on the same seeded inputs, element by element.

Forward parity: max vertex distance / rope length <= 1e-4 after the stated horizon (BASELINE.json north_star).
Sizes are the five configs reduced in batch (envs are independent, so a subset is sound) plus ragged vertex
counts that exercise every lanes-per-env layout (VPL 2/4/6/8), partial last lanes, odd rings and both stretch modes.
"""
import numpy as np
import pytest

from parity import POS_TOL, make_problem, oracle_position_spread, position_error, summarize

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def run_both(dlo, orc, P, horizon=None, stride=0):
    H = P["horizon"] if horizon is None else horizon
    sim = dlo.DloSim(P)
    sim.rollout(H, stride)
    got = sim.state()
    assert sim.n_bad() == 0
    sim.close()
    o = orc.OracleSim(P)
    ref = o.rollout(H, stride)
    o.close()
    return got, ref


FORWARD_CASES = [
    ("cfg1 full", dict(cfg_id=1), None),
    ("cfg2 64 envs", dict(cfg_id=2, batch=64), None),
    ("cfg3 64 envs", dict(cfg_id=3, batch=64), None),
    ("cfg4 32 envs", dict(cfg_id=4, batch=32), None),
    ("cfg5 16 envs, 60 steps", dict(cfg_id=5, batch=16, horizon=60), None),
    ("cfg5 16 envs, 300 steps", dict(cfg_id=5, batch=16, horizon=300), None),
    ("cfg2 N=37 (VPL 2, ragged)", dict(cfg_id=2, batch=8, n_verts=37, horizon=100), None),
    ("cfg5 N=100 (VPL 4, ragged)", dict(cfg_id=5, batch=8, n_verts=100, horizon=100), None),
    ("cfg5 N=130 (VPL 6)", dict(cfg_id=5, batch=4, n_verts=130, horizon=60), None),
    ("cfg5 N=200 (VPL 8)", dict(cfg_id=5, batch=4, n_verts=200, horizon=40), None),
    ("cfg4 N=45 (odd ring)", dict(cfg_id=4, batch=8, n_verts=45, horizon=150), None),
    ("cfg4 N=98 (even ring, ragged)", dict(cfg_id=4, batch=4, n_verts=98, horizon=100), None),
    ("cfg1 stretch energy", dict(cfg_id=1, n_verts=24), dict(stretch_mode=0, stretch=2.0e2)),
]


@pytest.mark.parametrize("name,kw,over", FORWARD_CASES, ids=[c[0] for c in FORWARD_CASES])
def test_forward_parity(dlo, orc, name, kw, over):
    P = make_problem(**kw)
    if over:
        P["config"]["stretch_mode"] = over["stretch_mode"]
        P["material"]["stretch"][:] = over["stretch"]
    got, ref = run_both(dlo, orc, P)
    err = position_error(P, got["x"], ref["x"])
    print(summarize(name, err))
    assert np.isfinite(got["x"]).all()
    E = P["config"]["n_verts"] - (0 if P["config"]["topology"] else 1)
    d1 = got["d1"][:, :, :E]
    assert np.abs(np.linalg.norm(d1, axis=1) - 1).max() < 1e-5          # frames stay unit (state invariant of A9), chaotic or not
    if err.max() > POS_TOL:
        # Some envs of the contact-rich workloads are chaotic at this horizon: the ORACLE's own final positions move by more
        # than the tolerance when its inputs move by one fp32 rounding.  The plain bar is asserted on
        # every env whose oracle result is stable under such a perturbation: the fp32 run injects one rounding-sized kick per
        # substep where the spread measures the effect of ONE, so "stable" is spread < tolerance / (2 sqrt(#substeps)); the
        # others are counted and held to a finite cap.  The plain-bar claim on those workloads is tests/test_teacher_forced_gpu.py's.
        spread = oracle_position_spread(orc, P, P["horizon"], ref["x"])
        stable = spread < POS_TOL / (2.0 * np.sqrt(P["horizon"] * P["config"]["n_substeps"]))
        print(summarize(name + " oracle spread", spread), "| oracle-stable envs: %d of %d" % (stable.sum(), len(err)))
        assert (err[stable] <= POS_TOL).all(), (name, err, spread)
        assert (err <= 0.5).all(), (name, err)
        return
    # frames and rest curvature follow the oracle's
    dref = ref["d1"][:, :, :E]
    assert np.abs(d1 - dref).max() < 5e-3
    assert np.abs(got["kappa_bar"] - ref["kappa_bar"]).max() < 5e-3 * max(1.0, np.abs(ref["kappa_bar"]).max())


def test_rollout_is_repeatable_bitwise(dlo):
    """two rollouts from the same state give identical bits (deterministic reductions, no atomics on the path)"""
    P = make_problem(4, batch=16, horizon=120)
    sim = dlo.DloSim(P)
    a = sim.rollout(120, 0).state()
    b = sim.rollout(120, 40).state()
    sim.close()
    for k in a:
        assert np.array_equal(a[k], b[k]), k


@pytest.mark.parametrize("cfg, B, H", [(4, 32, 400), (5, 32, 700)])
def test_lazy_self_contact_schedule_changes_no_bit(dlo, cfg, B, H, monkeypatch):
    """DESIGN.md section 5 "exact but lazy": when the pair list is rebuilt, which pairs sit in the near list and whether the
    warps of a CTA refresh together only decide WHEN distances are measured, never the result: the final state has the
    same bits under every schedule (the overrides are read at dlo_create)."""
    P = make_problem(cfg, batch=B, horizon=H)
    ref = None
    for env in ({}, {"DLO_NEAR": "0"}, {"DLO_NEAR": "3.9"}, {"DLO_LIST_MARGIN": "0.2"}, {"DLO_VOTE": "0"}, {"DLO_VOTE": "1", "DLO_LIST_MARGIN": "2.5"}):
        for k in ("DLO_NEAR", "DLO_LIST_MARGIN", "DLO_VOTE"):
            monkeypatch.delenv(k, raising=False)
        for k, v in env.items():
            monkeypatch.setenv(k, v)
        sim = dlo.DloSim(P)
        got = sim.rollout(H, 0).state()
        sim.close()
        if ref is None:
            ref = got
        for k in ref:
            assert np.array_equal(ref[k], got[k]), (env, k)


def test_empty_horizon_and_call_order(dlo):
    P = make_problem(1)
    sim = dlo.DloSim(P)
    s0 = sim.rollout(0, 0).state()
    assert np.allclose(s0["x"], P["x0"], atol=1e-7)
    with pytest.raises(dlo.DloError) as e:
        sim.backward(np.zeros((1, 3, 32)))
    assert e.value.status == -2
    sim.close()


# ---- edge cases: smallest and largest ropes, degenerate scenes, error behaviour ---------------------------------------
def _plain_rope(N, ring, B=3, H=25, seed=3, **cfg):
    from helpers import rope_problem
    rng = np.random.default_rng(seed)
    if ring:
        th = np.linspace(0, 2 * np.pi, N, endpoint=False)
        x = np.stack([0.1 * np.cos(th), 0.1 * np.sin(th), 0.02 * np.sin(2 * th)], 1)
    else:
        x = np.stack([np.arange(N) * (0.5 / max(N - 1, 1)), np.zeros(N), np.zeros(N)], 1)
    x = x[None].repeat(B, 0) + rng.normal(0, 2e-4, (B, N, 3))
    v = rng.normal(0, 0.05, (B, N, 3))
    pins = None if ring else [0]
    return rope_problem(x, v, ring=ring, dt=1e-3, horizon=H, pins=pins, material=dict(alpha=1e-4, gamma=0.05, stretch=1e-7), **cfg)


@pytest.mark.parametrize("N,ring", [(3, False), (4, True), (5, True), (256, False), (255, True), (64, False), (65, False)],
                         ids=["N=3 open (minimum)", "N=4 ring (minimum)", "N=5 odd ring", "N=256 open (maximum)", "N=255 odd ring",
                              "N=64 (full warp at VPL 2)", "N=65 (first size at VPL 4)"])
def test_extreme_sizes(dlo, orc, N, ring):
    P = _plain_rope(N, ring, H=15 if N > 200 else 25)
    got, ref = run_both(dlo, orc, P)
    err = position_error(P, got["x"], ref["x"])
    print(summarize("N=%d ring=%s" % (N, ring), err))
    assert err.max() <= POS_TOL


def test_no_projection_iterations_and_no_substep_split(dlo, orc):
    """N_C = 0 (pure symplectic Euler on the energies) and n_substeps = 1"""
    P = _plain_rope(20, False, n_proj_iters=0, n_substeps=1, stretch_mode=0)
    P["material"]["stretch"][:] = 50.0
    got, ref = run_both(dlo, orc, P)
    assert position_error(P, got["x"], ref["x"]).max() <= POS_TOL


def test_argument_and_order_errors(dlo):
    import torch
    P = make_problem(2, batch=4, n_verts=16, horizon=10)
    sim = dlo.DloSim(P)
    with pytest.raises(dlo.DloError) as e:          # horizon beyond the actions given
        dlo.dlo_rollout_forward(sim.h, 11, 0)
    assert e.value.status == -1
    with pytest.raises(dlo.DloError) as e:          # negative stride
        dlo.dlo_rollout_forward(sim.h, 5, -1)
    assert e.value.status == -1
    sim.rollout(10, 0)
    with pytest.raises(dlo.DloError) as e:          # backward without checkpoints
        sim.backward(np.zeros((4, 3, 16)))
    assert e.value.status == -2
    # changing the scene invalidates the state until dlo_set_state is called again
    dlo.dlo_set_pins(sim.h, torch.zeros((4, 16), dtype=torch.uint8, device="cuda"))
    with pytest.raises(dlo.DloError) as e:
        dlo.dlo_rollout_forward(sim.h, 5, 0)
    assert e.value.status == -2
    assert sim.n_bad() == 0
    sim.close()


def test_non_finite_state_is_flagged(dlo):
    P = make_problem(1)
    P["x0"][0, 0, 5] = np.nan
    sim = dlo.DloSim(P)
    sim.rollout(3, 0)
    assert sim.n_bad() == 1
    sim.close()


def test_host_buffer_calls_match_device_calls(dlo):
    """dlo_rollout_forward_host / dlo_backward_host (the e2e path of bench.py) give the same bits as the device-pointer calls"""
    P = make_problem(3, batch=8, n_verts=24, horizon=20, stride=7)
    from parity import loss_and_seed
    sim = dlo.DloSim(P)
    sim.rollout(20, 7)
    xd = sim.state_device()["x"].double().cpu().numpy()      # the fp32 positions dlo_get_state returns (without the residual)
    _, seed = loss_and_seed(P, xd)
    gd = sim.backward(seed)
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    x0, v0, act = f32(P["x0"]), f32(P["v0"]), f32(P["actions"])
    xT, vT = np.empty_like(x0), np.empty_like(x0)
    dlo.dlo_rollout_forward_host(sim.h, x0, v0, None, act, 20, 7, xT, vT)
    assert np.array_equal(xT.astype(np.float64), xd)
    ga, gx, gv, gm = np.empty_like(act), np.empty_like(x0), np.empty_like(x0), np.empty((8, 5), dtype=np.float32)
    dlo.dlo_backward_host(sim.h, f32(seed), None, ga, gx, gv, gm)
    assert np.allclose(gx, gd["g_x0"], rtol=1e-5, atol=1e-9) and np.allclose(gv, gd["g_v0"], rtol=1e-5, atol=1e-9)
    assert np.allclose(ga, gd["g_actions"], rtol=1e-4, atol=1e-7 * np.abs(gd["g_actions"]).max())
    sim.close()


def test_trajectory_matches_oracle_at_every_recorded_time(dlo, orc):
    """not only the final state: the state after 1, 2, 7, 23 and 60 frames (ring on posts with a gripper, config 4)"""
    P = make_problem(4, batch=4, n_verts=48, horizon=60)
    o = orc.OracleSim(P)
    o.rollout(60, 0, record=True)
    sim = dlo.DloSim(P)
    for t in (1, 2, 7, 23, 60):
        got = sim.rollout(t, 0).state()
        ref = o.record(t)
        assert position_error(P, got["x"], ref["x"]).max() <= POS_TOL, t
        assert np.abs(got["v"] - ref["v"]).max() <= 1e-3 * max(1.0, np.abs(ref["v"]).max()), t
    sim.close()
    o.close()


def test_rest_shape_is_stationary_on_the_gpu(dlo, orc):
    """a curved rope / a non-planar ring whose rest curvature is its own shape (kappa_bar_from_x0), no gravity: nothing moves
    (pin C-7 of the oracle, here for the CUDA path: frames, Eq.12 and the bending force are consistent)"""
    from helpers import rope_problem
    for ring in (False, True):
        N = 40
        if ring:
            th = np.linspace(0, 2 * np.pi, N, endpoint=False)
            x = np.stack([0.1 * np.cos(th), 0.1 * np.sin(th), 0.02 * np.sin(2 * th)], 1)
        else:
            s = np.linspace(0, 1, N)
            x = np.stack([0.3 * s, 0.05 * np.sin(3 * s), 0.04 * np.cos(2 * s)], 1)
        if not ring:      # equal edge lengths so that the stretch constraints are satisfied too
            from workloads.configs import _resample_polyline
            x = _resample_polyline(x, N)
        P = rope_problem(x[None], ring=ring, dt=1e-3, horizon=50, gravity=(0.0, 0.0, 0.0), kappa_bar_from_x0=1,
                         material=dict(alpha=1e-3, stretch=1e-5))
        sim = dlo.DloSim(P)
        got = sim.rollout(50, 0).state()
        sim.close()
        ref = orc.OracleSim(P).rollout(50, 0)
        L = np.linalg.norm(np.diff(x, axis=0), axis=1).sum()
        moved_gpu = np.linalg.norm(got["x"][0].T - x, axis=1).max()
        moved_orc = np.linalg.norm(ref["x"][0].T - x, axis=1).max()
        # the oracle itself moves only by the residual of unequal chord lengths against the mean rest length
        assert moved_gpu <= moved_orc + 2e-5 * L, (ring, moved_gpu, moved_orc)
        assert position_error(P, got["x"], ref["x"]).max() <= POS_TOL
        if not ring:
            assert moved_gpu <= 2e-5 * L
