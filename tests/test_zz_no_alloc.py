"""-m gpu: dlo_rollout_forward_static, the forward rollout for callers that cannot call cudaMalloc (scratch in a static
device array of DLO_STATIC_SCRATCH_BYTES, include/dlo.h), against the handle path (dlo_create ... dlo_rollout_forward) on the
same inputs, on two calls in a row of DIFFERENT shapes (the second call finds the first one's contents in the array) and a
third that repeats the first.  Collected last on purpose (the suite runs with pytest -x)."""
import numpy as np
import pytest

from parity import POS_TOL, make_problem, position_error

pytestmark = pytest.mark.gpu

VEL_TOL = 1e-3   # relative to the env's largest speed; the two paths run the same kernels, so both bars are met with a lot of room


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def upload(P, dev):
    import torch
    up = lambda a, dt=torch.float32: torch.as_tensor(np.ascontiguousarray(a), dtype=dt).to(dev).contiguous()
    cfg = P["config"]
    mat = {k: up(v) for k, v in P["material"].items()}
    scene = {}
    if P.get("pins") is not None:
        scene["pinned"] = up(P["pins"], torch.uint8)
    if cfg["n_primitives"] > 0:
        scene["prim_types"], scene["prim_params"] = np.asarray(P["prim_types"], dtype=np.int32), up(P["prim_params"])
    if cfg["n_grippers"] > 0:
        scene.update(init_pose=up(P["init_pose"]), finger_geom=up(P["finger_geom"]), grasp_verts=up(P["grasp_verts"], torch.int32),
                     actions=up(P["actions"]))
    kb = P.get("kappa_bar0")
    return mat, scene, up(P["x0"]), up(P["v0"]), None if kb is None else up(kb)


def static_rollout(dlo, P, H, dev, check_free=False):
    import torch
    cfg = P["config"]
    B, N = cfg["batch"], cfg["n_verts"]
    mat, scene, x0, v0, kb = upload(P, dev)
    xT, vT = torch.full((B, 3, N), float("nan"), device=dev), torch.full((B, 3, N), float("nan"), device=dev)
    flags = torch.full((B,), -1, dtype=torch.int32, device=dev)
    torch.cuda.synchronize(dev)
    free0 = torch.cuda.mem_get_info(dev)[0]
    dlo.dlo_rollout_forward_static(dlo.make_config(cfg), mat, scene, x0, v0, kb, H, xT, vT, flags, torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize(dev)
    if check_free:   # a cudaMalloc inside the call would show here (torch's own allocations were all made before)
        assert torch.cuda.mem_get_info(dev)[0] == free0
    return xT.double().cpu().numpy(), vT.double().cpu().numpy(), flags.cpu().numpy()


def handle_rollout(dlo, P, H):
    sim = dlo.DloSim(P)
    sim.rollout(H, 0)
    st = sim.state_device()
    assert sim.n_bad() == 0
    out = st["x"].double().cpu().numpy(), st["v"].double().cpu().numpy()
    sim.close()
    return out


def compare(P, got, want):
    e_pos = position_error(P, got[0], want[0])
    vmax = np.maximum(np.abs(want[1]).reshape(len(e_pos), -1).max(axis=1), 1e-2)
    e_vel = np.abs(got[1] - want[1]).reshape(len(e_pos), -1).max(axis=1) / vmax
    print("static vs handle: positions max %.2e (bar %.0e), velocities max %.2e (bar %.0e), bitwise equal: %s"
          % (e_pos.max(), POS_TOL, e_vel.max(), VEL_TOL, np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])))
    assert np.isfinite(got[0]).all() and np.isfinite(got[1]).all()
    assert e_pos.max() <= POS_TOL and e_vel.max() <= VEL_TOL
    assert (got[2] == 0).all()


def test_static_rollout_matches_the_handle_path_on_two_calls_in_a_row(dlo):
    import torch
    dev = torch.device("cuda:0")
    # ropes with grippers, primitives and self-contact (config 5's recipe), then a different shape (config 3's: 24 vertices, other
    # gripper count / horizon), then the first again with the allocation check on
    PA, HA = make_problem(5, batch=24, n_verts=40, horizon=12), 12
    PB, HB = make_problem(3, batch=37, n_verts=24, horizon=20), 20
    want_a, want_b = handle_rollout(dlo, PA, HA), handle_rollout(dlo, PB, HB)
    for c in (PA, PB):
        assert 0 < dlo.dlo_static_scratch_bytes(dlo.make_config(c["config"])) <= dlo.STATIC_SCRATCH_BYTES
    compare(PA, static_rollout(dlo, PA, HA, dev), want_a)
    compare(PB, static_rollout(dlo, PB, HB, dev), want_b)
    compare(PA, static_rollout(dlo, PA, HA, dev, check_free=True), want_a)


def test_static_rollout_refuses_what_does_not_fit(dlo):
    import torch
    dev = torch.device("cuda:0")
    P = make_problem(3, batch=8, n_verts=24, horizon=2)
    mat, scene, x0, v0, kb = upload(P, dev)
    big = dict(P["config"])
    big["batch"] = 1 << 16                                  # 65536 envs x 24 vertices: ~100 MB of state
    assert dlo.dlo_static_scratch_bytes(dlo.make_config(big)) > dlo.STATIC_SCRATCH_BYTES
    with pytest.raises(dlo.DloError) as e:                 # refused before any pointer is touched
        dlo.dlo_rollout_forward_static(dlo.make_config(big), mat, scene, x0, v0, kb, 2, None, None, None, 0)
    assert e.value.status == -5 and "DLO_STATIC_SCRATCH_BYTES" in str(e.value)
    bad = dict(P["config"])
    bad["n_verts"] = 2
    assert dlo.dlo_static_scratch_bytes(dlo.make_config(bad)) == 0
    with pytest.raises(dlo.DloError) as e:
        dlo.dlo_rollout_forward_static(dlo.make_config(bad), mat, scene, x0, v0, kb, 2, None, None, None, 0)
    assert e.value.status == -1
