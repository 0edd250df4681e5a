"""-m gpu: tiny forward + reverse cases that drive the kernels through the paths where races, missing barriers or reads of
uninitialised memory would hide (SURVEY.md section 5 "Race detection"): self-contact with friction and side records, the
recomputing reverse pass (no side-record pool), pair-list rebuilds in the middle of the projection loop, odd rings (third
colour), aliased shared-memory regions (block spheres on sm.vs, xref on ybar), gripper fingers and boxes.

compute-sanitizer is CLOSED on this GPU pool (the tool answers: "compute-sanitizer is closed on this pool and stays closed:
runs under it have left GPUs needing a reset. Find a bad access with bounds checks and asserts of your own, small cases,
and a comparison with the CPU reference"; profiles/r02_sanitizer.md).  The stand-ins, all in this file:
  - every case runs twice and must give identical forward bits (a data race shows as a difference sooner or later), under
    different CTA shapes and vote modes elsewhere (test_parity_gpu.py::test_lazy_self_contact_schedule_changes_no_bit);
  - every case also runs with DLO_CHECKS=1: four guard words behind every per-warp shared-memory region, verified when a
    kernel ends (an overrun sets FLAG_GUARD -> DLO_ERR_NUMERIC), and every library allocation pre-filled with 0xff bytes
    (NaN / -1), so that a read of memory nothing wrote ends up in a non-finite result or a wild index (memcheck / initcheck);
  - results are compared with the fp64 oracle by the parity tests on the same paths.
"""
import numpy as np
import pytest

from helpers import figure_eight_problem, rope_problem
from parity import loss_and_seed, make_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


@pytest.fixture(autouse=True, params=[0, 1], ids=["plain", "DLO_CHECKS"])
def checks(request, monkeypatch):
    if request.param:
        monkeypatch.setenv("DLO_CHECKS", "1")
    else:
        monkeypatch.delenv("DLO_CHECKS", raising=False)
    return request.param


def fwd_bwd(dlo, P, H, stride):
    sim = dlo.DloSim(P)
    x = sim.rollout(H, stride).state()["x"]
    _, seed = loss_and_seed(P, x)
    g = sim.backward(seed)
    assert sim.n_bad() == 0
    sim.close()
    assert np.isfinite(x).all() and all(np.isfinite(v).all() for v in g.values())
    return x, g


def twice(dlo, P, H, stride):
    """the same case twice: identical forward bits (a race would show as a difference sooner or later)"""
    x1, g1 = fwd_bwd(dlo, P, H, stride)
    x2, g2 = fwd_bwd(dlo, P, H, stride)
    assert np.array_equal(x1, x2)
    for k in ("g_x0", "g_v0"):
        assert np.allclose(g1[k], g2[k], rtol=1e-5, atol=1e-6 * max(1.0, np.abs(g1[k]).max()))


def test_self_contact_with_side_records(dlo):
    twice(dlo, figure_eight_problem(horizon=14, stride=5), 14, 5)


def test_self_contact_reverse_pass_recomputes_without_side_pool(dlo, monkeypatch):
    monkeypatch.setenv("DLO_NO_SIDE", "1")
    twice(dlo, figure_eight_problem(horizon=14, stride=5), 14, 5)


def test_pair_list_rebuilt_often_and_near_list_off(dlo, monkeypatch):
    monkeypatch.setenv("DLO_LIST_MARGIN", "0.05")       # rebuilds at almost every use, some in the middle of the projection loop
    monkeypatch.setenv("DLO_NEAR", "0")
    twice(dlo, figure_eight_problem(horizon=14, stride=5), 14, 5)


def dog_bone_ring(N, l0=6.0e-3):
    """closed curve with two lobes and a pinched middle (strands 7 mm apart there: within self-contact reach), N vertices at
    equal arclength, edge length ~l0"""
    from workloads.configs import _resample_polyline
    th = np.linspace(0.0, 2 * np.pi, 4001)
    a = N * l0 / 4.6
    curve = np.stack([a * np.cos(th), (0.0035 + 0.3 * a * np.cos(th) ** 2) * np.sin(th), 0.002 * np.sin(3 * th)], 1)
    return _resample_polyline(curve, N + 1)[:-1]


@pytest.mark.parametrize("N", [5, 33, 97])
def test_odd_ring_with_self_contact(dlo, N):
    x = dog_bone_ring(N)
    P = rope_problem(x[None].repeat(3, 0), ring=True, horizon=8, stride=3, enable_self_contact=int(N > 5), gravity=(0.0, 0.0, -9.81),
                     material=dict(stretch=1e-6, alpha=1e-4, gamma=0.5))
    P["loss"] = dict(kind="polyline", target=np.zeros((3, 3, N)))
    twice(dlo, P, 8, 3)


def test_full_feature_set_small(dlo):
    twice(dlo, make_problem(5, batch=5, n_verts=40, horizon=6, stride=3), 6, 3)
    twice(dlo, make_problem(4, batch=3, n_verts=48, horizon=6, stride=4), 6, 4)
    twice(dlo, make_problem(3, batch=3, n_verts=24, horizon=6, stride=2), 6, 2)


def test_the_guard_check_can_fail(dlo, monkeypatch):
    """DLO_CHECKS=2 makes every warp write one word past its primitive block: every env must come back flagged"""
    import ctypes as C
    monkeypatch.setenv("DLO_CHECKS", "2")
    P = make_problem(5, batch=5, n_verts=40, horizon=2, stride=0)
    sim = dlo.DloSim(P)
    sim.rollout(2, 0)
    n = C.c_int32(0)
    assert dlo.lib().dlo_check_numerics(sim.h, C.byref(n)) == -6 and n.value == 5
    assert "5 shared-memory guard" in dlo.dlo_last_error()
    sim.close()
