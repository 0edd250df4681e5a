"""-m gpu: boundary behaviour of the C-ABI that round 1 left untested (VERDICT r01 "Boundary details"):
handle-owned staging of the *_host calls with two live handles, and the self-contact candidate overflow flag."""
import ctypes as C

import numpy as np
import pytest

from helpers import rope_problem
from parity import loss_and_seed, make_problem

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def host_pass(dlo, sim, P, H, S, seed=None):
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    x0, v0, act = f32(P["x0"]), f32(P["v0"]), f32(P["actions"])
    xT, vT = np.empty_like(x0), np.empty_like(x0)
    dlo.dlo_rollout_forward_host(sim.h, x0, v0, None, act, H, S, xT, vT)
    return xT, vT


def host_backward(dlo, sim, P, xT, H):
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    _, seed = loss_and_seed(P, xT.astype(np.float64))
    B, N, G = P["config"]["batch"], P["config"]["n_verts"], P["config"]["n_grippers"]
    ga, gx, gv, gm = np.empty((H, B, G, 6), np.float32), np.empty((B, 3, N), np.float32), np.empty((B, 3, N), np.float32), np.empty((B, 5), np.float32)
    dlo.dlo_backward_host(sim.h, f32(seed), None, ga, gx, gv, gm)
    return ga, gx, gv, gm


def test_two_handles_interleave_through_the_host_calls(dlo):
    """Two live simulators of different sizes driven alternately through dlo_rollout_forward_host / dlo_backward_host give
    what each gives alone: the staging (and the borrowed device copy of the actions) belongs to the handle."""
    PA = make_problem(3, batch=8, n_verts=24, horizon=20, stride=7)
    PB = make_problem(5, batch=6, n_verts=40, horizon=12, stride=5)
    ref = []
    for P, H, S in ((PA, 20, 7), (PB, 12, 5)):
        sim = dlo.DloSim(P)
        xT, vT = host_pass(dlo, sim, P, H, S)
        ref.append((xT, vT) + host_backward(dlo, sim, P, xT, H))
        sim.close()
    a, b = dlo.DloSim(PA), dlo.DloSim(PB)
    xa, va = host_pass(dlo, a, PA, 20, 7)
    xb, vb = host_pass(dlo, b, PB, 12, 5)            # larger action array than a's: would have reallocated a shared buffer
    ga = host_backward(dlo, a, PA, xa, 20)           # a replays ITS actions
    gb = host_backward(dlo, b, PB, xb, 12)
    xa2, _ = host_pass(dlo, a, PA, 20, 7)
    for got, want in (((xa, va) + ga, ref[0]), ((xb, vb) + gb, ref[1])):
        assert np.array_equal(got[0], want[0]) and np.array_equal(got[1], want[1])
        for g, w in zip(got[2:], want[2:]):
            assert np.allclose(g, w, rtol=1e-5, atol=1e-7 * max(1.0, np.abs(w).max()))
    assert np.array_equal(xa2, xa)
    assert a.n_bad() == 0 and b.n_bad() == 0
    a.close()
    b.close()


def test_candidate_overflow_is_flagged(dlo):
    """An env whose self-contact candidate list cannot hold its pairs (a rope coiled into a ball smaller than the candidate
    distance) is flagged FLAG_CAND_OVERFLOW: dlo_check_numerics returns DLO_ERR_NUMERIC with the count; the env next to it is not."""
    N, l0 = 64, 2.0e-3
    s = np.arange(N) * l0
    R = 5.0e-3
    coil = np.stack([R * np.cos(s / R), R * np.sin(s / R), 0.05 + 1.0e-3 * s / (2 * np.pi * R)], 1)     # 4 turns, pitch 1 mm
    straight = np.stack([5.0 * s, np.zeros(N), np.full(N, 0.05)], 1)          # 1 cm edges: only a handful of candidate pairs
    P = rope_problem(np.stack([coil, straight]), horizon=2, enable_self_contact=1, gravity=(0.0, 0.0, 0.0),
                     material=dict(l0=np.array([l0, 5.0 * l0]), stretch=1e-6, alpha=1e-5, gamma=1.0))
    sim = dlo.DloSim(P)
    sim.rollout(2, 0)
    n = C.c_int32(0)
    st = dlo.lib().dlo_check_numerics(sim.h, C.byref(n))
    assert st == -6 and n.value == 1
    msg = dlo.dlo_last_error()
    assert "1 env(s) flagged" in msg and "1 self-contact candidate overflow" in msg, msg
    got = sim.state()
    assert np.isfinite(got["x"]).all()              # flagged, not crashed
    # the handle stays usable: a fresh state clears the flags
    sim.set_state(np.stack([P["x0"][0] * np.array([5.0, 5.0, 1.0])[:, None], P["x0"][1]]), P["v0"])   # the coil blown up: loose turns
    sim.rollout(2, 0)
    assert sim.n_bad() <= 1
    sim.close()
