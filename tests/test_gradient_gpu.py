"""-m gpu: reverse pass of the CUDA path (dlo_backward through the C-ABI) against the oracle's tape-AD gradient on the
same seeded inputs.  Tolerance: ||g_gpu - g_orc|| / ||g_orc|| <= 1e-3 per env and gradient tensor (BASELINE.json).
Horizons are kept short enough that the fp64 tape-AD oracle finishes in seconds; strides that do not divide the
horizon exercise the ragged last segment."""
import numpy as np
import pytest

from parity import GRAD_TOL, gradient_error, loss_and_seed, make_problem, summarize

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


CASES = [
    ("cfg1 full (g_v0)", dict(cfg_id=1), 200, 50, ("g_v0", "g_x0")),
    ("cfg1 ragged stride", dict(cfg_id=1, n_verts=20), 23, 7, ("g_v0", "g_x0", "g_material")),
    ("cfg2 ground+grippers", dict(cfg_id=2, batch=4, n_verts=24), 40, 16, ("g_actions", "g_x0", "g_v0", "g_material")),
    ("cfg3 plasticity+fingers", dict(cfg_id=3, batch=4, n_verts=24), 40, 10, ("g_actions", "g_x0", "g_v0", "g_material")),
    ("cfg4 ring+self-contact", dict(cfg_id=4, batch=2, n_verts=48), 30, 10, ("g_actions", "g_x0", "g_v0", "g_material")),
    ("cfg4 odd ring", dict(cfg_id=4, batch=2, n_verts=45), 20, 20, ("g_actions", "g_x0", "g_v0")),
    ("cfg5 full features N=128", dict(cfg_id=5, batch=2), 12, 5, ("g_actions", "g_x0", "g_v0", "g_material")),
    ("cfg5 N=70 (VPL 4 ragged)", dict(cfg_id=5, batch=2, n_verts=70), 12, 12, ("g_actions", "g_x0", "g_v0", "g_material")),
]


@pytest.mark.parametrize("name,kw,H,stride,keys", CASES, ids=[c[0] for c in CASES])
def test_gradient_parity(dlo, orc, name, kw, H, stride, keys):
    P = make_problem(horizon=H, stride=stride, **kw)
    got, ref = both_gradients(dlo, orc, P, H, stride)
    check(name, got, ref, keys)


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
            assert np.allclose(o[k], outs[0][k], rtol=1e-4, atol=1e-7 * np.abs(outs[0][k]).max()), k
