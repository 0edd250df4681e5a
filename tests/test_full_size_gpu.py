"""-m gpu: the five BASELINE.json configs at their FULL sizes, in the launch configuration bench.py times (whole batch, full
horizon, the config's checkpoint stride): the run completes, flags nothing, returns finite states and gradients, and is
compared with the oracle on sampled envs over the WHOLE horizon.

Over the whole horizon configs 2, 3 and 5 are chaotic: the oracle's own result moves by more than the
tolerances when its inputs move by one fp32 rounding.  This file therefore asserts the plain bars only on the envs whose
oracle result is stable under such a perturbation (spread < tolerance / (2 sqrt(#substeps)): the fp32 run injects one
rounding-sized kick per substep where the spread measures the effect of one), prints the errors
of all sampled envs next to the oracle's spread as a long-horizon diagnostic, and leaves the parity claim on the benchmarked
workload to tests/test_teacher_forced_gpu.py, which compares every 5-frame segment of these same rollouts at the plain bars."""
import numpy as np
import pytest

from parity import (GRAD_TOL, POS_TOL, gradient_error, loss_and_seed, make_problem, perturbed, position_error, subset, summarize)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def dlo():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def env_first(k, a):
    return np.moveaxis(a, 1, 0) if k == "g_actions" else a


@pytest.mark.parametrize("cfg_id,n_sample,with_grad", [(1, 1, True), (2, 16, False), (3, 8, True), (4, 4, True), (5, 4, True)])
def test_full_size_config(dlo, orc, cfg_id, n_sample, with_grad):
    P = make_problem(cfg_id)
    B, H, stride = P["config"]["batch"], P["horizon"], P["checkpoint_stride"]
    envs = np.arange(0, B, max(1, B // n_sample))[:n_sample]
    sim = dlo.DloSim(P)
    sim.rollout(H, stride)
    got = sim.state()
    assert sim.n_bad() == 0
    assert all(np.isfinite(v).all() for v in got.values())
    # oracle on the sampled envs (+ its own conditioning under fp32-sized input perturbations)
    Q = subset(P, envs)
    o = orc.OracleSim(Q)
    ref = o.rollout(H, stride)
    q = orc.OracleSim(perturbed(Q, np.random.default_rng(5)))
    ref_p = q.rollout(H, stride)
    err = position_error(Q, got["x"][envs], ref["x"])
    spread = position_error(Q, ref_p["x"], ref["x"])
    kicks = np.sqrt(H * P["config"]["n_substeps"])
    stable = spread < POS_TOL / (2.0 * kicks)
    print(summarize("cfg%d full size, %d frames: positions gpu" % (cfg_id, H), err), "|", summarize("oracle spread", spread),
          "| oracle-stable envs: %d of %d" % (stable.sum(), len(envs)))
    assert (err[stable] <= POS_TOL).all(), (err, spread)
    assert (err <= 0.5).all()                                        # chaotic, not lost: within half a rope length
    if with_grad:
        _, seed = loss_and_seed(Q, ref["x"])
        g_ref, g_prt = o.backward(seed), q.backward(seed)
        full_seed = np.zeros((B,) + seed.shape[1:])
        full_seed[envs] = seed
        g = sim.backward(full_seed)
        assert sim.n_bad() == 0
        for k in P["grad_wrt"]:
            a = env_first(k, g[k])[envs]
            assert np.isfinite(a).all()
            e = gradient_error(a, env_first(k, g_ref[k]))
            s = gradient_error(env_first(k, g_prt[k]), env_first(k, g_ref[k]))
            st = stable & (s < GRAD_TOL / (2.0 * kicks))
            print(summarize("cfg%d full size: %s gpu" % (cfg_id, k), e), "|", summarize("oracle spread", s), "| oracle-stable envs: %d of %d" % (st.sum(), len(envs)))
            assert (e[st] <= GRAD_TOL).all(), (k, e, s)
    o.close()
    q.close()
    sim.close()
