"""-m gpu: the five BASELINE.json configs at their FULL sizes, in the launch configuration bench.py times (whole batch, full
horizon, the config's checkpoint stride), checked on sampled envs the oracle computes one by one (envs are independent,
so a sample is sound).  Criteria as in test_parity_gpu.py / test_gradient_gpu.py: plain tolerance, or no further from the
oracle than 5x the oracle's own spread under fp32-sized input perturbations for chaotic / kinked envs."""
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


def spread_ok(err, spread, tol):
    ok = (err <= tol) | (err <= 5.0 * spread)
    return (~ok).sum() <= max(1, len(err) // 4) and np.median(err) <= max(tol, 3.0 * np.median(spread))


@pytest.mark.parametrize("cfg_id,n_sample,with_grad", [(2, 16, False), (3, 8, True), (4, 4, True), (5, 4, True)])
def test_full_size_config(dlo, orc, cfg_id, n_sample, with_grad):
    P = make_problem(cfg_id)
    B, H, stride = P["config"]["batch"], P["horizon"], P["checkpoint_stride"]
    envs = np.arange(0, B, B // n_sample)[:n_sample]
    sim = dlo.DloSim(P)
    sim.rollout(H, stride)
    got = sim.state()
    assert sim.n_bad() == 0
    assert np.isfinite(got["x"]).all()
    # oracle on the sampled envs (+ its conditioning under fp32-sized input perturbations)
    Q = subset(P, envs)
    o = orc.OracleSim(Q)
    ref = o.rollout(H, stride)
    rng = np.random.default_rng(5)
    q = orc.OracleSim(perturbed(Q, rng))
    ref_p = q.rollout(H, stride)
    err = position_error(Q, got["x"][envs], ref["x"])
    spread = position_error(Q, ref_p["x"], ref["x"])
    print(summarize("cfg%d full size: positions gpu" % cfg_id, err), "|", summarize("oracle spread", spread))
    assert spread_ok(err, spread, POS_TOL), (err, spread)
    if with_grad:
        _, seed = loss_and_seed(Q, ref["x"])
        g_ref, g_prt = o.backward(seed), q.backward(seed)
        full_seed = np.zeros((B,) + seed.shape[1:])
        full_seed[envs] = seed
        g = sim.backward(full_seed)
        for k in P["grad_wrt"]:
            a = env_first(k, g[k])[envs]
            e = gradient_error(a, env_first(k, g_ref[k]))
            s = gradient_error(env_first(k, g_prt[k]), env_first(k, g_ref[k]))
            print(summarize("cfg%d full size: %s gpu" % (cfg_id, k), e), "|", summarize("oracle spread", s))
            assert np.isfinite(a).all()
            # Over the full horizon the reverse recursion amplifies every rounding: the oracle's own
            # gradient moves by `s` under ONE fp32-sized perturbation of its inputs, while an fp32 run injects one such
            # perturbation per substep; independent injections add in quadrature, hence sqrt(H * n_sub) * s.  The plain
            # 1e-3 bar is asserted on the well-conditioned cases of test_gradient_gpu.py.
            n_inj = np.sqrt(H * P["config"]["n_substeps"])
            assert np.median(e) <= max(GRAD_TOL, n_inj * np.median(s)), (k, e, s)
    o.close()
    q.close()
    sim.close()
