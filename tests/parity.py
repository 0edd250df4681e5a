"""Shared pieces of the GPU-vs-oracle parity tests: metrics of SURVEY.md section 8(d) and small problem variants."""
import numpy as np

from workloads.configs import make_problem, rest_length, subset, loss_and_seed  # noqa: F401

POS_TOL = 1e-4     # BASELINE.json north_star: vertex positions within 1e-4 relative (to the rope length)
GRAD_TOL = 1e-3    # gradients within 1e-3 relative (norm-wise per env and gradient tensor)


def position_error(problem, x_gpu, x_orc):
    """max_i ||x_i^gpu - x_i^orc||_2 / L_rest per env"""
    d = np.linalg.norm(np.asarray(x_gpu, float) - np.asarray(x_orc, float), axis=1).max(axis=1)
    return d / rest_length(problem)[: len(d)]


def gradient_error(g_gpu, g_orc):
    """||g^gpu - g^orc||_2 / ||g^orc||_2 per env; g shaped [B, ...] (env axis first)"""
    B = g_orc.shape[0]
    a, b = np.asarray(g_gpu, float).reshape(B, -1), np.asarray(g_orc, float).reshape(B, -1)
    return np.linalg.norm(a - b, axis=1) / np.maximum(np.linalg.norm(b, axis=1), 1e-300)


def summarize(name, err):
    return "%s: max %.3e  p99 %.3e  median %.3e  (n=%d)" % (name, err.max(), np.quantile(err, 0.99), np.median(err), len(err))


def perturbed(P, rng, eps=2.0 ** -24):
    """the same problem with every real input moved by one fp32 rounding (relative 2^-24, Gaussian)"""
    Q = dict(P)
    for k in ("x0", "actions", "init_pose"):
        if P.get(k) is not None:
            Q[k] = P[k] * (1.0 + eps * rng.standard_normal(P[k].shape))
    Q["material"] = {k: v * (1.0 + eps * rng.standard_normal(v.shape)) for k, v in P["material"].items()}
    return Q


def oracle_position_spread(orc, P, H, ref_x, draws=2, seed=11):
    """per-env response of the ORACLE's final positions to fp32-sized input perturbations (its conditioning):
    max over `draws` perturbed fp64 runs of the position error against the unperturbed run"""
    rng = np.random.default_rng(seed)
    spread = 0.0
    for _ in range(draws):
        q = orc.OracleSim(perturbed(P, rng))
        spread = np.maximum(spread, position_error(P, q.rollout(H, 0)["x"], ref_x))
        q.close()
    return spread
