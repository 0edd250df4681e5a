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
