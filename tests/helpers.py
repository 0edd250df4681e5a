"""Test-side helpers: build small problem dicts for the oracle pins (no method arithmetic, just inputs)."""
import numpy as np

from workloads.configs import DEFAULTS, _material


def rope_problem(x0, v0=None, *, ring=False, dt=1e-3, horizon=10, stride=0, material=None, pins=None, **cfg_over):
    """Problem dict for a batch of ropes given as x0 [B][N][3] (AoS for convenience)."""
    x0 = np.asarray(x0, dtype=np.float64)
    if x0.ndim == 2:
        x0 = x0[None]
    B, N, _ = x0.shape
    cfg = dict(DEFAULTS)
    cfg.update(batch=B, n_verts=N, dt=dt, topology=1 if ring else 0)
    cfg.update(cfg_over)
    E = N if ring else N - 1
    mat = dict(l0=np.linalg.norm(np.roll(x0, -1, axis=1) - x0, axis=2)[:, :E].mean(axis=1))
    mat.update(material or {})
    P = dict(config=cfg, horizon=horizon, checkpoint_stride=stride, pins=None, kappa_bar0=None, actions=None)
    P["material"] = _material(B, **mat)
    P["x0"] = np.ascontiguousarray(x0.transpose(0, 2, 1))
    P["v0"] = np.zeros((B, 3, N)) if v0 is None else np.ascontiguousarray(np.asarray(v0, float).reshape(B, N, 3).transpose(0, 2, 1))
    if pins is not None:
        p = np.zeros((B, N), dtype=np.uint8)
        p[:, list(pins)] = 1
        P["pins"] = p
    return P


def aos(a):
    """[B][3][N] -> [B][N][3]"""
    return np.asarray(a).transpose(0, 2, 1)
