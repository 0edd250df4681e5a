"""Test-side helpers: build small problem dicts for the oracle pins (no method arithmetic, just inputs)."""
import numpy as np

from workloads.configs import DEFAULTS, _material


def rope_problem(x0, v0=None, *, ring=False, dt=1e-3, horizon=10, stride=0, material=None, pins=None, cuts=None, **cfg_over):
    """Problem dict for a batch of ropes given as x0 [B][N][3] (AoS for convenience).  cuts: vertex indices j whose edge
    (j, j+1) does not exist (several ropes back to back in one env)."""
    x0 = np.asarray(x0, dtype=np.float64)
    if x0.ndim == 2:
        x0 = x0[None]
    B, N, _ = x0.shape
    cfg = dict(DEFAULTS)
    cfg.update(batch=B, n_verts=N, dt=dt, topology=1 if ring else 0)
    cfg.update(cfg_over)
    E = N if ring else N - 1
    keep = np.ones(E, dtype=bool)
    if cuts is not None:
        keep[list(cuts)] = False
    mat = dict(l0=np.linalg.norm(np.roll(x0, -1, axis=1) - x0, axis=2)[:, :E][:, keep].mean(axis=1))
    mat.update(material or {})
    P = dict(config=cfg, horizon=horizon, checkpoint_stride=stride, pins=None, kappa_bar0=None, actions=None)
    P["material"] = _material(B, **mat)
    P["x0"] = np.ascontiguousarray(x0.transpose(0, 2, 1))
    P["v0"] = np.zeros((B, 3, N)) if v0 is None else np.ascontiguousarray(np.asarray(v0, float).reshape(B, N, 3).transpose(0, 2, 1))
    if pins is not None:
        p = np.zeros((B, N), dtype=np.uint8)
        p[:, list(pins)] = 1
        P["pins"] = p
    if cuts is not None:
        c = np.zeros((B, N), dtype=np.uint8)
        c[:, list(cuts)] = 1
        P["cuts"] = c
    return P


def aos(a):
    """[B][3][N] -> [B][N][3]"""
    return np.asarray(a).transpose(0, 2, 1)


def figure_eight_problem(N=32, gap=0.0062, B=2, horizon=30, stride=7, seed=0):
    """An open rope laid as a figure eight whose two strands cross once, `gap` apart vertically, and move towards each
    other slowly: one gentle self-contact (Eq.13) with sliding friction, no gravity.  Used to check the self-contact
    path and its adjoint on a well-conditioned case."""
    from workloads.configs import _resample_polyline
    rng = np.random.default_rng(seed)
    t = np.linspace(-0.3 * np.pi, 1.3 * np.pi, 2000)
    curve = np.stack([0.04 * np.sin(2 * t), 0.04 * np.sin(t), 0.5 * gap * np.cos(t)], 1)
    pts = _resample_polyline(curve, N)
    x = pts[None].repeat(B, 0) + rng.normal(0, 5e-5, (B, N, 3))
    v = np.zeros_like(x)
    v[..., 2] = -15.0 * x[..., 2]
    v[..., 0] = 0.05 * np.sign(x[..., 2])
    l0 = np.linalg.norm(np.diff(pts, axis=0), axis=1).mean()
    P = rope_problem(x, v, dt=1e-3, horizon=horizon, stride=stride, enable_self_contact=1, gravity=(0.0, 0.0, 0.0),
                     material=dict(stretch=1e-6, alpha=2e-4, gamma=0.05, mu_s=0.4, l0=l0))
    P["loss"] = dict(kind="polyline", target=np.zeros((B, 3, N)))
    P["grad_wrt"] = ()
    return P
