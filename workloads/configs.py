"""Seeded synthetic inputs for the five BASELINE.json configurations.

This module serves BOTH the fp64 oracle and the CUDA library and therefore holds none of the method's
arithmetic: it only lays out initial polylines, samples materials / scenes / action sequences from
`numpy.random.Generator(PCG64(seed))` with `seed = 20260604 + config_id`, and owns the loss heads of the
harness (the library itself takes dL/dx_T).  Everything is float64 numpy; the CUDA
binding casts to float32 on upload.  They stand in for the paper's task scenes (Table 3 / Table 11,
PAPER.md L412-428, L602-613), which are not available: same shapes (open ropes and one closed band, tens to
hundreds of vertices, frame = 5 substeps, hundreds to thousands of frames, posts / ground / gripper contact,
per-step end-effector pose actions).
"""
import numpy as np

SEED0 = 20260604
OPEN, RING = 0, 1
STRETCH_ENERGY, STRETCH_PROJECT = 0, 1
PRIM_PLANE, PRIM_CAPSULE, PRIM_CYLINDER, PRIM_BOX = 0, 1, 2, 3

DEFAULTS = dict(n_substeps=5, n_proj_iters=10, stretch_mode=STRETCH_PROJECT, enable_plasticity=0,
                enable_self_contact=0, self_skip=2, n_grippers=0, n_grasp_max=1, n_primitives=0,
                kappa_bar_from_x0=0, gravity=(0.0, 0.0, -9.81), rope_radius=2.5e-3, contact_softness=1e-3,
                influence_threshold=0.1, restitution=0.0, topology=OPEN)

FULL_SIZES = {1: dict(batch=1, n_verts=32, horizon=200, stride=50),
              2: dict(batch=1024, n_verts=64, horizon=300, stride=0),
              3: dict(batch=1024, n_verts=64, horizon=500, stride=50),
              4: dict(batch=2048, n_verts=96, horizon=400, stride=40),
              5: dict(batch=4096, n_verts=128, horizon=1000, stride=100)}


def _material(B, m=0.01, l0=None, stretch=0.0, alpha=1e-3, gamma=0.0, sigma_y=1e9, r_c=0.0, mu_r=0.5, mu_s=0.3):
    def arr(a):
        return np.broadcast_to(np.asarray(a, dtype=np.float64), (B,)).copy()
    return dict(mass_per_vertex=arr(m), rest_edge_len=arr(l0), stretch=arr(stretch), bend_stiffness=arr(alpha),
                damping=arr(gamma), yield_curv=arr(sigma_y), creep_rate=arr(r_c), mu_rigid=arr(mu_r), mu_self=arr(mu_s))


def _logu(rng, lo, hi, n):
    return np.exp(rng.uniform(np.log(lo), np.log(hi), n))


def _resample_polyline(pts, n):
    """n points at equal arclength along the polyline pts [M][3] (end points included)."""
    seg = np.linalg.norm(np.diff(pts, axis=0), axis=1)
    s = np.concatenate([[0.0], np.cumsum(seg)])
    si = np.linspace(0.0, s[-1], n)
    out = np.empty((n, 3))
    for k in range(3):
        out[:, k] = np.interp(si, s, pts[:, k])
    return out


CLEARANCE = 1.0e-4   # initial gap to a surface the rope is laid on / wrapped around
# Finger capsules stand FINGER_SLACK beyond touching distance on either side of the held rope: the vertices next to a grasped
# one move with the gripper, so against a finger that just touches them their approach speed u_n is zero to
# rounding for the whole rollout and the branch u_n < 0 - hence every action gradient - is decided by the last bit.  With
# 3 mm of slack (f = exp(-3) < the 0.1 threshold) the fingers act when the rope swings into them, not on what they carry.
FINGER_SLACK = 3.0e-3


def _slack_u(span, height, length, r, n):
    """Down-slope, flat stretch lying CLEARANCE above its rest height z=r, up-slope; total arclength `length`; ends `span`
    apart at `height`.  (Not at z=r exactly: phi = r is the kink of f = min(exp(d / eps_s), 1) of PAPER.md L103, where the
    derivative of the step jumps; a rope laid exactly there would make every gradient depend on the last bit of r - z.)"""
    r = r + CLEARANCE
    hh = height - r
    k = 0.5 * (length - span)                 # sqrt(d^2+hh^2) - d = k
    d = (hh * hh - k * k) / (2.0 * k)
    pts = np.array([[-0.5 * span, 0, height], [-0.5 * span + d, 0, r], [0.5 * span - d, 0, r], [0.5 * span, 0, height]])
    return _resample_polyline(pts, n)


def _smooth_random_actions(rng, H, B, G, max_trans, max_rot, box=25):
    """Cumulative sum of Gaussian increments, box-filtered, rescaled to the given total excursion. [H][B][G][6] offsets."""
    inc = rng.normal(0.0, 1.0, (H + box, B, G, 6))
    cs = np.cumsum(inc, axis=0)
    sm = (cs[box:] - cs[:-box]) / box                                   # box filter, [H][B][G][6]
    path = np.cumsum(sm, axis=0)
    tr = np.linalg.norm(path[..., :3], axis=-1).max(axis=0)          # [B][G]
    ro = np.linalg.norm(path[..., 3:], axis=-1).max(axis=0)
    scale_t = rng.uniform(0.5, 1.0, (B, G)) * max_trans / np.maximum(tr, 1e-12)
    scale_r = rng.uniform(0.5, 1.0, (B, G)) * max_rot / np.maximum(ro, 1e-12)
    path[..., :3] *= scale_t[None, :, :, None]
    path[..., 3:] *= scale_r[None, :, :, None]
    return path


def _smooth_target_polyline(rng, B, N, start, length):
    """Seeded smooth polyline of the given arclength starting at start[B][3] (loss target)."""
    l = length / (N - 1)
    out = np.zeros((B, 3, N))
    d = rng.normal(0, 1, (B, 3))
    d /= np.linalg.norm(d, axis=1, keepdims=True)
    p = np.array(start, dtype=np.float64)[:B].copy()
    for i in range(N):
        out[:, :, i] = p
        d = d + 0.15 * rng.normal(0, 1, (B, 3))
        d /= np.linalg.norm(d, axis=1, keepdims=True)
        p = p + l * d
    return out


def _base(cfg_id, batch, n_verts, horizon, stride):
    full = FULL_SIZES[cfg_id]
    B = full["batch"] if batch is None else batch
    N = full["n_verts"] if n_verts is None else n_verts
    H = full["horizon"] if horizon is None else horizon
    S = full["stride"] if stride is None else stride
    cfg = dict(DEFAULTS)
    cfg.update(batch=B, n_verts=N)
    return cfg, B, N, H, S


FLOAT_CONFIG_KEYS = ("dt", "rope_radius", "contact_softness", "influence_threshold", "restitution")
ARRAY_KEYS = ("x0", "v0", "kappa_bar0", "prim_params", "init_pose", "finger_geom", "actions")


def representable(P):
    """Rounds every real input of a problem dict to its nearest fp32 value (still stored as float64), so that the fp64
    oracle and the fp32 library read the SAME numbers.  The step has branches decided at exact thresholds (a vertex
    resting at phi = r sits on the kink of f = min(exp(d / eps_s), 1)): with r = 2.5e-3 given to one side as
    a double and to the other as its fp32 rounding, the two would take different sides of every such tie by construction."""
    f = lambda a: np.asarray(a, dtype=np.float32).astype(np.float64)
    P = dict(P)
    cfg = dict(P["config"])
    for k in FLOAT_CONFIG_KEYS:
        cfg[k] = float(np.float32(cfg[k]))
    cfg["gravity"] = tuple(float(np.float32(g)) for g in cfg["gravity"])
    P["config"] = cfg
    P["material"] = {k: f(v) for k, v in P["material"].items()}
    for k in ARRAY_KEYS:
        if P.get(k) is not None:
            P[k] = f(P[k])
    if P.get("loss") is not None:
        P["loss"] = dict(P["loss"], target=f(P["loss"]["target"]))
    return P


def make_problem(cfg_id, batch=None, n_verts=None, horizon=None, stride=None):
    """Problem dict for BASELINE.json config `cfg_id` (1..5); size overrides give the reduced parity cases.  Every real
    input is fp32-representable (see `representable`)."""
    return representable(_make_problem(cfg_id, batch, n_verts, horizon, stride))


def _make_problem(cfg_id, batch=None, n_verts=None, horizon=None, stride=None):
    rng = np.random.Generator(np.random.PCG64(SEED0 + cfg_id))
    cfg, B, N, H, S = _base(cfg_id, batch, n_verts, horizon, stride)
    P = dict(config=cfg, horizon=H, checkpoint_stride=S, config_id=cfg_id, pins=None, kappa_bar0=None, actions=None)

    if cfg_id == 1:
        l0 = 1.0 / (N - 1)
        cfg.update(dt=1e-3)
        P["material"] = _material(B, l0=l0, stretch=0.0, alpha=1e-3)
        x0 = np.zeros((B, 3, N))
        x0[:, 0, :] = np.arange(N) * l0
        x0[:, :, 1:] += rng.normal(0.0, 1e-3, (B, 3, N - 1))
        P["x0"], P["v0"] = x0, np.zeros((B, 3, N))
        pins = np.zeros((B, N), dtype=np.uint8)
        pins[:, 0] = 1
        P["pins"] = pins
        target = np.stack([rng.uniform(0.6, 0.9, B), rng.uniform(-0.1, 0.1, B), rng.uniform(-0.4, -0.1, B)], axis=1)
        P["loss"] = dict(kind="tip", target=target)
        P["grad_wrt"] = ("g_v0",)
        return P

    if cfg_id == 2:
        l0 = 1.0 / (N - 1)
        cfg.update(dt=1e-3, n_grippers=2, n_grasp_max=1, n_primitives=1)
        P["material"] = _material(B, l0=l0, stretch=_logu(rng, 1e-8, 1e-4, B), alpha=_logu(rng, 1e-5, 1e-2, B),
                                  gamma=rng.uniform(0, 0.1, B), mu_r=0.5)
        shape = _slack_u(0.5, 0.25, 1.0, cfg["rope_radius"], N)
        x0 = np.repeat(shape.T[None], B, axis=0)
        x0[:, 1, 1:-1] += rng.normal(0.0, 0.02 * l0, (B, N - 2))          # lateral noise breaks the planar symmetry
        P["x0"], P["v0"] = x0, np.zeros((B, 3, N))
        P["prim_types"] = np.array([PRIM_PLANE], dtype=np.int32)
        pp = np.zeros((B, 1, 10))
        pp[:, 0, 2] = 1.0                                                # n = +z, o = 0
        P["prim_params"] = pp
        gv = np.full((B, 2, 1), -1, dtype=np.int32)
        gv[:, 0, 0], gv[:, 1, 0] = 0, N - 1
        P["grasp_verts"] = gv
        pose0 = np.zeros((B, 2, 6))
        pose0[:, 0, :3], pose0[:, 1, :3] = x0[:, :, 0], x0[:, :, -1]
        P["init_pose"] = pose0
        fg = np.zeros((B, 2, 4))
        fg[..., 0], fg[..., 1], fg[..., 2] = 0.2, 0.04, 0.01           # wide-open fingers: far from the rope
        P["finger_geom"] = fg
        # p_g(t) = p_g(0) + sum_k A_k [sin(2 pi f_k t + phi_k) - sin(phi_k)],  sum ||A_k|| <= 0.2 m
        A = rng.normal(0, 1, (B, 2, 4, 3))
        A *= (rng.uniform(0.3, 1.0, (B, 2, 1, 1)) * 0.2 / np.linalg.norm(A, axis=-1).sum(axis=-1)[..., None, None])
        f = rng.uniform(0.5, 3.0, (B, 2, 4))
        ph = rng.uniform(0, 2 * np.pi, (B, 2, 4))
        tt = (np.arange(H) + 1)[:, None, None, None] * cfg["dt"]
        s = np.sin(2 * np.pi * f[None] * tt + ph[None]) - np.sin(ph[None])           # [H][B][2][4]
        act = np.zeros((H, B, 2, 6))
        act[..., :3] = pose0[None, :, :, :3] + np.einsum("hbgk,bgkc->hbgc", s, A)
        P["actions"] = act
        P["loss"] = dict(kind="polyline", target=_smooth_target_polyline(rng, B, N, x0[:, :, 0], 1.0))
        P["grad_wrt"] = ()
        return P

    if cfg_id == 3:
        l0 = 1.0 / (N - 1)
        r, rf = cfg["rope_radius"], 0.01
        cfg.update(dt=1e-3, n_grippers=1, n_grasp_max=2, enable_plasticity=1)
        P["material"] = _material(B, l0=l0, stretch=0.0, alpha=_logu(rng, 1e-4, 1e-2, B), gamma=rng.uniform(0, 0.1, B),
                                  sigma_y=rng.uniform(0.5, 5.0, B), r_c=rng.uniform(0.1, 1.0, B))
        x0 = np.zeros((B, 3, N))
        x0[:, 0, :] = (np.arange(N) - 0.5) * l0                           # gripper frame origin between vertices 0 and 1
        x0[:, 1:, 2:] += rng.normal(0.0, 1e-4, (B, 2, N - 2))
        P["x0"], P["v0"] = x0, np.zeros((B, 3, N))
        gv = np.zeros((B, 1, 2), dtype=np.int32)
        gv[:, 0, 1] = 1
        P["grasp_verts"] = gv
        pose0 = np.zeros((B, 1, 6))
        pose0[:, 0, 5] = 0.5 * np.pi                                      # fingers straddle the rope (local x -> world y)
        P["init_pose"] = pose0
        fg = np.zeros((B, 1, 4))
        fg[..., 0], fg[..., 1], fg[..., 2] = 2 * (rf + r + FINGER_SLACK), 0.04, rf
        P["finger_geom"] = fg
        P["actions"] = pose0[None] + _smooth_random_actions(rng, H, B, 1, 0.2, 1.0)
        P["loss"] = dict(kind="polyline", target=_smooth_target_polyline(rng, B, N, P["actions"][-1, :, 0, :3], 1.0))
        P["grad_wrt"] = ("g_actions",)
        return P

    if cfg_id == 4:
        R, r = 0.02, cfg["rope_radius"]
        circ = 0.6
        l0 = circ / N
        cfg.update(dt=1e-3, topology=RING, n_grippers=1, n_grasp_max=1, n_primitives=2, enable_self_contact=1)
        P["material"] = _material(B, l0=l0, stretch=1e-5, alpha=1e-3, gamma=rng.uniform(0, 0.1, B), mu_r=0.5, mu_s=0.3)
        D = rng.uniform(0.24, 0.27, B)
        c1 = np.stack([-0.5 * D + rng.uniform(-5e-3, 5e-3, B), rng.uniform(-5e-3, 5e-3, B)], axis=1)
        c2 = np.stack([+0.5 * D + rng.uniform(-5e-3, 5e-3, B), rng.uniform(-5e-3, 5e-3, B)], axis=1)
        z0, rho = 0.1, R + r + CLEARANCE          # wrapped CLEARANCE off the posts (see _slack_u)
        x0 = np.zeros((B, 3, N))
        grasp = np.zeros(B, dtype=np.int64)
        for b in range(B):
            u = (c2[b] - c1[b]) / np.linalg.norm(c2[b] - c1[b])
            n = np.array([-u[1], u[0]])                                   # +y side
            ang = np.linspace(0, np.pi, 33)
            arc2 = [c2[b] + rho * (np.cos(a) * n + np.sin(a) * u) for a in ang]          # +n -> -n around post 2
            arc1 = [c1[b] + rho * (-np.cos(a) * n - np.sin(a) * u) for a in ang]         # -n -> +n around post 1
            loop = np.array([c1[b] + rho * n] + arc2 + arc1)
            loop = np.concatenate([loop, np.full((len(loop), 1), z0)], axis=1)
            x0[b] = _resample_polyline(loop, N + 1)[:N].T                 # closed: drop the repeated end point
            mid = 0.5 * (c1[b] + c2[b]) + rho * n
            grasp[b] = np.argmin(np.linalg.norm(x0[b, :2].T - mid, axis=1))
        x0[:, 2, :] += rng.normal(0.0, 2e-4, (B, N))
        P["x0"], P["v0"] = x0, np.zeros((B, 3, N))
        P["prim_types"] = np.array([PRIM_CYLINDER, PRIM_CYLINDER], dtype=np.int32)
        pp = np.zeros((B, 2, 10))
        for k, c in enumerate((c1, c2)):
            pp[:, k, 0:2], pp[:, k, 2] = c, z0
            pp[:, k, 5], pp[:, k, 6], pp[:, k, 7] = 1.0, R, 0.1
        P["prim_params"] = pp
        P["grasp_verts"] = grasp.astype(np.int32).reshape(B, 1, 1)
        pose0 = np.zeros((B, 1, 6))
        pose0[:, 0, :3] = x0[np.arange(B), :, grasp]
        pose0[:, 0, 5] = 0.5 * np.pi
        P["init_pose"] = pose0
        fg = np.zeros((B, 1, 4))
        fg[..., 0], fg[..., 1], fg[..., 2] = 2 * (0.01 + r + FINGER_SLACK), 0.04, 0.01
        P["finger_geom"] = fg
        dy, dz = rng.uniform(-0.09, -0.06, B), rng.uniform(0.0, 0.03, B)
        s = (np.arange(H) + 1) / H
        s = s * s * (3 - 2 * s)                                           # smooth-step in time
        act = np.repeat(pose0[None], H, axis=0)
        act[:, :, 0, 1] += s[:, None] * dy[None]
        act[:, :, 0, 2] += s[:, None] * dz[None]
        P["actions"] = act
        th = np.linspace(0, 2 * np.pi, N, endpoint=False)
        rad = circ / (2 * np.pi)
        tgt = np.zeros((B, 3, N))
        cx, cy = rng.uniform(-0.03, 0.03, B), rng.uniform(-0.03, 0.03, B)
        ecc = rng.uniform(0.8, 1.25, B)
        tgt[:, 0] = cx[:, None] + rad * ecc[:, None] * np.cos(th)[None]
        tgt[:, 1] = cy[:, None] + rad / ecc[:, None] * np.sin(th)[None]
        tgt[:, 2] = z0
        P["loss"] = dict(kind="polyline", target=tgt)
        P["grad_wrt"] = ("g_actions", "g_x0", "g_v0")
        return P

    if cfg_id == 5:
        l0 = 1.0 / (N - 1)
        r, rf = cfg["rope_radius"], 0.01
        cfg.update(dt=5e-4, n_grippers=2, n_grasp_max=2, n_primitives=4, enable_plasticity=1, enable_self_contact=1)
        P["material"] = _material(B, l0=l0, stretch=_logu(rng, 1e-8, 1e-4, B), alpha=_logu(rng, 1e-5, 1e-2, B),
                                  gamma=rng.uniform(0, 0.1, B), sigma_y=rng.uniform(0.5, 5.0, B), r_c=rng.uniform(0.1, 1.0, B),
                                  mu_r=0.5, mu_s=0.3)
        shape = _slack_u(0.6, 0.2, 1.0, r, N)
        x0 = np.repeat(shape.T[None], B, axis=0)
        x0[:, 1, 2:-2] += rng.normal(0.0, 0.02 * l0, (B, N - 4))
        P["x0"], P["v0"] = x0, np.zeros((B, 3, N))
        types = np.array([PRIM_PLANE, PRIM_BOX, PRIM_CYLINDER, PRIM_BOX], dtype=np.int32)
        P["prim_types"] = types
        pp = np.zeros((B, 4, 10))
        pp[:, 0, 2] = 1.0
        for k in (1, 2, 3):
            foot = rng.uniform(0.02, 0.06, (B, 2))
            hgt = rng.uniform(0.05, 0.15, B)
            cx = rng.uniform(-0.3, 0.3, B)
            side = np.where(rng.uniform(0, 1, B) < 0.5, -1.0, 1.0)
            cy = side * rng.uniform(0.5 * foot.max(axis=1) + 0.015, 0.3, B)   # beside the initial rope line, inside the patch
            if types[k] == PRIM_BOX:
                pp[:, k, 0], pp[:, k, 1], pp[:, k, 2] = cx, cy, 0.5 * hgt
                pp[:, k, 3], pp[:, k, 4], pp[:, k, 5] = 0.5 * foot[:, 0], 0.5 * foot[:, 1], 0.5 * hgt
                pp[:, k, 8] = rng.uniform(-np.pi / 4, np.pi / 4, B)          # yaw
            else:
                pp[:, k, 0], pp[:, k, 1], pp[:, k, 2] = cx, cy, 0.5 * hgt
                pp[:, k, 5], pp[:, k, 6], pp[:, k, 7] = 1.0, 0.5 * foot[:, 0], 0.5 * hgt
        P["prim_params"] = pp
        gv = np.zeros((B, 2, 2), dtype=np.int32)
        gv[:, 0], gv[:, 1] = (0, 1), (N - 2, N - 1)
        P["grasp_verts"] = gv
        pose0 = np.zeros((B, 2, 6))
        pose0[:, 0, :3] = 0.5 * (x0[:, :, 0] + x0[:, :, 1])
        pose0[:, 1, :3] = 0.5 * (x0[:, :, -2] + x0[:, :, -1])
        P["init_pose"] = pose0
        fg = np.zeros((B, 2, 4))
        fg[..., 0], fg[..., 1], fg[..., 2] = 2 * (rf + r + FINGER_SLACK), 0.04, rf
        P["finger_geom"] = fg
        P["actions"] = pose0[None] + _smooth_random_actions(rng, H, B, 2, 0.2, 1.0)
        P["loss"] = dict(kind="polyline", target=_smooth_target_polyline(rng, B, N, P["actions"][-1, :, 0, :3], 1.0))
        P["grad_wrt"] = ("g_actions", "g_material")
        return P

    raise ValueError("config id must be 1..5")


def rest_length(problem):
    """L_rest used to normalise position errors (rope length / ring circumference), per env."""
    cfg = problem["config"]
    E = cfg["n_verts"] if cfg["topology"] == RING else cfg["n_verts"] - 1
    return problem["material"]["rest_edge_len"] * E


def loss_and_seed(problem, xT):
    """Harness-owned loss head: returns (L [B], dL/dx_T [B][3][N]) for final positions xT [B][3][N] (float64)."""
    spec = problem["loss"]
    xT = np.asarray(xT, dtype=np.float64)
    B, _, N = xT.shape
    g = np.zeros_like(xT)
    if spec["kind"] == "tip":                      # || x_{N-1}(T) - p* ||^2
        d = xT[:, :, -1] - spec["target"][:B]
        g[:, :, -1] = 2.0 * d
        return (d * d).sum(axis=1), g
    if spec["kind"] == "polyline":                 # mean_i || x_i(T) - q_i ||^2
        d = xT - spec["target"][:B]
        return (d * d).sum(axis=(1, 2)) / N, 2.0 * d / N
    raise ValueError(spec["kind"])


def subset(problem, envs):
    """Problem restricted to the given env indices (envs are independent, so a subset is sound)."""
    envs = np.asarray(envs, dtype=np.int64)
    Q = dict(problem)
    Q["config"] = dict(problem["config"], batch=len(envs))
    Q["material"] = {k: v[envs] for k, v in problem["material"].items()}
    for k in ("pins", "cuts", "prim_params", "init_pose", "finger_geom", "grasp_verts", "x0", "v0", "kappa_bar0"):
        if problem.get(k) is not None:
            Q[k] = problem[k][envs]
    if problem.get("actions") is not None:
        Q["actions"] = problem["actions"][:, envs]
    Q["loss"] = dict(problem["loss"], target=problem["loss"]["target"][envs])
    return Q
