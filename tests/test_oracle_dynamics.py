"""Pins of the oracle's time stepping against closed forms and invariants."""
import numpy as np
import pytest
from numpy.polynomial import laguerre

from helpers import aos, rope_problem
from workloads import make_problem

G = 9.81


def straight(n, l, axis=0, origin=(0, 0, 0)):
    x = np.zeros((n, 3))
    x[:, axis] = np.arange(n) * l
    return x + np.asarray(origin, float)


FREE = dict(stretch_mode=0, material=dict(stretch=0.0, alpha=0.0))       # no internal forces at all: free particles


# --- C-5: symplectic Euler on free fall is exact ---------------------------------------------------------
def test_free_fall_closed_form(orc):
    x0 = straight(4, 0.1, origin=(0, 0, 5.0))
    v0 = np.tile([0.3, -0.2, 1.0], (4, 1))
    H, nsub, dt = 40, 5, 1e-3
    P = rope_problem(x0, v0, dt=dt, horizon=H, n_substeps=nsub, **FREE)
    st = orc.OracleSim(P).rollout()
    n, h = H * nsub, dt / nsub
    g = np.array([0, 0, -G])
    xe = x0 + n * h * v0 + 0.5 * g * h * h * n * (n + 1)
    assert np.abs(aos(st["x"])[0] - xe).max() < 1e-13
    assert np.abs(aos(st["v"])[0] - (v0 + n * h * g)).max() < 1e-13


def test_damped_fall_recurrence_and_terminal_velocity(orc):
    gamma, dt = 4.0, 1e-3
    x0 = straight(3, 0.1, origin=(0, 0, 50.0))
    P = rope_problem(x0, dt=dt, horizon=50, n_substeps=1, stretch_mode=0, material=dict(stretch=0.0, alpha=0.0, gamma=gamma))
    st = orc.OracleSim(P).rollout()
    v = 0.0
    for _ in range(50):
        v = (v - dt * G) / (1 + gamma * dt)              # implicit viscous damping (reading B-7)
    assert abs(st["v"][0, 2, 1] - v) < 1e-14
    P["horizon"] = 6000
    st = orc.OracleSim(P).rollout()
    assert abs(st["v"][0, 2, 1] + G / gamma) < 1e-8      # terminal velocity g / gamma


# --- C-6: energy behaviour of symplectic Euler (mode 0, no damping) ------------------------------------------
def total_energy(orc, P, st, ks, alpha, l0, m):
    x, v = aos(st["x"])[0], aos(st["v"])[0]
    E = len(x) - 1
    d1 = aos(st["d1"])[0][:E]
    kb = aos(st["kappa_bar"])[0]
    return (0.5 * m * (v * v).sum() + m * G * x[:, 2].sum() + orc.stretch_energy(x, ks, l0)
            + orc.bend_energy(x, d1, kb, alpha, l0))


def test_energy_oscillation_scales_with_h_no_drift(orc):
    rng = np.random.default_rng(3)
    N, l0, m, alpha, ks = 16, 1.0 / 15, 0.01, 1e-3, (1.0 / 15) / 1e-4
    x0 = straight(N, l0) + rng.normal(0, 1e-3, (N, 3))
    x0[0] = 0
    dev = {}
    for h in (2e-4, 1e-4):
        P = rope_problem(x0, dt=h, horizon=int(0.4 / h), n_substeps=1, stretch_mode=0, pins=[0],
                         material=dict(l0=l0, stretch=ks, alpha=alpha, m=m))
        sim = orc.OracleSim(P)
        sim.rollout(record=True)
        Es = np.array([total_energy(orc, P, sim.record(t), ks, alpha, l0, m) for t in range(0, P["horizon"] + 1, 5)])
        scale = m * G * N * 0.5
        dev[h] = np.abs(Es - Es[0]).max() / scale
        half = len(Es) // 2
        assert abs(Es[half:].mean() - Es[:half].mean()) / scale < 0.5 * dev[h] + 1e-9     # no secular trend
    assert 1.6 < dev[2e-4] / dev[1e-4] < 2.4                                               # error is O(h)


# --- C-7: rest-state stationarity ----------------------------------------------------------------------------
def test_rest_state_stationary_open_curved(orc):
    rng = np.random.default_rng(4)
    l = 0.04
    x = np.zeros((14, 3))
    d = np.array([1.0, 0, 0])
    for i in range(1, 14):
        d = d + 0.5 * rng.normal(size=3)
        d /= np.linalg.norm(d)
        x[i] = x[i - 1] + l * d
    P = rope_problem(x, horizon=100, gravity=(0, 0, 0), kappa_bar_from_x0=1, material=dict(l0=l, alpha=5e-3))
    st = orc.OracleSim(P).rollout()
    assert np.abs(aos(st["x"])[0] - x).max() < 1e-13


@pytest.mark.parametrize("planar", [True, False])
def test_rest_state_stationary_ring(orc, planar):
    N = 20
    th = np.linspace(0, 2 * np.pi, N, endpoint=False)
    z = np.zeros(N) if planar else 0.03 * (-1.0) ** np.arange(N)          # "crown": non-planar, all edges equal
    x = np.stack([0.1 * np.cos(th), 0.1 * np.sin(th), z], 1)
    l = np.linalg.norm(x[1] - x[0])
    P = rope_problem(x, ring=True, horizon=100, gravity=(0, 0, 0), kappa_bar_from_x0=1, material=dict(l0=l, alpha=5e-3))
    st = orc.OracleSim(P).rollout()
    assert np.abs(aos(st["x"])[0] - x).max() < 1e-13
    # a random non-planar closed curve with unequal edges is stationary too once stretching is switched off
    rng = np.random.default_rng(5)
    y = x + 0.01 * rng.normal(size=x.shape)
    P = rope_problem(y, ring=True, horizon=100, gravity=(0, 0, 0), kappa_bar_from_x0=1, stretch_mode=0,
                     material=dict(stretch=0.0, alpha=5e-3))
    st = orc.OracleSim(P).rollout()
    assert np.abs(aos(st["x"])[0] - y).max() < 1e-13


# --- C-8: length preservation on config 1 -----------------------------------------------------------------------
def test_length_preservation_config1(orc):
    strains = []
    for NC in (5, 10, 20, 40):
        P = make_problem(1)
        P["config"]["n_proj_iters"] = NC
        sim = orc.OracleSim(P)
        sim.rollout(record=True)
        worst = 0.0
        for t in range(20, 201, 20):                   # after the initial perturbation has been projected out
            x = aos(sim.record(t)["x"])[0]
            L = np.linalg.norm(np.diff(x, axis=0), axis=1)
            worst = max(worst, np.abs(L * 31 - 1).max())
        strains.append(worst)
    assert strains[1] <= 1e-2                           # N_C = 10
    assert all(a > b for a, b in zip(strains, strains[1:]))   # monotone in N_C


# --- C-9: N-link small-angle pendulum vs Laguerre roots --------------------------------------------------------------
@pytest.mark.parametrize("links,mode", [(2, 0), (3, 0), (3, 1)])
def test_chain_pendulum_frequency(orc, links, mode):
    l, amp, h = 0.1, 1e-3, 1e-4
    n = links
    # stiffness matrix of the linearised hanging chain (tension in link k = (n-k) m g), built independently here
    T = np.arange(n, 0, -1.0)
    A = np.zeros((n, n))
    for k in range(n):
        A[k, k] += T[k]
        if k > 0:
            A[k, k - 1] -= T[k]
        if k < n - 1:
            A[k, k] += T[k + 1]
            A[k, k + 1] -= T[k + 1]
    w2, V = np.linalg.eigh(A)
    xi = np.sort(laguerre.lagroots([0] * n + [1]))
    assert np.allclose(w2, xi, rtol=1e-10)              # omega_k^2 = (g/l) xi_k, xi_k roots of L_n
    shape = V[:, mode] / np.abs(V[:, mode]).max()
    omega = np.sqrt(G / l * xi[mode])
    x = np.zeros((n + 1, 3))
    for k in range(1, n + 1):
        dx = amp * (shape[k - 1] - (shape[k - 2] if k > 1 else 0.0))
        x[k] = x[k - 1] + [dx, 0, -np.sqrt(l * l - dx * dx)]
    periods = 3.25
    H = int(periods * 2 * np.pi / omega / h)
    P = rope_problem(x, dt=h, horizon=H, n_substeps=1, n_proj_iters=20, pins=[0], material=dict(l0=l, alpha=0.0))
    sim = orc.OracleSim(P)
    sim.rollout(record=True)
    tip = np.array([sim.record(t)["x"][0, 0, n] for t in range(H + 1)])
    zc = np.where((tip[:-1] > 0) & (tip[1:] <= 0))[0]
    tz = [(i + tip[i] / (tip[i] - tip[i + 1])) * h for i in zc]
    assert len(tz) >= 3
    period = (tz[-1] - tz[0]) / (len(tz) - 1)
    assert abs(period * omega / (2 * np.pi) - 1) < 2e-4


# --- C-10: discrete catenary ---------------------------------------------------------------------------------------
def test_discrete_catenary(orc):
    N, span, m = 21, 0.7, 0.01
    l = 1.0 / (N - 1)
    x = np.zeros((N, 3))
    half = (N - 1) // 2
    for k in range(1, N):
        dx = span / (N - 1)
        x[k] = x[k - 1] + [dx, 0, np.sqrt(l * l - dx * dx) * (-1 if k <= half else 1)]
    P = rope_problem(x, dt=2e-4, horizon=60000, n_substeps=1, n_proj_iters=30, pins=[0, N - 1],
                     material=dict(l0=l, alpha=0.0, gamma=20.0, m=m))
    st = orc.OracleSim(P).rollout()
    assert np.abs(st["v"]).max() < 1e-6
    Ne = N - 1
    jj = np.arange(Ne) - (Ne - 1) / 2
    f = lambda Hh: np.sum(l / np.sqrt(1 + (m * G * jj / Hh) ** 2)) - span      # horizontal tension from the span
    lo, hi = 1e-6, 1e3
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        lo, hi = (lo, mid) if f(mid) > 0 else (mid, hi)
    th = np.arctan(m * G * jj / (0.5 * (lo + hi)))
    xz = np.zeros((N, 2))
    for k in range(1, N):
        xz[k] = xz[k - 1] + l * np.array([np.cos(th[k - 1]), np.sin(th[k - 1])])
    assert np.abs(aos(st["x"])[0][:, [0, 2]] - xz).max() < 1e-4


# --- C-4: discrete cantilever ------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N", [11, 21])
def test_cantilever_tip_deflection(orc, N):
    alpha, rho, g, L = 1e-2, 0.02, 0.02, 1.0
    l = L / (N - 1)
    m = rho * l
    P = rope_problem(straight(N, l), dt=2e-4, horizon=50000, n_substeps=1, n_proj_iters=20, pins=[0, 1],
                     gravity=(0, 0, -g), material=dict(l0=l, alpha=alpha, gamma=5.0, m=m))
    st = orc.OracleSim(P).rollout()
    assert np.abs(st["v"]).max() < 1e-9
    nn = np.arange(1, N - 1)
    delta = m * g * l ** 3 / alpha * np.sum(nn ** 2 * (nn + 1) / 2.0)     # chain of hinges of compliance l/alpha
    assert abs(-st["x"][0, 2, -1] / delta - 1) < 1e-4
    assert abs(delta / (rho * g * L ** 4 / (8 * alpha)) - 1) < 0.3          # -> w L^4 / (8 alpha) as N grows


# --- C-11: momentum conservation through self-contact + friction (Fig. 12) ------------------------------------------
def hairpin(n_arm, l, gap):
    """two parallel arms `gap` apart joined by a semicircular turn, all edges ~ l"""
    R = gap / 2
    n_turn = max(3, int(round(np.pi * R / l)))
    pts = [[-i * l, R, 0] for i in range(n_arm, 0, -1)]
    pts += [[R * np.sin(a), R * np.cos(a), 0] for a in np.linspace(0, np.pi, n_turn + 1)]
    pts += [[-i * l, -R, 0] for i in range(1, n_arm + 1)]
    return np.array(pts, float)


def test_momentum_conserved_through_self_contact(orc):
    l, gap, m = 0.01, 0.03, 0.01
    x = hairpin(14, l, gap)
    N = len(x)
    v = np.zeros((N, 3))
    v[:14, 1], v[-14:, 1] = -0.6, 0.6                 # arms approach each other
    v[:14, 0], v[-14:, 0] = 0.3, -0.3                 # ... and slide along each other (friction engages)
    v[:, 2] = 0.05 * np.sin(np.arange(N))
    common = dict(dt=1e-3, horizon=60, gravity=(0, 0, 0), material=dict(l0=l, alpha=1e-4, m=m, mu_s=0.3, stretch=1e-6))
    res = {}
    for sc in (0, 1):
        P = rope_problem(x, v, enable_self_contact=sc, **common)
        sim = orc.OracleSim(P)
        sim.rollout(record=True)
        p0 = m * aos(sim.record(0)["v"])[0].sum(axis=0)
        err, mind = 0.0, 1e9
        for t in range(1, 61):
            r = sim.record(t)
            err = max(err, np.abs(m * aos(r["v"])[0].sum(axis=0) - p0).max())
            xs = aos(r["x"])[0]
            mind = min(mind, np.linalg.norm(xs[:10, None, :] - xs[None, -10:, :], axis=2).min())
        res[sc] = (err / np.abs(p0).max() if np.abs(p0).max() > 0 else err, mind, err)
    assert res[1][2] < 1e-12 * m * 0.6 * N + 1e-15    # paper: 1e-13..1e-14
    assert res[0][1] < 0.003                          # without self-contact the arms pass through each other
    assert res[1][1] > 0.004                          # with Eq.13 they stay about one thickness (5 mm) apart


# --- C-12: rigid coupling closed forms ----------------------------------------------------------------------------------
def plane_problem(x0, v0, horizon, mu=0.5, e=0.0, g=(0, 0, -G), **kw):
    P = rope_problem(x0, v0, dt=1e-3, horizon=horizon, n_primitives=1, restitution=e, gravity=g,
                     stretch_mode=0, material=dict(stretch=0.0, alpha=0.0, mu_r=mu), **kw)
    P["prim_types"] = np.array([0], dtype=np.int32)
    pp = np.zeros((1, 1, 10))
    pp[0, 0, 2] = 1.0
    P["prim_params"] = pp
    return P


def test_particle_rebound_and_rest_height(orc):
    r = 2.5e-3
    x0 = straight(3, 0.1, origin=(0, 0, r))
    v0 = np.tile([0, 0, -1.0], (3, 1))
    st = orc.OracleSim(plane_problem(x0, v0, 1, e=0.4, g=(0, 0, 0), n_substeps=1)).rollout()
    assert np.allclose(st["v"][0, 2], 0.4)                       # rebound e |v_n| at f = 1
    st = orc.OracleSim(plane_problem(x0, np.zeros((3, 3)), 300)).rollout()
    assert np.abs(st["x"][0, 2] - r).max() < 1e-12               # rests at z = r under gravity
    assert np.abs(st["v"][0]).max() < 1e-12


def test_particle_sliding_friction_stop(orc):
    r, mu, v0 = 2.5e-3, 0.5, 1.0
    x0 = straight(3, 0.1, axis=1, origin=(0, 0, r))
    v = np.tile([v0, 0, 0], (3, 1))
    P = plane_problem(x0, v, 400, mu=mu)
    sim = orc.OracleSim(P)
    sim.rollout(record=True)
    vx = np.array([sim.record(t)["v"][0, 0, 1] for t in range(401)])
    t_stop = np.argmax(vx <= 1e-12) * 1e-3
    assert abs(t_stop - v0 / (mu * G)) < 2e-3                    # v0 / (mu g) = 0.2039 s
    assert abs(sim.record(400)["x"][0, 0, 1] - v0 ** 2 / (2 * mu * G)) < 2e-4     # v0^2 / (2 mu g) = 0.1019 m
    assert np.abs(sim.record(400)["v"]).max() < 1e-12


def test_taut_ring_stays_on_posts(orc):
    P = make_problem(4, batch=4, horizon=200)
    P["config"]["n_grippers"] = 0                                # band + posts only
    for k in ("init_pose", "finger_geom", "grasp_verts", "actions"):
        P[k] = None
    st = orc.OracleSim(P).rollout()
    R, r = 0.02, P["config"]["rope_radius"]
    for b in range(4):
        for k in range(2):
            c = P["prim_params"][b, k, :2]
            dist = np.linalg.norm(st["x"][b, :2].T - c, axis=1)
            assert dist.min() > R + r - 1e-4                     # never sinks into a post (reading B-31, App. D-4)
    x = aos(st["x"])
    strain = np.linalg.norm(np.roll(x, -1, axis=1) - x, axis=2) / P["material"]["rest_edge_len"][:, None] - 1
    assert strain.mean() > 0.02                                  # still stretched over the posts


# --- kinematic attachment follows p + R q exactly ------------------------------------------------------------------------------
def test_grasped_vertices_follow_gripper(orc):
    from scipy.spatial.transform import Rotation
    P = make_problem(3, batch=3, horizon=40)
    st = orc.OracleSim(P).rollout()
    for b in range(3):
        p0, rho0 = P["init_pose"][b, 0, :3], P["init_pose"][b, 0, 3:]
        pT, rhoT = P["actions"][-1, b, 0, :3], P["actions"][-1, b, 0, 3:]
        R0, RT = Rotation.from_rotvec(rho0).as_matrix(), Rotation.from_rotvec(rhoT).as_matrix()
        for k in (0, 1):
            q = R0.T @ (P["x0"][b, :, k] - p0)
            assert np.abs(st["x"][b, :, k] - (pT + RT @ q)).max() < 1e-13
