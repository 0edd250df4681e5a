"""Pins of the oracle's operators against what the paper and the mathematics fix.

None of these re-types the oracle's formula: they use the identities the paper prints (tests/golden/paper_identities.txt),
finite differences of the energy, closed forms, brute force and scipy routines.
"""
import os

import numpy as np
import pytest
from scipy.spatial.transform import Rotation

GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "paper_identities.txt")) as fh:
    for line in fh:
        line = line.split("#")[0].split()
        if len(line) == 2:
            GOLD[line[0]] = float(line[1])


def unit(v):
    return np.asarray(v, float) / np.linalg.norm(v)


def rot_about(axis, ang):
    return Rotation.from_rotvec(unit(axis) * ang).as_matrix()


def walk_polyline(rng, n, l, wiggle=0.4):
    """polyline with n vertices and exactly equal edge length l (random smooth 3-D directions)."""
    x = np.zeros((n, 3))
    d = unit(rng.normal(size=3))
    for i in range(1, n):
        d = unit(d + wiggle * rng.normal(size=3))
        x[i] = x[i - 1] + l * d
    return x


# --- Eq.4 ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("deg", [0, 60, 90, 120])
def test_curvature_binormal_printed_identity(orc, deg):
    ta = np.array([1.0, 0, 0])
    tb = np.array([np.cos(np.radians(deg)), np.sin(np.radians(deg)), 0])
    kb = orc.curvature_binormal(ta, tb)
    assert abs(np.linalg.norm(kb) - GOLD["kb_norm_phi_deg_%d" % deg]) < 1e-14
    if deg:
        assert np.allclose(unit(kb), [0, 0, 1])          # along t^{i-1} x t^i (right-handed)


def test_curvature_binormal_random(orc):
    rng = np.random.default_rng(0)
    for _ in range(200):
        ta, tb = unit(rng.normal(size=3)), unit(rng.normal(size=3))
        phi = np.arccos(np.clip(ta @ tb, -1, 1))
        kb = orc.curvature_binormal(ta, tb)
        assert abs(np.linalg.norm(kb) - 2 * np.tan(phi / 2)) < 1e-12 * max(1, np.linalg.norm(kb))
        assert abs(kb @ ta) < 1e-12 and abs(kb @ tb) < 1e-12


# --- Eq.5: component order as printed, and |kappa| = |kb| for twist-free frames ------------------------
def test_material_curvature_component_order(orc):
    # planar curve in the xy-plane turning towards +y; d1 = z on both edges => kb = |kb| z = |kb| d1
    x = np.array([[0, 0, 0], [1, 0, 0], [1 + np.cos(0.3), np.sin(0.3), 0.0]])
    d1 = np.array([[0, 0, 1.0], [0, 0, 1.0]])
    k = orc.material_curvature(x, d1)
    assert abs(k[1, 0]) < 1e-15                      # first component  = kb . d2 = 0
    assert abs(k[1, 1] - 2 * np.tan(0.15)) < 1e-14   # second component = kb . d1 = |kb|   (P:L360 as printed)
    assert np.all(k[0] == 0) and np.all(k[2] == 0)   # end vertices carry no curvature


def test_material_curvature_norm_twist_free(orc):
    rng = np.random.default_rng(1)
    x = walk_polyline(rng, 12, 0.1)
    d1, _ = orc.frames_init(x)
    k = orc.material_curvature(x, d1)
    for i in range(1, 11):
        ta, tb = unit(x[i] - x[i - 1]), unit(x[i + 1] - x[i])
        assert abs(np.linalg.norm(k[i]) - np.linalg.norm(orc.curvature_binormal(ta, tb))) < 1e-13


# --- frames: adapted, unit, parallel transport = rotation about a x b -------------------------------------
def test_parallel_transport_is_minimal_rotation(orc):
    rng = np.random.default_rng(2)
    for _ in range(50):
        a, b, u = unit(rng.normal(size=3)), unit(rng.normal(size=3)), rng.normal(size=3)
        ang = np.arccos(np.clip(a @ b, -1, 1))
        ref = rot_about(np.cross(a, b), ang) @ u
        assert np.allclose(orc.ptransport(a, b, u), ref, atol=1e-12)
        assert np.allclose(orc.ptransport(a, b, a), b, atol=1e-12)


def test_frames_init_adapted_unit(orc):
    rng = np.random.default_rng(3)
    x = walk_polyline(rng, 20, 0.05)
    d1, psi = orc.frames_init(x)
    t = np.array([unit(x[j + 1] - x[j]) for j in range(19)])
    assert np.abs(np.sum(d1 * t, axis=1)).max() < 1e-13
    assert np.abs(np.linalg.norm(d1, axis=1) - 1).max() < 1e-13
    assert psi == 0.0
    # first frame: component of z perpendicular to t0
    assert np.allclose(d1[0], unit(np.array([0, 0, 1.0]) - t[0][2] * t[0]))
    # straight rope along z falls back to y
    xs = np.zeros((4, 3)); xs[:, 2] = np.arange(4)
    assert np.allclose(orc.frames_init(xs)[0][0], [0, 1, 0])


# --- Eq.12 loop holonomy --------------------------------------------------------------------------------
def vertex_twists(x, d1):
    """signed angle (about the outgoing tangent) from the transported incoming d1 to the outgoing d1, every vertex of a ring"""
    N = len(x)
    t = np.array([unit(x[(j + 1) % N] - x[j]) for j in range(N)])
    out = []
    for i in range(N):
        a, b = (i - 1) % N, i
        ang = np.arccos(np.clip(t[a] @ t[b], -1, 1))
        u = rot_about(np.cross(t[a], t[b]), ang) @ d1[a] if ang > 1e-14 else d1[a]
        out.append(np.arctan2(np.cross(u, d1[b]) @ t[b], u @ d1[b]))
    return np.array(out)


def test_loop_frames_equal_twist_everywhere(orc):
    rng = np.random.default_rng(4)
    N = 24
    th = np.linspace(0, 2 * np.pi, N, endpoint=False)
    x = np.stack([np.cos(th) * (1 + 0.3 * np.cos(3 * th)), np.sin(th) * (1 + 0.3 * np.cos(3 * th)), 0.4 * np.sin(2 * th) + 0.2 * np.cos(5 * th)], 1)
    x += 0.02 * rng.normal(size=x.shape)
    d1, psi = orc.frames_init(x, ring=True)
    assert abs(psi) > 1e-3                                  # genuinely non-planar: there IS a holonomy
    tw = vertex_twists(x, d1)
    assert np.abs(tw - tw.mean()).max() < 1e-12             # "consistent and continuous across the entire loop"
    assert abs(np.angle(np.exp(1j * (tw.sum() + psi)))) < 1e-10   # the twists add up to -psi_H (mod 2 pi)
    t = np.array([unit(x[(j + 1) % N] - x[j]) for j in range(N)])
    assert np.abs(np.sum(d1 * t, axis=1)).max() < 1e-13 and np.abs(np.linalg.norm(d1, axis=1) - 1).max() < 1e-13


def test_loop_frames_planar_ring_has_no_holonomy(orc):
    N = 16
    th = np.linspace(0, 2 * np.pi, N, endpoint=False)
    x = np.stack([np.cos(th), np.sin(th), 0 * th], 1)
    d1, psi = orc.frames_init(x, ring=True)
    assert abs(psi) < 1e-13
    assert np.allclose(d1, np.tile([0, 0, 1.0], (N, 1)), atol=1e-13)


# --- Eq.6-7 bending energy / force ---------------------------------------------------------------------
@pytest.mark.parametrize("ring", [False, True])
def test_bend_force_is_minus_energy_gradient(orc, ring):
    rng = np.random.default_rng(5)
    N = 8
    if ring:
        th = np.linspace(0, 2 * np.pi, N, endpoint=False)
        x = np.stack([np.cos(th), np.sin(th), 0.3 * np.sin(2 * th)], 1) * 0.1 + 0.004 * rng.normal(size=(N, 3))
    else:
        x = walk_polyline(rng, N, 0.05)
    d1, _ = orc.frames_init(x, ring=ring)
    kbar = 0.1 * rng.normal(size=(N, 2))
    alpha, lbar = 1.3e-3, 0.05
    F = orc.bend_force(x, d1, kbar, alpha, lbar, ring=ring)
    Fd = np.zeros_like(F)
    eps = 1e-6
    for i in range(N):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, c] += eps; xm[i, c] -= eps
            Fd[i, c] = -(orc.bend_energy(xp, d1, kbar, alpha, lbar, ring=ring) - orc.bend_energy(xm, d1, kbar, alpha, lbar, ring=ring)) / (2 * eps)
    assert np.linalg.norm(F - Fd) / np.linalg.norm(F) < 1e-8
    assert np.abs(F.sum(axis=0)).max() < 1e-15 * max(1, np.abs(F).max()) * 100     # internal force: no net force


def test_bend_energy_regular_polygon_closed_form(orc):
    alpha, R = 2e-3, 0.1
    for N in (6, 16, 96):
        th = np.linspace(0, 2 * np.pi, N, endpoint=False)
        x = R * np.stack([np.cos(th), np.sin(th), 0 * th], 1)
        lbar = 2 * R * np.sin(np.pi / N)
        d1, _ = orc.frames_init(x, ring=True)
        U = orc.bend_energy(x, d1, np.zeros((N, 2)), alpha, lbar, ring=True)
        assert abs(U - N * alpha / (2 * lbar) * 4 * np.tan(np.pi / N) ** 2) < 1e-12 * U
    assert abs(U - np.pi * alpha / R) / U < 1e-3          # continuum limit pi alpha / R


def test_bend_energy_zero_at_rest_curvature(orc):
    rng = np.random.default_rng(6)
    x = walk_polyline(rng, 10, 0.03)
    d1, _ = orc.frames_init(x)
    k = orc.material_curvature(x, d1)
    assert orc.bend_energy(x, d1, k, 1e-2, 0.03) < 1e-30
    assert np.abs(orc.bend_force(x, d1, k, 1e-2, 0.03)).max() < 1e-15


# --- Eq.2-3 stretching ----------------------------------------------------------------------------------
def test_stretch_energy_and_force(orc):
    rng = np.random.default_rng(7)
    x = walk_polyline(rng, 3, 0.1)
    x[2] = x[1] + 1.1 * (x[2] - x[1])           # second edge strained by 10 %
    ks, l0 = 50.0, 0.1
    assert abs(orc.stretch_energy(x, ks, l0) - 0.5 * ks * 0.1 ** 2 * l0) < 1e-14      # 1/2 k eps^2 l0 (Eq.3)
    F = orc.stretch_force(x, ks, l0)
    eps = 1e-7
    for i in range(3):
        for c in range(3):
            xp, xm = x.copy(), x.copy()
            xp[i, c] += eps; xm[i, c] -= eps
            fd = -(orc.stretch_energy(xp, ks, l0) - orc.stretch_energy(xm, ks, l0)) / (2 * eps)
            assert abs(F[i, c] - fd) < 1e-7
    assert np.allclose(F[2], -ks * 0.1 * unit(x[2] - x[1]))                           # pulls the far vertex back


# --- Eq.10 --------------------------------------------------------------------------------------------------
def test_project_edge_exact_single_constraint(orc):
    rng = np.random.default_rng(8)
    for _ in range(20):
        a, b = rng.normal(size=3), rng.normal(size=3)
        wa, wb, l0 = rng.uniform(1, 200), rng.uniform(1, 200), rng.uniform(0.1, 2)
        a2, b2, S = orc.project_edge(a, b, wa, wb, l0)
        assert abs(np.linalg.norm(b2 - a2) - l0) < 1e-14                  # exact projection of one constraint
        assert np.allclose((a2 - a) / wa + (b2 - b) / wb, 0, atol=1e-15)  # sum m dx = 0
        assert np.allclose(np.cross(a2 - a, b - a), 0, atol=1e-13)        # along the edge tangent
        assert abs(S - (np.linalg.norm(b - a) - l0) / (wa + wb)) < 1e-14  # lambda as printed
    a2, b2, _ = orc.project_edge(a, b, 0.0, wb, l0)
    assert np.array_equal(a2, a) and abs(np.linalg.norm(b2 - a2) - l0) < 1e-14   # kinematic vertex does not move
    a2, b2, _ = orc.project_edge(a, b, 0.0, 0.0, l0)
    assert np.array_equal(a2, a) and np.array_equal(b2, b)


def test_project_edge_compliant_form(orc):
    a, b = np.zeros(3), np.array([1.2, 0, 0])
    w, l0, atil = 100.0, 1.0, 50.0
    a2, b2, S = orc.project_edge(a, b, w, w, l0, atil=atil)
    C0, C1 = 0.2, np.linalg.norm(b2 - a2) - l0
    assert abs(C1 - C0 * atil / (2 * w + atil)) < 1e-15                   # residual of the regularised projection
    # second application with the accumulated multiplier converges to the compliant fixed point C = -atil * S
    a3, b3, S2 = orc.project_edge(a2, b2, w, w, l0, atil=atil, S=S)
    lam2 = (C1 - atil * S) / (2 * w + atil)
    assert abs(S2 - (S + lam2)) < 1e-15


# --- closest points (B-14) vs brute force -------------------------------------------------------------------------
def test_closest_points_brute_force(orc):
    rng = np.random.default_rng(9)
    g = np.linspace(0, 1, 401)
    T, U = np.meshgrid(g, g, indexing="ij")
    for _ in range(30):
        p1, q1, p2, q2 = (rng.normal(size=3) for _ in range(4))
        t, u = orc.closest_points(p1, q1, p2, q2)
        assert 0 <= t <= 1 and 0 <= u <= 1
        d = np.linalg.norm((1 - t) * p1 + t * q1 - (1 - u) * p2 - u * q2)
        D = np.linalg.norm(((1 - T)[..., None] * p1 + T[..., None] * q1) - ((1 - U)[..., None] * p2 + U[..., None] * q2), axis=-1)
        assert d <= D.min() + 1e-12
        assert d >= D.min() - 2e-2 * (np.linalg.norm(q1 - p1) + np.linalg.norm(q2 - p2)) / 400 * 4


def test_closest_points_parallel_rule(orc):
    t, u = orc.closest_points([0, 0, 0], [1, 0, 0], [0.25, 1, 0], [0.75, 1, 0])
    assert t == 0.0 or (0 <= t <= 1)
    d = np.linalg.norm(np.array([t, 0, 0]) - np.array([0.25 + 0.5 * u, 1, 0]))
    assert abs(d - 1.0) < 1e-15 or abs(d - np.hypot(0.25, 1)) < 1e-15     # rule: t=0, then u clamped, then t re-solved
    t, u = orc.closest_points([0, 0, 0], [1, 0, 0], [2, 0, 0], [3, 0, 0])  # collinear, disjoint
    assert (t, u) == (1.0, 0.0)


# --- Eq.13 -----------------------------------------------------------------------------------------------
def test_self_contact_separates_exactly_and_conserves_momentum(orc):
    rng = np.random.default_rng(10)
    hits = 0
    for _ in range(200):
        x = rng.normal(size=(4, 3)) * 0.02
        w = rng.uniform(50, 150, 4)
        rsum = 0.012
        hit, x2, depth, tu = orc.self_contact(x, w, rsum)
        t, u = tu
        ca, cb = (1 - t) * x[0] + t * x[1], (1 - u) * x[2] + u * x[3]
        assert abs(depth - (rsum - np.linalg.norm(ca - cb))) < 1e-15
        if not hit:
            assert depth <= 0
            continue
        hits += 1
        ca2, cb2 = (1 - t) * x2[0] + t * x2[1], (1 - u) * x2[2] + u * x2[3]
        assert abs(np.linalg.norm(ca2 - cb2) - rsum) < 1e-14          # same barycentrics: separated by exactly d
        assert np.abs(((x2 - x) / w[:, None]).sum(axis=0)).max() < 1e-17   # sum m dx = 0
    assert hits > 20
    # a kinematic segment (w=0) does not move; the other takes the whole correction
    x = np.array([[0, 0, 0], [1, 0, 0], [0.5, -0.5, 0.005], [0.5, 0.5, 0.005]])
    hit, x2, depth, _ = orc.self_contact(x, [0, 0, 100, 100], 0.01)
    assert hit and np.array_equal(x2[:2], x[:2]) and np.allclose(x2[2:, 2], 0.01)


# --- Eq.11 ---------------------------------------------------------------------------------------------------
def test_plasticity_unit_pins(orc):
    kappa, kbar = np.array([0.3, -0.4]), np.array([0.05, 0.02])
    el = kappa - kbar
    n0 = np.linalg.norm(el)
    Y = 0.2
    kb1 = orc.plasticity(kappa, kbar, Y, 1.0)                       # r_c = 1: back onto the yield surface
    assert abs(np.linalg.norm(kappa - kb1) - Y) < 1e-15
    assert np.allclose(np.cross(kappa - kb1, el), 0)                # radial return
    kb = kbar.copy()
    for k in range(1, 6):                                           # excess decays by (1 - r_c) per update
        kb = orc.plasticity(kappa, kb, Y, 0.3)
        assert abs((np.linalg.norm(kappa - kb) - Y) - (n0 - Y) * 0.7 ** k) < 1e-15
    assert np.array_equal(orc.plasticity(kappa, kbar, 1.0, 0.5), kbar)   # below yield: unchanged


# --- Rodrigues -------------------------------------------------------------------------------------------------
def test_rodrigues_matches_scipy(orc):
    rng = np.random.default_rng(11)
    for scale in (1e-7, 1e-5, 0.9e-4, 1.1e-4, 1e-2, 1.0, 3.0):
        rho = unit(rng.normal(size=3)) * scale
        assert np.abs(orc.rodrigues(rho) - Rotation.from_rotvec(rho).as_matrix()).max() < 1e-15
    assert np.array_equal(orc.rodrigues([0, 0, 0]), np.eye(3))


# --- SDFs ------------------------------------------------------------------------------------------------------
def fd_grad(orc, ptype, params, y, eps=1e-6):
    g = np.zeros(3)
    for c in range(3):
        yp, ym = np.array(y, float), np.array(y, float)
        yp[c] += eps; ym[c] -= eps
        g[c] = (orc.sdf(ptype, params, yp)[1] - orc.sdf(ptype, params, ym)[1]) / (2 * eps)
    return g


def test_sdf_closed_form_cases(orc):
    s2 = np.sqrt(2)
    # plane z = 0.1
    ok, phi, n = orc.sdf(0, [0, 0, 1, 0.1], [3, 4, 0.35]); assert ok and abs(phi - 0.25) < 1e-15 and np.allclose(n, [0, 0, 1])
    # capsule from (0,0,0) to (0,0,1), R = 0.1
    cap = [0, 0, 0, 0, 0, 1, 0.1]
    ok, phi, n = orc.sdf(1, cap, [0.5, 0, 0.5]); assert abs(phi - 0.4) < 1e-15 and np.allclose(n, [1, 0, 0])
    ok, phi, n = orc.sdf(1, cap, [0.3, 0, 1.4]); assert abs(phi - 0.4) < 1e-15 and np.allclose(n, [0.6, 0, 0.8])
    ok, phi, n = orc.sdf(1, cap, [0, 0, -0.05]); assert abs(phi + 0.05) < 1e-15 and np.allclose(n, [0, 0, -1])
    assert not orc.sdf(1, cap, [0, 0, 0.5])[0]                         # on the axis: gradient undefined, skipped
    # cylinder centre (0,0,0.1), axis z, R = 0.02, half height 0.1
    cyl = [0, 0, 0.1, 0, 0, 1, 0.02, 0.1]
    ok, phi, n = orc.sdf(2, cyl, [0.05, 0, 0.1]); assert abs(phi - 0.03) < 1e-15 and np.allclose(n, [1, 0, 0])
    ok, phi, n = orc.sdf(2, cyl, [0.01, 0, 0.25]); assert abs(phi - 0.05) < 1e-15 and np.allclose(n, [0, 0, 1])
    ok, phi, n = orc.sdf(2, cyl, [0.05, 0, 0.23]); assert abs(phi - 0.03 * s2) < 1e-15 and np.allclose(n, [1 / s2, 0, 1 / s2])
    ok, phi, n = orc.sdf(2, cyl, [0.015, 0, 0.1]); assert abs(phi + 0.005) < 1e-15 and np.allclose(n, [1, 0, 0])
    ok, phi, n = orc.sdf(2, cyl, [0.001, 0, 0.004]); assert abs(phi + 0.004) < 1e-15 and np.allclose(n, [0, 0, -1])
    # axis-aligned box centre (1,2,3), half extents (0.1,0.2,0.3)
    box = [1, 2, 3, 0.1, 0.2, 0.3, 0, 0, 0]
    ok, phi, n = orc.sdf(3, box, [1.5, 2, 3]); assert abs(phi - 0.4) < 1e-15 and np.allclose(n, [1, 0, 0])
    ok, phi, n = orc.sdf(3, box, [1.4, 2.6, 3]); assert abs(phi - 0.5) < 1e-15 and np.allclose(n, [0.6, 0.8, 0])
    ok, phi, n = orc.sdf(3, box, [0.8, 1.6, 2.6]); assert abs(phi - np.sqrt(0.01 + 0.04 + 0.01)) < 1e-15
    ok, phi, n = orc.sdf(3, box, [1.05, 2.0, 3.0]); assert abs(phi + 0.05) < 1e-15 and np.allclose(n, [1, 0, 0])
    ok, phi, n = orc.sdf(3, box, [1.0, 2.0, 2.75]); assert abs(phi + 0.05) < 1e-15 and np.allclose(n, [0, 0, -1])
    # rotated box: 90 deg yaw swaps the x/y half extents
    boxr = [0, 0, 0, 0.1, 0.2, 0.3, 0, 0, np.pi / 2]
    ok, phi, n = orc.sdf(3, boxr, [0.5, 0, 0]); assert abs(phi - 0.3) < 1e-12 and np.allclose(n, [1, 0, 0])


def test_sdf_gradient_is_unit_and_matches_fd(orc):
    rng = np.random.default_rng(12)
    prims = [(0, list(unit([0.2, -0.3, 1])) + [0.05]), (1, [0.1, 0, 0, -0.2, 0.3, 0.4, 0.03]),
             (2, [0.1, -0.1, 0.2] + list(unit([0.3, 0.2, 1])) + [0.05, 0.12]),
             (3, [0.05, 0.02, -0.03, 0.06, 0.1, 0.04, 0.3, -0.5, 0.8])]
    for ptype, prm in prims:
        for _ in range(60):
            y = rng.uniform(-0.4, 0.4, 3)
            ok, phi, n = orc.sdf(ptype, prm, y)
            assert ok
            assert abs(np.linalg.norm(n) - 1) < 1e-12
            g = fd_grad(orc, ptype, prm, y)
            if np.linalg.norm(g - n) > 1e-5:                    # FD straddles a medial-axis / face switch: check one side
                continue
            # moving along -n by phi lands on the surface (exact Euclidean distance, outside points)
            if phi > 0:
                assert abs(orc.sdf(ptype, prm, y - phi * n)[1]) < 1e-10


# --- P:L103 soft coupling response --------------------------------------------------------------------------------
def test_rigid_response_closed_forms(orc):
    n = np.array([0, 0, 1.0])
    z = np.zeros(3)
    # f = 1 (d >= 0): restitution on the normal component
    assert np.allclose(orc.rigid_response([0, 0, -2.0], z, n, 0.0, e_rest=0.3, mu=0.0), [0, 0, 0.6])
    assert GOLD["influence_at_d0"] == 1.0
    # Coulomb: sliding loses mu (1+e) |u_n| of tangential speed; sticking stops
    assert np.allclose(orc.rigid_response([1.0, 0, -1.0], z, n, 1e-3, e_rest=0.0, mu=0.5), [0.5, 0, 0])
    assert np.allclose(orc.rigid_response([0.3, 0, -1.0], z, n, 1e-3, e_rest=0.0, mu=0.5), [0, 0, 0])
    assert np.allclose(orc.rigid_response([1.0, 0, -1.0], z, n, 1e-3, e_rest=0.5, mu=0.2), [0.7, 0, 0.5])
    # separating: untouched
    assert np.array_equal(orc.rigid_response([1.0, 0, 0.1], z, n, 1e-3), [1.0, 0, 0.1])
    # below the influence threshold f <= 0.1: untouched; just above: blended by f
    eps = 1e-3
    d_thr = eps * np.log(GOLD["influence_threshold"])
    assert np.array_equal(orc.rigid_response([0, 0, -1.0], z, n, d_thr * 1.001, eps_s=eps), [0, 0, -1.0])
    v = orc.rigid_response([0, 0, -1.0], z, n, eps * np.log(0.5), eps_s=eps, mu=0.0)
    assert np.allclose(v, [0, 0, -0.5])                                  # v + f (u' - u), f = 0.5, e = 0
    # moving body: response acts on the relative velocity
    assert np.allclose(orc.rigid_response([0, 0, 0.0], [0, 0, 1.0], n, 0.0, mu=0.0), [0, 0, 1.0])
