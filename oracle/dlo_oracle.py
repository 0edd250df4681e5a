"""ORACLE — test infrastructure only (ctypes binding of oracle/liboracle_dlo.so).

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / `--impl reference` legs may import this.
It imports nothing from the product package and the product never imports it.  All arrays are float64 numpy,
laid out like the product C-ABI (x,v,d1: [B][3][N]; kappa_bar: [B][2][N]; actions: [H][B][G][6]).
"""
import ctypes as C
import numpy as np

from . import build as _build

_F = C.c_double
_P = C.POINTER(C.c_double)


class OracleConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "batch", "n_verts", "topology", "n_substeps", "n_proj_iters", "stretch_mode", "enable_plasticity",
        "enable_self_contact", "self_skip", "n_grippers", "n_grasp_max", "n_primitives", "kappa_bar_from_x0")] + [
        ("dt", _F), ("gravity", _F * 3), ("rope_radius", _F), ("contact_softness", _F),
        ("influence_threshold", _F), ("restitution", _F)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(_build.build())
        _lib.oracle_create.restype = C.c_void_p
        _lib.oracle_op_bend_energy.restype = _F
        _lib.oracle_op_stretch_energy.restype = _F
        for name in ("oracle_rollout_forward", "oracle_backward", "oracle_get_record", "oracle_num_threads",
                     "oracle_op_self_contact", "oracle_op_sdf", "oracle_num_margins", "oracle_set_cuts"):
            getattr(_lib, name).restype = C.c_int32
    return _lib


def _d(a):
    return np.ascontiguousarray(a, dtype=np.float64)


def _ptr(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


MARGIN_NAMES = ("approach", "stick", "f_kink", "f_threshold", "yield", "contact", "friction")   # MG_* of rod_step.hpp
MATERIAL_KEYS = ("mass_per_vertex", "rest_edge_len", "stretch", "bend_stiffness", "damping", "yield_curv",
                 "creep_rate", "mu_rigid", "mu_self")


def make_config(cfg: dict) -> OracleConfig:
    oc = OracleConfig()
    for name, _ in OracleConfig._fields_:
        if name == "gravity":
            oc.gravity = (_F * 3)(*[float(g) for g in cfg["gravity"]])
        else:
            setattr(oc, name, cfg[name])
    return oc


class OracleSim:
    """fp64 CPU rollout + tape-AD backward for a problem dict (see workloads/configs.py). `envs` selects a subset."""

    def __init__(self, problem: dict, envs=None, frozen_init=None):
        L = lib()
        cfg = dict(problem["config"])
        B_all = cfg["batch"]
        self.envs = np.arange(B_all) if envs is None else np.asarray(envs, dtype=np.int64)
        cfg["batch"] = len(self.envs)
        self.cfg = cfg
        self.B, self.N, self.G, self.K = cfg["batch"], cfg["n_verts"], cfg["n_grippers"], cfg["n_primitives"]
        self.M = cfg["n_grasp_max"]
        self._oc = make_config(cfg)
        mat = np.stack([_d(problem["material"][k])[self.envs] for k in MATERIAL_KEYS], axis=1)
        self.h = C.c_void_p(L.oracle_create(C.byref(self._oc), _ptr(_d(mat))))
        if problem.get("pins") is not None:
            pins = np.ascontiguousarray(problem["pins"][self.envs], dtype=np.uint8)
            L.oracle_set_pins(self.h, _ptr(pins))
        if problem.get("cuts") is not None:      # several DLOs in one env: absent edges
            cuts = np.ascontiguousarray(problem["cuts"][self.envs], dtype=np.uint8)
            if L.oracle_set_cuts(self.h, _ptr(cuts)) != 0:
                raise ValueError("cuts need the open topology")
        if self.K > 0:
            types = np.ascontiguousarray(problem["prim_types"], dtype=np.int32)
            L.oracle_set_primitives(self.h, _ptr(types), _ptr(_d(problem["prim_params"][self.envs])))
        if self.G > 0:
            gv = np.ascontiguousarray(problem["grasp_verts"][self.envs], dtype=np.int32)
            L.oracle_set_grippers(self.h, _ptr(_d(problem["init_pose"][self.envs])),
                                  _ptr(_d(problem["finger_geom"][self.envs])), _ptr(gv))
        kb = problem.get("kappa_bar0")
        kb = None if kb is None else _d(kb[self.envs])
        L.oracle_set_state(self.h, _ptr(_d(problem["x0"][self.envs])), _ptr(_d(problem["v0"][self.envs])), _ptr(kb))
        if frozen_init is not None:      # test hook: hold the A0 products (frames, grasp-local coordinates) fixed
            d1, q = frozen_init.get("d1"), frozen_init.get("q")
            L.oracle_override_init(self.h, _ptr(None if d1 is None else _d(d1)), _ptr(None if q is None or self.G == 0 else _d(q)))
        self.H = int(problem.get("horizon", 0))
        self.stride = int(problem.get("checkpoint_stride", 0))
        if self.G > 0 and problem.get("actions") is not None:
            self.set_actions(problem["actions"][:, self.envs])

    def init_products(self):
        """A0 products: initial frames d1 [B][3][N] (call before rollout) and grasp-local coordinates q [B][G][M][3]."""
        q = np.zeros((self.B, max(self.G, 0), self.M, 3))
        if self.G > 0:
            lib().oracle_get_grasp_local(self.h, _ptr(q))
        return {"d1": self.state()["d1"], "q": q}

    def set_actions(self, actions):
        a = _d(actions)
        assert a.shape[1:] == (self.B, self.G, 6), a.shape
        lib().oracle_set_actions(self.h, _ptr(a), C.c_int32(a.shape[0]))

    def set_state(self, x0, v0, kappa_bar0=None):
        kb = None if kappa_bar0 is None else _d(kappa_bar0)
        lib().oracle_set_state(self.h, _ptr(_d(x0)), _ptr(_d(v0)), _ptr(kb))

    def restore(self, state, t_start):
        """Harness plumbing: put a full state dict (x, v, d1, kappa_bar as state() returns them) back as the start of
        the next rollout, which then runs frames t_start, t_start+1, ... (no A0; g_actions of backward() is indexed
        from t_start)."""
        lib().oracle_restore_state(self.h, _ptr(_d(state["x"])), _ptr(_d(state["v"])), _ptr(_d(state["d1"])),
                                   _ptr(_d(state["kappa_bar"])), C.c_int32(int(t_start)))

    def rollout(self, horizon=None, stride=None, record=False):
        H = self.H if horizon is None else int(horizon)
        s = self.stride if stride is None else int(stride)
        rc = lib().oracle_rollout_forward(self.h, C.c_int32(H), C.c_int32(s), C.c_int32(1 if record else 0))
        if rc != 0:
            raise RuntimeError("oracle_rollout_forward failed: %d" % rc)
        self.H_done = H
        return self.state()

    def _alloc(self):
        B, N = self.B, self.N
        return (np.zeros((B, 3, N)), np.zeros((B, 3, N)), np.zeros((B, 3, N)), np.zeros((B, 2, N)))

    def state(self):
        x, v, d1, kb = self._alloc()
        lib().oracle_get_state(self.h, _ptr(x), _ptr(v), _ptr(d1), _ptr(kb))
        return {"x": x, "v": v, "d1": d1, "kappa_bar": kb}

    def record(self, t):
        x, v, d1, kb = self._alloc()
        rc = lib().oracle_get_record(self.h, C.c_int32(t), _ptr(x), _ptr(v), _ptr(d1), _ptr(kb))
        if rc != 0:
            raise IndexError(t)
        return {"x": x, "v": v, "d1": d1, "kappa_bar": kb}

    def margins(self):
        """diagnostics: per env, the smallest relative distance to each branch threshold of the step during the last
        rollout, as a dict of arrays [B] keyed by MARGIN_NAMES (inf = the branch was never evaluated)"""
        L = lib()
        n = int(L.oracle_num_margins())
        out = np.zeros((self.B, n))
        L.oracle_get_margins(self.h, _ptr(out))
        out[out > 1e299] = np.inf
        return {name: out[:, i] for i, name in enumerate(MARGIN_NAMES[:n])}

    def backward(self, dL_dxT=None, dL_dvT=None):
        B, N, G, H = self.B, self.N, self.G, self.H_done
        gx = None if dL_dxT is None else _d(dL_dxT)
        gv = None if dL_dvT is None else _d(dL_dvT)
        out = {"g_actions": np.zeros((H, B, max(G, 0), 6)), "g_x0": np.zeros((B, 3, N)), "g_v0": np.zeros((B, 3, N)),
               "g_d10": np.zeros((B, 3, N)), "g_kappa_bar0": np.zeros((B, 2, N)), "g_material": np.zeros((B, 5))}
        rc = lib().oracle_backward(self.h, _ptr(gx), _ptr(gv), _ptr(out["g_actions"]) if G > 0 else None,
                                   _ptr(out["g_x0"]), _ptr(out["g_v0"]), _ptr(out["g_d10"]), _ptr(out["g_kappa_bar0"]),
                                   _ptr(out["g_material"]))
        if rc != 0:
            raise RuntimeError("oracle_backward failed: %d (needs a rollout with checkpoint stride > 0)" % rc)
        return out

    def close(self):
        if self.h:
            lib().oracle_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def num_threads() -> int:
    return int(lib().oracle_num_threads())


# ---------------------------------------------------------------------------------------------------------
# operator-level wrappers (same C++ functions the substep calls); vertex arrays are [N][3] here for convenience
def _soa(a):
    return _d(np.asarray(a, dtype=np.float64).T)


def curvature_binormal(ta, tb):
    out = np.zeros(3)
    lib().oracle_op_curvature_binormal(_ptr(_d(ta)), _ptr(_d(tb)), _ptr(out))
    return out


def frames_init(x, ring=False):
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    d1 = np.zeros((3, N))
    psi = C.c_double(0.0)
    lib().oracle_op_frames_init(C.c_int32(N), C.c_int32(1 if ring else 0), _ptr(_soa(x)), _ptr(d1), C.byref(psi))
    E = N if ring else N - 1
    return d1.T[:E].copy(), psi.value


def _pad_edges(d1, N):
    d = np.zeros((N, 3))
    d[: len(d1)] = d1
    return d


def material_curvature(x, d1, ring=False):
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    k = np.zeros((2, N))
    lib().oracle_op_material_curvature(C.c_int32(N), C.c_int32(1 if ring else 0), _ptr(_soa(x)),
                                       _ptr(_soa(_pad_edges(d1, N))), _ptr(k))
    return k.T.copy()


def bend_energy(x, d1, kbar, alpha, lbar, ring=False):
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    return float(lib().oracle_op_bend_energy(C.c_int32(N), C.c_int32(1 if ring else 0), _ptr(_soa(x)),
                                             _ptr(_soa(_pad_edges(d1, N))), _ptr(_soa(kbar)), _F(alpha), _F(lbar)))


def bend_force(x, d1, kbar, alpha, lbar, ring=False):
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    f = np.zeros((3, N))
    lib().oracle_op_bend_force(C.c_int32(N), C.c_int32(1 if ring else 0), _ptr(_soa(x)), _ptr(_soa(_pad_edges(d1, N))),
                               _ptr(_soa(kbar)), _F(alpha), _F(lbar), _ptr(f))
    return f.T.copy()


def stretch_energy(x, ks, l0, ring=False):
    x = np.asarray(x, dtype=np.float64)
    return float(lib().oracle_op_stretch_energy(C.c_int32(x.shape[0]), C.c_int32(1 if ring else 0), _ptr(_soa(x)), _F(ks), _F(l0)))


def stretch_force(x, ks, l0, ring=False):
    x = np.asarray(x, dtype=np.float64)
    N = x.shape[0]
    f = np.zeros((3, N))
    lib().oracle_op_stretch_force(C.c_int32(N), C.c_int32(1 if ring else 0), _ptr(_soa(x)), _F(ks), _F(l0), _ptr(f))
    return f.T.copy()


def project_edge(xj, xj1, wj, wj1, l0, atil=0.0, S=0.0):
    a, b = _d(xj).copy(), _d(xj1).copy()
    s = C.c_double(S)
    lib().oracle_op_project_edge(_ptr(a), _ptr(b), _F(wj), _F(wj1), _F(l0), _F(atil), C.byref(s))
    return a, b, s.value


def closest_points(p1, q1, p2, q2):
    t, u = C.c_double(0), C.c_double(0)
    lib().oracle_op_closest_points(_ptr(_d(p1)), _ptr(_d(q1)), _ptr(_d(p2)), _ptr(_d(q2)), C.byref(t), C.byref(u))
    return t.value, u.value


def self_contact(x4, w4, rsum):
    x = _d(x4).copy()
    depth = C.c_double(0)
    tu = np.zeros(2)
    hit = lib().oracle_op_self_contact(_ptr(x), _ptr(_d(w4)), _F(rsum), C.byref(depth), _ptr(tu))
    return bool(hit), x, depth.value, tu


def plasticity(kappa, kbar, Y, r_c):
    kb = _d(kbar).copy()
    lib().oracle_op_plasticity(_ptr(_d(kappa)), _ptr(kb), _F(Y), _F(r_c))
    return kb


def sdf(ptype, params, y):
    p = np.zeros(10)
    p[: len(params)] = params
    phi = C.c_double(0)
    n = np.zeros(3)
    ok = lib().oracle_op_sdf(C.c_int32(ptype), _ptr(p), _ptr(_d(y)), C.byref(phi), _ptr(n))
    return bool(ok), phi.value, n


def rigid_response(v, vb, n, d, eps_s=1e-3, f_thresh=0.1, e_rest=0.0, mu=0.5):
    vv = _d(v).copy()
    lib().oracle_op_rigid_response(_ptr(vv), _ptr(_d(vb)), _ptr(_d(n)), _F(d), _F(eps_s), _F(f_thresh), _F(e_rest), _F(mu))
    return vv


def rodrigues(rho):
    R = np.zeros(9)
    lib().oracle_op_rodrigues(_ptr(_d(rho)), _ptr(R))
    return R.reshape(3, 3)


def ptransport(a, b, u):
    out = np.zeros(3)
    lib().oracle_op_ptransport(_ptr(_d(a)), _ptr(_d(b)), _ptr(_d(u)), _ptr(out))
    return out
