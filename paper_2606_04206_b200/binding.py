"""ctypes binding of libdlo_b200.so (include/dlo.h).  Argument marshalling only: every step of the path runs in
the CUDA kernels.  The `dlo_*` functions mirror the C entry points one to one (torch CUDA tensors or raw
integer device pointers in, status checked, DloError raised); `DloSim` bundles the usual call sequence for a
problem dict of workloads/configs.py.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

_F = C.c_float
STATUS_CALLS = ("dlo_create", "dlo_destroy", "dlo_set_pins", "dlo_set_cuts", "dlo_set_primitives", "dlo_set_grippers", "dlo_set_state",
                "dlo_restore_state", "dlo_set_actions", "dlo_rollout_forward", "dlo_get_state", "dlo_get_position_residual",
                "dlo_backward",
                "dlo_get_state_adjoint", "dlo_rollout_forward_host", "dlo_backward_host", "dlo_check_numerics",
                "dlo_set_kernel_timing", "dlo_get_kernel_timing", "dlo_measure_fp32_peak", "dlo_rollout_forward_static")
EXPORTS = STATUS_CALLS + ("dlo_scratch_bytes", "dlo_static_scratch_bytes", "dlo_launch_count", "dlo_last_error", "dlo_version")
STATIC_SCRATCH_BYTES = 4 << 20   # DLO_STATIC_SCRATCH_BYTES of include/dlo.h
MATERIAL_KEYS = ("mass_per_vertex", "rest_edge_len", "stretch", "bend_stiffness", "damping", "yield_curv",
                 "creep_rate", "mu_rigid", "mu_self")
STATUS = {0: "DLO_OK", -1: "DLO_ERR_INVALID_ARG", -2: "DLO_ERR_BAD_STATE", -3: "DLO_ERR_CUDA", -4: "DLO_ERR_OOM",
          -5: "DLO_ERR_UNSUPPORTED", -6: "DLO_ERR_NUMERIC"}


class DloConfig(C.Structure):
    _fields_ = [(n, C.c_int32) for n in (
        "batch", "n_verts", "topology", "n_substeps", "n_proj_iters", "stretch_mode", "enable_plasticity",
        "enable_self_contact", "self_skip", "n_grippers", "n_grasp_max", "n_primitives", "kappa_bar_from_x0")] + [
        ("dt", _F), ("gravity", _F * 3), ("rope_radius", _F), ("contact_softness", _F),
        ("influence_threshold", _F), ("restitution", _F)]


class DloMaterial(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in MATERIAL_KEYS]


class DloScene(C.Structure):
    _fields_ = [(n, C.c_void_p) for n in ("pinned", "prim_types", "prim_params", "init_pose", "finger_geom", "grasp_verts", "actions")]


class DloError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS.get(status, status), msg))
        self.status = status


_lib = None


def lib():
    """Loads (building if stale) the C-ABI library.  Fails loudly if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.build()
        L = C.CDLL(path)
        for name in EXPORTS:
            getattr(L, name)            # AttributeError if a declared symbol is missing
        L.dlo_last_error.restype = C.c_char_p
        L.dlo_version.restype = C.c_char_p
        L.dlo_scratch_bytes.restype = C.c_size_t
        L.dlo_static_scratch_bytes.restype = C.c_size_t
        L.dlo_launch_count.restype = C.c_int64
        L.dlo_launch_count.argtypes = [C.c_void_p]
        for name in STATUS_CALLS:
            getattr(L, name).restype = C.c_int32
        _lib = L
    return _lib


def _chk(status):
    if status != 0:
        raise DloError(status, (lib().dlo_last_error() or b"").decode())


def _p(t):
    """device / host pointer of a torch tensor, numpy array, int or None"""
    if t is None:
        return C.c_void_p(None)
    if isinstance(t, int):
        return C.c_void_p(t)
    if isinstance(t, np.ndarray):
        assert t.flags["C_CONTIGUOUS"]
        return C.c_void_p(t.ctypes.data)
    assert t.is_contiguous(), "tensor must be contiguous"
    return C.c_void_p(t.data_ptr())


def make_config(cfg: dict) -> DloConfig:
    c = DloConfig()
    for name, _ in DloConfig._fields_:
        if name == "gravity":
            c.gravity = (_F * 3)(*[float(g) for g in cfg["gravity"]])
        else:
            setattr(c, name, cfg[name])
    return c


# ---- one-to-one wrappers -------------------------------------------------------------------------------------
def dlo_create(cfg: DloConfig, material: dict, stream=0):
    m = DloMaterial()
    for k in MATERIAL_KEYS:
        setattr(m, k, material[k].data_ptr())
    h = C.c_void_p()
    _chk(lib().dlo_create(C.byref(cfg), C.byref(m), C.c_void_p(stream), C.byref(h)))
    return h


def dlo_destroy(h):
    _chk(lib().dlo_destroy(h))


def dlo_set_pins(h, pinned):
    _chk(lib().dlo_set_pins(h, _p(pinned)))


def dlo_set_cuts(h, cut):
    _chk(lib().dlo_set_cuts(h, _p(cut)))


def dlo_set_primitives(h, types_host, params):
    t = np.ascontiguousarray(types_host, dtype=np.int32)
    _chk(lib().dlo_set_primitives(h, _p(t), _p(params)))


def dlo_set_grippers(h, init_pose, finger_geom, grasp_verts):
    _chk(lib().dlo_set_grippers(h, _p(init_pose), _p(finger_geom), _p(grasp_verts)))


def dlo_set_state(h, x0, v0, kappa_bar0=None):
    _chk(lib().dlo_set_state(h, _p(x0), _p(v0), _p(kappa_bar0)))


def dlo_restore_state(h, x, x_lo, v, d1, kappa_bar, step_index):
    _chk(lib().dlo_restore_state(h, _p(x), _p(x_lo), _p(v), _p(d1), _p(kappa_bar), C.c_int32(step_index)))


def dlo_get_position_residual(h, x_lo):
    _chk(lib().dlo_get_position_residual(h, _p(x_lo)))


def dlo_get_state_adjoint(h, g_x=None, g_v=None, g_d1=None, g_kappa_bar=None):
    _chk(lib().dlo_get_state_adjoint(h, _p(g_x), _p(g_v), _p(g_d1), _p(g_kappa_bar)))


def dlo_set_actions(h, actions, horizon):
    _chk(lib().dlo_set_actions(h, _p(actions), C.c_int32(horizon)))


def dlo_rollout_forward(h, horizon, checkpoint_stride):
    _chk(lib().dlo_rollout_forward(h, C.c_int32(horizon), C.c_int32(checkpoint_stride)))


def dlo_get_state(h, x=None, v=None, d1=None, kappa_bar=None):
    _chk(lib().dlo_get_state(h, _p(x), _p(v), _p(d1), _p(kappa_bar)))


def dlo_backward(h, dL_dxT=None, dL_dvT=None, g_actions=None, g_x0=None, g_v0=None, g_material=None):
    _chk(lib().dlo_backward(h, _p(dL_dxT), _p(dL_dvT), _p(g_actions), _p(g_x0), _p(g_v0), _p(g_material)))


def dlo_rollout_forward_host(h, x0, v0, kappa_bar0, actions, horizon, checkpoint_stride, x_T=None, v_T=None):
    _chk(lib().dlo_rollout_forward_host(h, _p(x0), _p(v0), _p(kappa_bar0), _p(actions), C.c_int32(horizon),
                                        C.c_int32(checkpoint_stride), _p(x_T), _p(v_T)))


def dlo_backward_host(h, dL_dxT=None, dL_dvT=None, g_actions=None, g_x0=None, g_v0=None, g_material=None):
    _chk(lib().dlo_backward_host(h, _p(dL_dxT), _p(dL_dvT), _p(g_actions), _p(g_x0), _p(g_v0), _p(g_material)))


def dlo_check_numerics(h):
    n = C.c_int32(0)
    st = lib().dlo_check_numerics(h, C.byref(n))
    if st not in (0, -6):
        _chk(st)
    return int(n.value)


def dlo_set_kernel_timing(h, on):
    _chk(lib().dlo_set_kernel_timing(h, C.c_int32(1 if on else 0)))


def dlo_get_kernel_timing(h, kernel_class):
    """(launches, total ms, env-steps) of kernel class 0 forward / 1 replay / 2 adjoint since dlo_set_kernel_timing(on)"""
    n, ms, units = C.c_int32(0), C.c_double(0.0), C.c_int64(0)
    _chk(lib().dlo_get_kernel_timing(h, C.c_int32(kernel_class), C.byref(n), C.byref(ms), C.byref(units)))
    return int(n.value), float(ms.value), int(units.value)


def dlo_measure_fp32_peak(stream=0):
    """(TFLOP/s, elapsed ms, SM count) of the FFMA-chain microbenchmark on the current device"""
    tf, ms, n = C.c_double(0.0), C.c_double(0.0), C.c_int32(0)
    _chk(lib().dlo_measure_fp32_peak(C.c_void_p(stream), C.byref(tf), C.byref(ms), C.byref(n)))
    return float(tf.value), float(ms.value), int(n.value)


def dlo_scratch_bytes(cfg: DloConfig, horizon, checkpoint_stride):
    return int(lib().dlo_scratch_bytes(C.byref(cfg), C.c_int32(horizon), C.c_int32(checkpoint_stride)))


def dlo_static_scratch_bytes(cfg: DloConfig):
    return int(lib().dlo_static_scratch_bytes(C.byref(cfg)))


def dlo_rollout_forward_static(cfg: DloConfig, material: dict, scene: dict, x0, v0, kappa_bar0, horizon, x_T=None, v_T=None,
                               env_flags=None, stream=0):
    """The forward rollout without any allocation in the library (scratch in a static device array; include/dlo.h).  `scene`:
    dict with any of pinned, prim_types (host int32 array), prim_params, init_pose, finger_geom, grasp_verts, actions."""
    m = DloMaterial()
    for k in MATERIAL_KEYS:
        setattr(m, k, material[k].data_ptr())
    sc = DloScene()
    keep = None
    for k, _ in DloScene._fields_:
        v = (scene or {}).get(k)
        if k == "prim_types" and v is not None:
            keep = v = np.ascontiguousarray(v, dtype=np.int32)
        setattr(sc, k, _p(v).value)
    _chk(lib().dlo_rollout_forward_static(C.byref(cfg), C.byref(m), C.byref(sc), _p(x0), _p(v0), _p(kappa_bar0), C.c_int32(horizon),
                                          _p(x_T), _p(v_T), _p(env_flags), C.c_void_p(stream)))
    del keep


def dlo_launch_count(h):
    return int(lib().dlo_launch_count(h))


def dlo_last_error():
    return (lib().dlo_last_error() or b"").decode()


def dlo_version():
    return lib().dlo_version().decode()


# ---- convenience: a problem dict (workloads/configs.py) -> a simulator ----------------------------------------
class DloSim:
    """Uploads a problem dict as fp32 and drives the C-ABI.  `envs` selects a subset of environments."""

    def __init__(self, problem: dict, envs=None, device="cuda:0", stream=None):
        import torch
        if not torch.cuda.is_available():
            raise DloError(-3, "no CUDA device: the DLO library has no CPU path")
        self.torch = torch
        self.dev = torch.device(device)
        cfg = dict(problem["config"])
        sel = np.arange(cfg["batch"]) if envs is None else np.asarray(envs, dtype=np.int64)
        cfg["batch"] = len(sel)
        self.cfg, self.sel = cfg, sel
        self.B, self.N, self.G, self.K = cfg["batch"], cfg["n_verts"], cfg["n_grippers"], cfg["n_primitives"]
        self.H = int(problem.get("horizon", 0))
        self.stride = int(problem.get("checkpoint_stride", 0))
        self._keep = []
        self.ccfg = make_config(cfg)
        with torch.cuda.device(self.dev):
            self.stream = stream.cuda_stream if stream is not None else torch.cuda.current_stream().cuda_stream
            mat = {k: self._up(problem["material"][k][sel]) for k in MATERIAL_KEYS}
            self.h = dlo_create(self.ccfg, mat, self.stream)
            if problem.get("pins") is not None:
                dlo_set_pins(self.h, self._up(problem["pins"][sel], torch.uint8))
            if problem.get("cuts") is not None:
                dlo_set_cuts(self.h, self._up(problem["cuts"][sel], torch.uint8))
            if self.K > 0:
                dlo_set_primitives(self.h, problem["prim_types"], self._up(problem["prim_params"][sel]))
            if self.G > 0:
                dlo_set_grippers(self.h, self._up(problem["init_pose"][sel]), self._up(problem["finger_geom"][sel]),
                                 self._up(problem["grasp_verts"][sel], torch.int32))
            kb = problem.get("kappa_bar0")
            self.x0, self.v0 = self._up(problem["x0"][sel]), self._up(problem["v0"][sel])
            self.kb0 = None if kb is None else self._up(kb[sel])
            dlo_set_state(self.h, self.x0, self.v0, self.kb0)
            self.actions = None
            if self.G > 0 and problem.get("actions") is not None:
                self.set_actions(problem["actions"][:, sel])

    def _up(self, a, dtype=None):
        torch = self.torch
        t = torch.as_tensor(np.ascontiguousarray(a), dtype=dtype or torch.float32).to(self.dev).contiguous()
        self._keep.append(t)
        return t

    def set_actions(self, actions):
        self.actions = self._up(actions) if not hasattr(actions, "data_ptr") else actions
        dlo_set_actions(self.h, self.actions, int(self.actions.shape[0]))

    def set_state(self, x0, v0, kappa_bar0=None):
        self.x0, self.v0 = self._up(x0), self._up(v0)
        self.kb0 = None if kappa_bar0 is None else self._up(kappa_bar0)
        dlo_set_state(self.h, self.x0, self.v0, self.kb0)

    def restore(self, state, step_index):
        """exact restore of a state dict (x, v, d1, kappa_bar and optionally x_lo: numpy or device tensors) as the start
        of the next rollout.  fp64 numpy positions without an x_lo are split into their nearest fp32 and the fp32 residual."""
        t = {k: (state[k] if hasattr(state[k], "data_ptr") else self._up(state[k])) for k in ("v", "d1", "kappa_bar")}
        x, xl = state["x"], state.get("x_lo")
        if hasattr(x, "data_ptr"):
            t["x"], t["x_lo"] = x, xl
        else:
            a = np.asarray(x, dtype=np.float64)
            hi = a.astype(np.float32)
            t["x"] = self._up(hi)
            t["x_lo"] = self._up((a - hi.astype(np.float64)).astype(np.float32) if xl is None else xl)
        self._restored = t
        dlo_restore_state(self.h, t["x"], t["x_lo"], t["v"], t["d1"], t["kappa_bar"], int(step_index))

    def state_device(self):
        """current state as fp32 device tensors (no host copy)"""
        torch = self.torch
        B, N = self.B, self.N
        out = {"x": torch.empty((B, 3, N), device=self.dev), "v": torch.empty((B, 3, N), device=self.dev),
               "d1": torch.empty((B, 3, N), device=self.dev), "kappa_bar": torch.empty((B, 2, N), device=self.dev),
               "x_lo": torch.empty((B, 3, N), device=self.dev)}
        dlo_get_state(self.h, out["x"], out["v"], out["d1"], out["kappa_bar"])
        dlo_get_position_residual(self.h, out["x_lo"])
        return out

    def state_adjoint(self):
        """adjoint of the rollout's whole start state after backward() (g_x, g_v, g_d1, g_kappa_bar)"""
        torch = self.torch
        B, N = self.B, self.N
        out = {"g_x": torch.empty((B, 3, N), device=self.dev), "g_v": torch.empty((B, 3, N), device=self.dev),
               "g_d1": torch.empty((B, 3, N), device=self.dev), "g_kappa_bar": torch.empty((B, 2, N), device=self.dev)}
        dlo_get_state_adjoint(self.h, out["g_x"], out["g_v"], out["g_d1"], out["g_kappa_bar"])
        torch.cuda.synchronize(self.dev)
        return {k: t.double().cpu().numpy() for k, t in out.items()}

    def rollout(self, horizon=None, stride=None):
        H = self.H if horizon is None else int(horizon)
        s = self.stride if stride is None else int(stride)
        dlo_rollout_forward(self.h, H, s)
        self.H_done = H
        return self

    def state(self):
        torch = self.torch
        B, N = self.B, self.N
        x, v, d1 = (torch.empty((B, 3, N), device=self.dev) for _ in range(3))
        kb = torch.empty((B, 2, N), device=self.dev)
        xl = torch.empty((B, 3, N), device=self.dev)
        dlo_get_state(self.h, x, v, d1, kb)
        dlo_get_position_residual(self.h, xl)
        torch.cuda.synchronize(self.dev)
        # positions as the library carries them: x + x_lo, summed in fp64
        return {"x": (x.double() + xl.double()).cpu().numpy(), "v": v.double().cpu().numpy(), "d1": d1.double().cpu().numpy(),
                "kappa_bar": kb.double().cpu().numpy()}

    def backward(self, dL_dxT=None, dL_dvT=None):
        torch = self.torch
        B, N, G, H = self.B, self.N, self.G, self.H_done
        gx = None if dL_dxT is None else self._up(dL_dxT)
        gv = None if dL_dvT is None else self._up(dL_dvT)
        out = {"g_actions": torch.zeros((H, B, max(G, 0), 6), device=self.dev), "g_x0": torch.zeros((B, 3, N), device=self.dev),
               "g_v0": torch.zeros((B, 3, N), device=self.dev), "g_material": torch.zeros((B, 5), device=self.dev)}
        dlo_backward(self.h, gx, gv, out["g_actions"] if G > 0 else None, out["g_x0"], out["g_v0"], out["g_material"])
        torch.cuda.synchronize(self.dev)
        return {k: t.double().cpu().numpy() for k, t in out.items()}

    def n_bad(self):
        return dlo_check_numerics(self.h)

    def close(self):
        if getattr(self, "h", None):
            dlo_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
