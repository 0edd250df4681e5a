"""C-ABI boundary (include/dlo.h): the library builds for sm_100a, loads, exports every declared symbol, and its
host-side argument checks work without a GPU.  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from workloads.configs import make_problem

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def dlo():
    import paper_2606_04206_b200 as pkg
    pkg.lib()
    return pkg


def declared_symbols():
    src = open(os.path.join(ROOT, "include", "dlo.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(dlo_[a-z0-9_]+)\s*\(", src)))


def test_every_declared_symbol_is_exported(dlo):
    names = declared_symbols()
    assert len(names) >= 20
    L = dlo.lib()
    for n in names:
        assert hasattr(L, n), n
    assert sorted(dlo.EXPORTS) == names


def test_version_and_struct_sizes(dlo):
    assert "sm_100a" in dlo.dlo_version()
    assert C.sizeof(dlo.DloConfig) == 13 * 4 + 8 * 4
    assert C.sizeof(dlo.DloMaterial) == 9 * C.sizeof(C.c_void_p)


def test_scratch_bytes_matches_layout(dlo):
    from paper_2606_04206_b200.binding import make_config
    P = make_problem(5)
    cfg = make_config(P["config"])
    B, N, H, S = 4096, 128, 1000, 100
    blk = 14 * N * 4                    # x, v, d1 (3 rows each), kappa_bar (2), position residual x_lo (3)
    n = dlo.dlo_scratch_bytes(cfg, H, S)
    ckpt, tape = (H // S + 1) * B * blk, 2 * (S * 5 + 1) * B * (22 + 10) * N * 4     # two tape buffers of 22 + N_C rows per record (14 state, dx 3, v1 3, S, mask)
    # two side-record pools (one substep in twelve; header, v^1, 480 candidate codes and depth sums, N_C x 3 x 132 corrections)
    side = 2 * ((S * 5 + 1) * B // 12) * (4 + 3 * N + 240 + 480 + 10 * 3 * 132) * 4
    assert n > ckpt + tape + side and n < ckpt + tape + side + 450e6
    assert dlo.dlo_scratch_bytes(cfg, H, 0) < 100e6          # forward only: constants + two state copies
    bad = make_config(dict(P["config"], n_verts=1000))
    assert dlo.dlo_scratch_bytes(bad, H, S) == 0


@pytest.mark.parametrize("field,value", [("n_verts", 2), ("n_verts", 257), ("batch", 0), ("topology", 7), ("n_substeps", 0),
                                         ("n_grippers", 5), ("n_primitives", 17), ("dt", 0.0), ("stretch_mode", 3)])
def test_create_rejects_bad_config_without_touching_the_gpu(dlo, field, value):
    from paper_2606_04206_b200.binding import make_config
    cfg = make_config(dict(make_problem(1)["config"], **{field: value}))
    m = dlo.DloMaterial()
    h = C.c_void_p()
    st = dlo.lib().dlo_create(C.byref(cfg), C.byref(m), None, C.byref(h))
    assert st == -1 and h.value is None
    assert dlo.dlo_last_error()


def test_create_without_device_fails_loudly(dlo):
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2606_04206_b200.binding import make_config
    cfg = make_config(make_problem(1)["config"])
    m = dlo.DloMaterial()
    one = np.ones(1, dtype=np.float32)
    for k, _ in dlo.DloMaterial._fields_:
        setattr(m, k, one.ctypes.data)
    h = C.c_void_p()
    st = dlo.lib().dlo_create(C.byref(cfg), C.byref(m), None, C.byref(h))
    assert st == -3 and "no CPU path" in dlo.dlo_last_error()
    with pytest.raises(dlo.DloError):
        dlo.DloSim(make_problem(1))


def test_null_handle_is_an_error_not_a_crash(dlo):
    L = dlo.lib()
    assert L.dlo_rollout_forward(None, 1, 0) == -1
    assert L.dlo_backward(None, None, None, None, None, None, None) == -1
    assert L.dlo_destroy(None) == 0
