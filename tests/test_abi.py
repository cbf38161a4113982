"""-m "not gpu": the C-ABI library loads, exports every symbol include/r360.h declares, and its
host-side argument checks work without a CUDA device (no compute calls)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def r360():
    import __graft_entry__ as g
    g.build()
    import paper_2208_02705_b200 as m
    return m


def test_every_declared_symbol_is_exported(r360):
    hdr = open(os.path.join(ROOT, "include", "r360.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    names = set(re.findall(r"\b(r360_[a-z_0-9]+)\s*\(", hdr))
    assert {"r360_scene_create", "r360_render", "r360_scene_destroy", "r360_render_batch",
            "r360_render_batch_host", "r360_set_precision", "r360_set_stream", "r360_get_stats",
            "r360_debug_samples", "r360_status_string"} <= names
    L = C.CDLL(r360.lib_path())
    for n in names:
        assert hasattr(L, n), n
    assert "sm_100a" in r360.version()


def test_params_per_subfield(r360):
    assert r360.params_per_subfield(hidden_width=32, n_hidden=2) == 6212
    assert r360.params_per_subfield(hidden_width=32, n_hidden=3) == 7268
    assert r360.params_per_subfield(hidden_width=64, n_hidden=3) == 22724
    assert r360.params_per_subfield(hidden_width=48, n_hidden=3) == 0          # unsupported width


def _args(P=6212):
    return dict(occupancy=np.full(8, 255, np.uint8), voxel_subfield=np.zeros(8, np.int32),
                weights=np.zeros(P, np.float32), dims=(2, 2, 2), box_min=(0, 0, 0), box_max=(1, 1, 1),
                n_subfields=1, occ_threshold=128)


@pytest.mark.parametrize("bad,status", [
    (dict(dims=(0, 2, 2)), 1), (dict(box_max=(1, 0, 1)), 1), (dict(n_subfields=0), 1),
    (dict(hidden_width=48), 1), (dict(samples_per_voxel=0), 1), (dict(samples_per_voxel=129), 1),
    (dict(t_threshold=float("nan")), 1), (dict(t_threshold=-1.0), 1), (dict(occ_threshold=0), 1),
    (dict(voxel_subfield=np.ones(8, np.int32)), 2), (dict(voxel_subfield=-np.ones(8, np.int32)), 2),
])
def test_scene_create_rejects_before_touching_cuda(r360, bad, status):
    kw = _args()
    kw.update(bad)
    if "dims" in bad:
        kw["occupancy"] = np.zeros(0, np.uint8)
        kw["voxel_subfield"] = np.zeros(0, np.int32)
    with pytest.raises(r360.R360Error) as e:
        r360.Scene(**kw)
    assert e.value.status == status


def test_scene_create_rejects_nonfinite_weights(r360):
    kw = _args()
    kw["weights"][100] = np.inf
    with pytest.raises(r360.R360Error) as e:
        r360.Scene(**kw)
    assert e.value.status == 3


def test_null_handles(r360):
    L = r360.lib()
    L.r360_scene_destroy(None)                                   # NULL is a no-op
    assert L.r360_set_precision(None, 0) == 1
    assert L.r360_render(None, None, 4, 2, None, None) == 1
    assert L.r360_status_string(2).decode().startswith("occupied voxel")
