"""The C-ABI library loads and exports every symbol include/ddf.h declares; argument checks that
need no GPU (host logic).  No compute call is made here."""
import ctypes as C
import os
import re

import numpy as np
import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def libddf():
    from paper_2606_00817_b200 import build, lib
    build()
    return lib()


def _declared_symbols():
    src = open(os.path.join(ROOT, "include", "ddf.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    names = re.findall(r"\b((?:ddf|sdf)_[a-z_0-9]+)\s*\(", src)
    return sorted(set(names))


def test_every_declared_symbol_is_exported(libddf):
    from paper_2606_00817_b200 import EXPORTED_SYMBOLS
    decl = _declared_symbols()
    assert len(decl) >= 19
    for name in decl:
        assert hasattr(libddf, name), name
    assert sorted(EXPORTED_SYMBOLS) == decl


def test_binding_mirrors_the_header():
    import paper_2606_00817_b200 as pkg
    for name in _declared_symbols():
        if name in ("ddf_last_cuda_error",):
            continue
        assert hasattr(pkg, name), name


def test_status_strings(libddf):
    from paper_2606_00817_b200 import ddf_status_string
    assert ddf_status_string(0) == "ok"
    assert ddf_status_string(-1) == "invalid argument"
    assert ddf_status_string(-2) == "bad layout"
    assert "unknown" in ddf_status_string(-99)


def test_layout_struct_matches_header():
    from paper_2606_00817_b200 import DdfLayout, DdfCamera, DdfScene, SdfTraceParams
    assert C.sizeof(DdfLayout) == 44 and C.sizeof(DdfCamera) == 28 and C.sizeof(DdfScene) == 40
    assert C.sizeof(SdfTraceParams) == 28


def test_argument_errors_without_gpu(libddf):
    from paper_2606_00817_b200 import DdfLayout, DdfCamera
    h = C.c_void_p(0)
    assert libddf.ddf_create(None, None, C.byref(h)) == -1
    bad = DdfLayout(44, 99, 0, 4, 4, 3, 64, -1, 2, 0, 0)                 # wrong version
    w = np.zeros(16, np.float32)
    assert libddf.ddf_create(w.ctypes.data_as(C.c_void_p), C.byref(bad), C.byref(h)) == -2
    bad = DdfLayout(44, 1, 0, 4, 4, 3, 64, 3, 2, 0, 0)                   # skip_layer out of range
    assert libddf.ddf_create(w.ctypes.data_as(C.c_void_p), C.byref(bad), C.byref(h)) == -2
    bad = DdfLayout(44, 1, 0, 4, 4, 3, 64, -1, 3, 0, 0)                  # n_out
    assert libddf.ddf_create(w.ctypes.data_as(C.c_void_p), C.byref(bad), C.byref(h)) == -2
    assert libddf.ddf_destroy(None) == 0
    assert libddf.ddf_query(None, None, None, C.c_int64(0), None, None, None) == -1
    assert libddf.ddf_gen_camera(None, 4, 4, None, None, None) == -1
    cam = DdfCamera()
    assert libddf.ddf_gen_camera(C.byref(cam), 0, 0, None, None, None) == 0     # n == 0 is a no-op
    assert libddf.ddf_gen_sphere_points(C.c_uint64(1), C.c_uint64(1), C.c_int64(-1), C.c_float(1), None, None, None) == -1
    assert libddf.ddf_ao_reduce(None, None, C.c_int64(0), 16, C.c_float(1), None, None) == 0
    assert libddf.ddf_ao_reduce(None, None, C.c_int64(4), 0, C.c_float(1), None, None) == -1
    assert libddf.ddf_reserve(None, C.c_uint32(1), C.c_int64(16), 0) == -1
    assert libddf.ddf_query_ao(None, None, None, C.c_int64(1 << 30), 16, C.c_float(1), None, None) == -1


def test_camera_from_seed_matches_oracle_twin(libddf, orc):
    from ddf_inputs import MASTER_SEED, STREAMS
    from paper_2606_00817_b200 import ddf_camera_from_seed
    cam = ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    want = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    assert np.allclose(list(cam.pos), list(want.pos), atol=3e-7)
    assert cam.fov_deg == 50.0 and list(cam.look_at) == [0, 0, 0]


def test_no_gpu_means_loud_failure(libddf):
    """Without a CUDA device ddf_create must fail (no CPU fallback)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from ddf_inputs import layout_c0, make_weights
    from paper_2606_00817_b200 import ddf_create, DdfError
    with pytest.raises(DdfError):
        ddf_create(make_weights(layout_c0()), layout_c0())


def test_product_does_not_import_oracle():
    pkg = os.path.join(ROOT, "paper_2606_00817_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                src = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in src and "from oracle" not in src and "ddf_oracle" not in src, f
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c", ".h")):
            src = open(os.path.join(ROOT, "oracle", f)).read()
            assert "paper_2606_00817_b200" not in src.replace("under paper_2606_00817_b200/", "").replace(
                "the product (paper_2606_00817_b200)", ""), f


def test_hashgrid_host_logic_without_gpu(libddf, orc):
    """Level sizing of the hash-grid field is host logic: the library's count must be
    the paper's 6,529,022 entries (13.06M parameters) and agree with the oracle on other shapes."""
    from ddf_inputs import HashLayout, layout_hash_paper
    from paper_2606_00817_b200 import DdfHashgridLayout, make_hashgrid_layout, ddf_hashgrid_table_entries, DdfError
    assert C.sizeof(DdfHashgridLayout) == 80
    assert ddf_hashgrid_table_entries(layout_hash_paper()) == 6_529_022
    for lay in (HashLayout(n_levels=5, base_res=3, growth=2.0, log2_table=10), HashLayout(n_levels=12, growth=1.3819, log2_table=14)):
        assert ddf_hashgrid_table_entries(lay) == orc.hash_table_entries(lay)
    bad = make_hashgrid_layout(layout_hash_paper()); bad.version = 7
    assert libddf.ddf_hashgrid_table_entries(C.byref(bad)) == -2
    bad = make_hashgrid_layout(HashLayout(box_min=(1.0, 0.0, 0.0), box_max=(1.0, 1.0, 1.0)))
    assert libddf.ddf_hashgrid_table_entries(C.byref(bad)) == -2
    h = C.c_void_p(0)
    assert libddf.ddf_create_hashgrid(None, None, None, C.byref(h)) == -1
    w = np.zeros(16, np.float32)
    wide = make_hashgrid_layout(HashLayout(width=128))                     # shape this build does not serve
    assert libddf.ddf_create_hashgrid(w.ctypes.data_as(C.c_void_p), w.ctypes.data_as(C.c_void_p), C.byref(wide), C.byref(h)) == -3
    with pytest.raises(DdfError):
        ddf_hashgrid_table_entries(HashLayout(n_out=5))


def test_trainer_and_wavefront_argument_errors_without_gpu(libddf):
    """struct sizes and the argument checks of the training / wavefront entry points that run before
    any CUDA call"""
    from ddf_inputs import HashLayout, layout_hash_paper
    from paper_2606_00817_b200 import DdfTrainParams, make_train_params, make_hashgrid_layout, DdfScene
    assert C.sizeof(DdfTrainParams) == 40
    h = C.c_void_p(0)
    w = np.zeros(16, np.float32); wp = w.ctypes.data_as(C.c_void_p)
    L = make_hashgrid_layout(layout_hash_paper()); P = make_train_params()
    assert libddf.ddf_trainer_create(None, wp, C.byref(L), C.byref(P), C.byref(h)) == -1
    bad = make_train_params(); bad.struct_size = 3
    assert libddf.ddf_trainer_create(wp, wp, C.byref(L), C.byref(bad), C.byref(h)) == -2
    assert libddf.ddf_trainer_create(wp, wp, C.byref(L), C.byref(make_train_params(lr0=-1.0)), C.byref(h)) == -1
    assert libddf.ddf_trainer_create(wp, wp, C.byref(L), C.byref(make_train_params(beta2=1.0)), C.byref(h)) == -1
    assert libddf.ddf_trainer_create(wp, wp, C.byref(L), C.byref(make_train_params(arithmetic=2)), C.byref(h)) == -1
    f16 = make_hashgrid_layout(HashLayout(table_dtype=2))                 # training wants fp32 master copies
    assert libddf.ddf_trainer_create(wp, wp, C.byref(f16), C.byref(P), C.byref(h)) == -2
    deep = make_hashgrid_layout(HashLayout(n_hidden=3))
    assert libddf.ddf_trainer_create(wp, wp, C.byref(deep), C.byref(P), C.byref(h)) == -3
    assert libddf.ddf_trainer_destroy(None) == 0 and libddf.ddf_trainer_steps(None) == -1
    assert libddf.ddf_trainer_step(None, None, None, None, None, C.c_int64(4), None, None) == -1
    sc = DdfScene((0.0, 0.0, 0.0), 0.5, (-0.9, -0.9, -0.9), (0.9, 0.9, -0.6))
    assert libddf.ddf_scene_raycast(C.byref(sc), None, None, C.c_int64(0), None, None, None) == 0
    assert libddf.ddf_scene_raycast(C.byref(sc), None, None, C.c_int64(5), None, None, None) == -1
    assert libddf.ddf_gen_train_batch(C.byref(sc), C.c_uint64(1), C.c_uint64(1), C.c_int64(-1), C.c_int64(4), C.c_float(2.0), None, None, None, None, None) == -1
    li = (C.c_float * 3)(1, 2, 3)
    assert libddf.ddf_query_shadowed(None, None, None, C.c_int64(4), li, C.c_float(1e-3), None, None, None, None, None) == -1
    assert libddf.ddf_query_shadowed_lights(None, None, None, C.c_int64(4), li, C.c_int(1), C.c_float(1e-3), None, None, None, None, None) == -1
    assert libddf.ddf_gen_shadow_from_hits(None, None, None, None, None, C.c_int64(4), li, C.c_float(1e-3), None, None, None, None, None, None) == -1
