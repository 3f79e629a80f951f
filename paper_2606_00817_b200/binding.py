"""ctypes binding of libddf.so - same names as include/ddf.h, argument marshalling only.

Tensors are torch CUDA tensors (float32, contiguous); the stream defaults to torch's current
stream.  Nothing here computes: a missing library or device raises DdfError.
"""
import ctypes as C
import os

import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB_PATH = os.path.join(_HERE, "libddf.so")

EXPORTED_SYMBOLS = [
    "ddf_create", "ddf_destroy", "ddf_status_string", "ddf_last_cuda_error", "ddf_set_path",
    "ddf_get_info", "ddf_reserve", "ddf_query", "ddf_query_host", "ddf_query_logits", "ddf_camera_from_seed",
    "ddf_gen_camera", "ddf_gen_sphere_points", "ddf_gen_shadow", "ddf_gen_gbuffer", "ddf_gen_ao",
    "ddf_ao_reduce", "ddf_query_ao", "ddf_shadow_test", "sdf_sphere_trace",
    "ddf_hashgrid_table_entries", "ddf_create_hashgrid", "ddf_gen_shadow_from_hits", "ddf_query_shadowed", "ddf_query_shadowed_lights",
    "ddf_gen_ao_from_hits", "ddf_query_ao_wavefront", "ddf_query_shaded", "ddf_query_ao_points",
    "ddf_trainer_create", "ddf_trainer_destroy", "ddf_trainer_step", "ddf_trainer_loss_grads", "ddf_trainer_export",
    "ddf_trainer_steps", "ddf_scene_raycast", "ddf_gen_train_batch", "ddf_query_camera",
    "ddf_gen_shadow_from_hits_static",
]


class DdfError(RuntimeError):
    pass


class DdfLayout(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("version", C.c_uint32), ("input_kind", C.c_uint32),
                ("n_freq_origin", C.c_uint32), ("n_freq_dir", C.c_uint32), ("n_hidden", C.c_uint32),
                ("width", C.c_uint32), ("skip_layer", C.c_int32), ("n_out", C.c_uint32),
                ("weight_dtype", C.c_uint32), ("weights_on_device", C.c_uint32)]


class DdfHashgridLayout(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("version", C.c_uint32), ("n_levels", C.c_uint32),
                ("n_features", C.c_uint32), ("log2_table_size", C.c_uint32), ("base_resolution", C.c_uint32),
                ("growth", C.c_float), ("box_min", C.c_float * 3), ("box_max", C.c_float * 3),
                ("n_freq_dir", C.c_uint32), ("n_hidden", C.c_uint32), ("width", C.c_uint32), ("n_out", C.c_uint32),
                ("table_dtype", C.c_uint32), ("mlp_dtype", C.c_uint32), ("weights_on_device", C.c_uint32)]


class DdfTrainParams(C.Structure):
    _fields_ = [("struct_size", C.c_uint32), ("lr0", C.c_float), ("lr_final_frac", C.c_float), ("total_steps", C.c_int32),
                ("beta1", C.c_float), ("beta2", C.c_float), ("adam_eps", C.c_float), ("dist_clamp", C.c_float),
                ("ce_weight", C.c_float), ("arithmetic", C.c_uint32)]


class DdfCamera(C.Structure):
    _fields_ = [("pos", C.c_float * 3), ("look_at", C.c_float * 3), ("fov_deg", C.c_float)]


class DdfScene(C.Structure):
    _fields_ = [("sphere_c", C.c_float * 3), ("sphere_r", C.c_float),
                ("box_min", C.c_float * 3), ("box_max", C.c_float * 3)]


class SdfTraceParams(C.Structure):
    _fields_ = [("max_steps", C.c_int32), ("eps", C.c_float), ("t_max", C.c_float),
                ("base_radius", C.c_float), ("alpha", C.c_float), ("early_exit", C.c_int32), ("omega", C.c_float)]


_lib = None


def lib_path():
    return _LIB_PATH


def lib():
    """Loads libddf.so (built in-tree by paper_2606_00817_b200.build.build()); fails loudly."""
    global _lib
    if _lib is None:
        if not os.path.exists(_LIB_PATH):
            raise DdfError("libddf.so is not built: run `python -m paper_2606_00817_b200.build` "
                           "(there is no CPU or PyTorch fallback)")
        _lib = C.CDLL(_LIB_PATH)
        _lib.ddf_status_string.restype = C.c_char_p
        _lib.ddf_get_info.restype = C.c_int64
        _lib.ddf_hashgrid_table_entries.restype = C.c_int64
        _lib.ddf_trainer_steps.restype = C.c_int64
    return _lib


def ddf_status_string(rc):
    return lib().ddf_status_string(C.c_int(rc)).decode()


def _check(rc, what):
    if rc != 0:
        extra = ""
        if rc == -4:
            extra = " (cudaError %d)" % lib().ddf_last_cuda_error()
        raise DdfError("%s failed: %s%s" % (what, ddf_status_string(rc), extra))


def _stream(stream):
    if stream is None:
        stream = torch.cuda.current_stream()
    return C.c_void_p(stream.cuda_stream if hasattr(stream, "cuda_stream") else int(stream))


def _dev(t, dtype=torch.float32):
    if t is None:
        return C.c_void_p(0)
    if not (t.is_cuda and t.is_contiguous() and t.dtype == dtype):
        raise DdfError("expected a contiguous CUDA tensor of %s" % dtype)
    return C.c_void_p(t.data_ptr())


def _host(t, dtype=torch.float32):
    if t is None:
        return C.c_void_p(0)
    if t.is_cuda or not t.is_contiguous() or t.dtype != dtype:
        raise DdfError("expected a contiguous host tensor of %s" % dtype)
    return C.c_void_p(t.data_ptr())


class Model:
    """Owns a ddf_model*; see ddf_create."""

    def __init__(self, handle, layout):
        self.handle = handle
        self.layout = layout

    def close(self):
        if self.handle:
            ddf_destroy(self)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def make_layout(lay, weights_on_device=0):
    """lay: any object with the ddf_layout field names (e.g. ddf_inputs.Layout)."""
    return DdfLayout(C.sizeof(DdfLayout), 1, lay.input_kind, lay.n_freq_origin, lay.n_freq_dir, lay.n_hidden,
                     lay.width, lay.skip_layer, lay.n_out, lay.weight_dtype, weights_on_device)


def ddf_create(weights, lay):
    """weights: numpy array (float32 / uint16 bf16 bits) or a CUDA tensor of the blob."""
    import numpy as np
    if isinstance(weights, torch.Tensor):
        L = make_layout(lay, 1 if weights.is_cuda else 0)
        ptr = C.c_void_p(weights.data_ptr())
    else:
        weights = np.ascontiguousarray(weights)
        L = make_layout(lay, 0)
        ptr = weights.ctypes.data_as(C.c_void_p)
    h = C.c_void_p(0)
    _check(lib().ddf_create(ptr, C.byref(L), C.byref(h)), "ddf_create")
    return Model(h, lay)


def make_hashgrid_layout(lay, weights_on_device=0):
    """lay: any object with the ddf_hashgrid_layout field names (e.g. ddf_inputs.HashLayout)."""
    return DdfHashgridLayout(C.sizeof(DdfHashgridLayout), 1, lay.n_levels, lay.n_features, lay.log2_table,
                             lay.base_res, float(lay.growth), (C.c_float * 3)(*lay.box_min),
                             (C.c_float * 3)(*lay.box_max), lay.n_freq_dir, lay.n_hidden, lay.width, lay.n_out,
                             lay.table_dtype, lay.mlp_dtype, weights_on_device)


def ddf_hashgrid_table_entries(lay):
    L = make_hashgrid_layout(lay)
    n = int(lib().ddf_hashgrid_table_entries(C.byref(L)))
    if n < 0:
        _check(n, "ddf_hashgrid_table_entries")
    return n


def ddf_create_hashgrid(table, mlp, lay):
    """table, mlp: numpy arrays (host) or CUDA tensors (both on the device)."""
    import numpy as np
    if isinstance(table, torch.Tensor):
        if not (table.is_cuda and isinstance(mlp, torch.Tensor) and mlp.is_cuda):
            raise DdfError("table and mlp must both be host arrays or both CUDA tensors")
        L = make_hashgrid_layout(lay, 1)
        pt, pm = C.c_void_p(table.data_ptr()), C.c_void_p(mlp.data_ptr())
    else:
        table, mlp = np.ascontiguousarray(table), np.ascontiguousarray(mlp)
        L = make_hashgrid_layout(lay, 0)
        pt, pm = table.ctypes.data_as(C.c_void_p), mlp.ctypes.data_as(C.c_void_p)
    h = C.c_void_p(0)
    _check(lib().ddf_create_hashgrid(pt, pm, C.byref(L), C.byref(h)), "ddf_create_hashgrid")
    return Model(h, lay)


def ddf_destroy(model):
    if model.handle:
        rc = lib().ddf_destroy(model.handle)
        model.handle = None
        _check(rc, "ddf_destroy")


RESERVE_HOST, RESERVE_RAYS, RESERVE_TRACE, RESERVE_WAVE, RESERVE_ALL = 1, 2, 4, 8, 15


def ddf_reserve(model, what, max_rays, spp=0):
    _check(lib().ddf_reserve(model.handle, C.c_uint32(what), C.c_int64(max_rays), C.c_int(spp)), "ddf_reserve")


def ddf_set_path(model, path):
    _check(lib().ddf_set_path(model.handle, C.c_int(path)), "ddf_set_path")


def ddf_get_info(model, which):
    return int(lib().ddf_get_info(model.handle, C.c_int(which)))


def ddf_query(model, origins, dirs, n, out_dist, out_vis, stream=None):
    _check(lib().ddf_query(model.handle, _dev(origins), _dev(dirs), C.c_int64(n), _dev(out_dist), _dev(out_vis),
                           _stream(stream)), "ddf_query")


def ddf_query_host(model, origins, dirs, n, out_dist, out_vis, stream=None):
    _check(lib().ddf_query_host(model.handle, _host(origins), _host(dirs), C.c_int64(n), _host(out_dist),
                                _host(out_vis), _stream(stream)), "ddf_query_host")


def ddf_query_logits(model, origins, dirs, n, out_z, stream=None):
    _check(lib().ddf_query_logits(model.handle, _dev(origins), _dev(dirs), C.c_int64(n), _dev(out_z),
                                  _stream(stream)), "ddf_query_logits")


def ddf_query_ao(model, o, d, n_pts, spp, ao_radius, ao, stream=None):
    _check(lib().ddf_query_ao(model.handle, _dev(o), _dev(d), C.c_int64(n_pts), C.c_int(spp), C.c_float(ao_radius),
                              _dev(ao), _stream(stream)), "ddf_query_ao")


def ddf_camera_from_seed(seed, rng_stream, radius=2.5):
    cam = DdfCamera()
    _check(lib().ddf_camera_from_seed(C.c_uint64(seed), C.c_uint64(rng_stream), C.c_float(radius), C.byref(cam)),
           "ddf_camera_from_seed")
    return cam


def ddf_gen_camera(cam, width, height, o, d, stream=None):
    _check(lib().ddf_gen_camera(C.byref(cam), C.c_int(width), C.c_int(height), _dev(o), _dev(d), _stream(stream)),
           "ddf_gen_camera")


def ddf_gen_sphere_points(seed, rng_stream, n, radius, p, nrm, stream=None):
    _check(lib().ddf_gen_sphere_points(C.c_uint64(seed), C.c_uint64(rng_stream), C.c_int64(n), C.c_float(radius),
                                       _dev(p), _dev(nrm), _stream(stream)), "ddf_gen_sphere_points")


def ddf_gen_shadow(p, nrm, n, light, eps, o, d, tmax, stream=None):
    li = (C.c_float * 3)(*[float(x) for x in light])
    _check(lib().ddf_gen_shadow(_dev(p), _dev(nrm), C.c_int64(n), li, C.c_float(eps), _dev(o), _dev(d), _dev(tmax),
                                _stream(stream)), "ddf_gen_shadow")


def ddf_gen_gbuffer(cam, scene, width, height, p, nrm, t_hit, stream=None):
    _check(lib().ddf_gen_gbuffer(C.byref(cam), C.byref(scene), C.c_int(width), C.c_int(height), _dev(p), _dev(nrm),
                                 _dev(t_hit), _stream(stream)), "ddf_gen_gbuffer")


def ddf_gen_ao(p, nrm, n_pts, spp, seed, rng_stream, eps, o, d, stream=None):
    _check(lib().ddf_gen_ao(_dev(p), _dev(nrm), C.c_int64(n_pts), C.c_int(spp), C.c_uint64(seed),
                            C.c_uint64(rng_stream), C.c_float(eps), _dev(o), _dev(d), _stream(stream)), "ddf_gen_ao")


def ddf_ao_reduce(vis, dist, n_pts, spp, ao_radius, ao, stream=None):
    _check(lib().ddf_ao_reduce(_dev(vis), _dev(dist), C.c_int64(n_pts), C.c_int(spp), C.c_float(ao_radius), _dev(ao),
                               _stream(stream)), "ddf_ao_reduce")


def ddf_shadow_test(vis, dist, tmax, n, shadow, stream=None):
    _check(lib().ddf_shadow_test(_dev(vis), _dev(dist), _dev(tmax), C.c_int64(n), _dev(shadow, torch.uint8),
                                 _stream(stream)), "ddf_shadow_test")


def sdf_sphere_trace(model, o, d, n, params, out_t, out_hit, out_steps, trace_p=None, trace_s=None,
                     total_evals=None, stream=None):
    _check(lib().sdf_sphere_trace(model.handle, _dev(o), _dev(d), C.c_int64(n), C.byref(params), _dev(out_t),
                                  _dev(out_hit, torch.uint8), _dev(out_steps, torch.int32), _dev(trace_p),
                                  _dev(trace_s), _dev(total_evals, torch.int64), _stream(stream)),
           "sdf_sphere_trace")


def ddf_gen_shadow_from_hits(model, o, d, dist, vis, n, light, eps, o2, d2, tmax, index, count, stream=None):
    li = (C.c_float * 3)(*[float(x) for x in light])
    _check(lib().ddf_gen_shadow_from_hits(model.handle, _dev(o), _dev(d), _dev(dist), _dev(vis), C.c_int64(n), li,
                                          C.c_float(eps), _dev(o2), _dev(d2), _dev(tmax), _dev(index, torch.int32),
                                          _dev(count, torch.int64), _stream(stream)), "ddf_gen_shadow_from_hits")


STATIC_MAX_RAYS = 1 << 24


def ddf_gen_shadow_from_hits_static(o, d, dist, vis, n, light, eps, o2, d2, tmax, index, count, stream=None):
    """ddf_gen_shadow_from_hits without a model and without any device allocation: for programs whose own pool
    already holds all device memory, or that cannot afford the stall of a cudaMalloc inside a frame.  The
    compaction's scratch is a fixed array inside libddf.so, so n is limited to STATIC_MAX_RAYS (DdfError beyond it),
    the first call on a device should be made at start-up, and calls must not overlap on the GPU (one stream, or
    streams ordered by events).  Same results, bit for bit, as ddf_gen_shadow_from_hits."""
    li = (C.c_float * 3)(*[float(x) for x in light])
    _check(lib().ddf_gen_shadow_from_hits_static(_dev(o), _dev(d), _dev(dist), _dev(vis), C.c_int64(n), li,
                                                 C.c_float(eps), _dev(o2), _dev(d2), _dev(tmax), _dev(index, torch.int32),
                                                 _dev(count, torch.int64), _stream(stream)), "ddf_gen_shadow_from_hits_static")


def ddf_query_shadowed(model, o, d, n, light, eps, out_dist, out_vis, out_lit, out_count=None, stream=None):
    li = (C.c_float * 3)(*[float(x) for x in light])
    _check(lib().ddf_query_shadowed(model.handle, _dev(o), _dev(d), C.c_int64(n), li, C.c_float(eps), _dev(out_dist),
                                    _dev(out_vis), _dev(out_lit, torch.uint8), _dev(out_count, torch.int64),
                                    _stream(stream)), "ddf_query_shadowed")


def ddf_query_shadowed_lights(model, o, d, n, lights, eps, out_dist, out_vis, out_lit_mask, out_count=None, stream=None):
    flat = [float(x) for l in lights for x in l]
    li = (C.c_float * len(flat))(*flat)
    _check(lib().ddf_query_shadowed_lights(model.handle, _dev(o), _dev(d), C.c_int64(n), li, C.c_int(len(flat) // 3), C.c_float(eps),
                                           _dev(out_dist), _dev(out_vis), _dev(out_lit_mask, torch.uint8),
                                           _dev(out_count, torch.int64), _stream(stream)), "ddf_query_shadowed_lights")


def ddf_query_ao_points(model, p, nrm, n_pts, spp, seed, rng_stream, eps, ao_radius, ao, stream=None):
    _check(lib().ddf_query_ao_points(model.handle, _dev(p), _dev(nrm), C.c_int64(n_pts), C.c_int(spp), C.c_uint64(int(seed)),
                                     C.c_uint64(int(rng_stream)), C.c_float(eps), C.c_float(ao_radius), _dev(ao),
                                     _stream(stream)), "ddf_query_ao_points")


def ddf_gen_ao_from_hits(model, o, d, dist, vis, width, height, spp, seed, rng_stream, eps, p_c, nrm_c, index, o2, d2, count,
                         stream=None):
    _check(lib().ddf_gen_ao_from_hits(model.handle, _dev(o), _dev(d), _dev(dist), _dev(vis), C.c_int(width), C.c_int(height),
                                      C.c_int(spp), C.c_uint64(int(seed)), C.c_uint64(int(rng_stream)), C.c_float(eps),
                                      _dev(p_c), _dev(nrm_c), _dev(index, torch.int32), _dev(o2), _dev(d2),
                                      _dev(count, torch.int64), _stream(stream)), "ddf_gen_ao_from_hits")


def ddf_query_ao_wavefront(model, o, d, width, height, spp, seed, rng_stream, eps, ao_radius, out_dist, out_vis, out_nrm,
                           out_ao, out_count=None, stream=None):
    _check(lib().ddf_query_ao_wavefront(model.handle, _dev(o), _dev(d), C.c_int(width), C.c_int(height), C.c_int(spp),
                                        C.c_uint64(int(seed)), C.c_uint64(int(rng_stream)), C.c_float(eps),
                                        C.c_float(ao_radius), _dev(out_dist), _dev(out_vis), _dev(out_nrm), _dev(out_ao),
                                        _dev(out_count, torch.int64), _stream(stream)), "ddf_query_ao_wavefront")


def ddf_query_shaded(model, o, d, width, height, lights, spp, seed, rng_stream, eps, ao_radius, out_dist, out_vis, out_lit_mask,
                     out_nrm, out_ao, out_counts=None, stream=None):
    flat = [float(x) for l in lights for x in l]
    li = (C.c_float * max(len(flat), 1))(*flat)
    _check(lib().ddf_query_shaded(model.handle, _dev(o), _dev(d), C.c_int(width), C.c_int(height), li, C.c_int(len(flat) // 3),
                                  C.c_int(spp), C.c_uint64(int(seed)), C.c_uint64(int(rng_stream)), C.c_float(eps),
                                  C.c_float(ao_radius), _dev(out_dist), _dev(out_vis), _dev(out_lit_mask, torch.uint8),
                                  _dev(out_nrm), _dev(out_ao), _dev(out_counts, torch.int64), _stream(stream)), "ddf_query_shaded")


# ------------------------------------------------------------------ training

def make_train_params(lr0=3e-3, lr_final_frac=0.05, total_steps=30000, beta1=0.9, beta2=0.999, adam_eps=1e-8,
                      dist_clamp=6.0, ce_weight=0.3, arithmetic=0):
    """arithmetic: DDF_TRAIN_BF16X3 (0, tensor cores) or DDF_TRAIN_FP32 (1, CUDA cores); include/ddf.h."""
    return DdfTrainParams(C.sizeof(DdfTrainParams), lr0, lr_final_frac, total_steps, beta1, beta2, adam_eps, dist_clamp,
                          ce_weight, arithmetic)


class Trainer:
    def __init__(self, handle, layout):
        self.handle, self.layout = handle, layout

    def __del__(self):
        try:
            if self.handle:
                ddf_trainer_destroy(self)
        except Exception:
            pass


def ddf_trainer_create(table, mlp, lay, params):
    import numpy as np
    table = np.ascontiguousarray(table, dtype=np.float32); mlp = np.ascontiguousarray(mlp, dtype=np.float32)
    L = make_hashgrid_layout(lay, 0)
    h = C.c_void_p(0)
    _check(lib().ddf_trainer_create(table.ctypes.data_as(C.c_void_p), mlp.ctypes.data_as(C.c_void_p), C.byref(L),
                                    C.byref(params), C.byref(h)), "ddf_trainer_create")
    return Trainer(h, lay)


def ddf_trainer_destroy(tr):
    if tr.handle:
        rc = lib().ddf_trainer_destroy(tr.handle)
        tr.handle = None
        _check(rc, "ddf_trainer_destroy")


def ddf_trainer_step(tr, o, d, t, hit, n, loss=None, stream=None):
    _check(lib().ddf_trainer_step(tr.handle, _dev(o), _dev(d), _dev(t), _dev(hit, torch.uint8), C.c_int64(n), _dev(loss),
                                  _stream(stream)), "ddf_trainer_step")


def ddf_trainer_loss_grads(tr, o, d, t, hit, n, loss, grad_table, grad_mlp, stream=None):
    _check(lib().ddf_trainer_loss_grads(tr.handle, _dev(o), _dev(d), _dev(t), _dev(hit, torch.uint8), C.c_int64(n), _dev(loss),
                                        _dev(grad_table), _dev(grad_mlp), _stream(stream)), "ddf_trainer_loss_grads")


def ddf_trainer_export(tr, n_table, n_mlp):
    """Returns (table, mlp) as float32 numpy arrays."""
    import numpy as np
    table = np.empty(n_table, np.float32); mlp = np.empty(n_mlp, np.float32)
    _check(lib().ddf_trainer_export(tr.handle, table.ctypes.data_as(C.c_void_p), mlp.ctypes.data_as(C.c_void_p)),
           "ddf_trainer_export")
    return table, mlp


def ddf_trainer_steps(tr):
    return int(lib().ddf_trainer_steps(tr.handle))


def ddf_scene_raycast(scene, o, d, n, t, hit, stream=None):
    _check(lib().ddf_scene_raycast(C.byref(scene), _dev(o), _dev(d), C.c_int64(n), _dev(t), _dev(hit, torch.uint8),
                                   _stream(stream)), "ddf_scene_raycast")


def ddf_gen_train_batch(scene, seed, rng_stream, step, n, sample_half, o, d, t, hit, stream=None):
    _check(lib().ddf_gen_train_batch(C.byref(scene), C.c_uint64(seed), C.c_uint64(rng_stream), C.c_int64(step), C.c_int64(n),
                                     C.c_float(sample_half), _dev(o), _dev(d), _dev(t), _dev(hit, torch.uint8),
                                     _stream(stream)), "ddf_gen_train_batch")


def ddf_query_camera(model, cam, width, height, out_dist, out_vis, stream=None):
    _check(lib().ddf_query_camera(model.handle, C.byref(cam), C.c_int(width), C.c_int(height), _dev(out_dist), _dev(out_vis),
                                  _stream(stream)), "ddf_query_camera")
