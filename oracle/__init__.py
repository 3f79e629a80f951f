"""ctypes binding of the CPU oracle (oracle/ddf_oracle.c).  TEST INFRASTRUCTURE, NOT PRODUCT.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this package; the product (paper_2606_00817_b200) never does.  Argument marshalling
only - every number comes from the C file.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "ddf_oracle.c")
_SRCS = [_SRC, os.path.join(_HERE, "ddf_hash_oracle.c")]
_HDRS = [os.path.join(_HERE, "ddf_oracle.h"), os.path.join(_HERE, "ddf_hash_oracle.h")]
_LIB = os.path.join(_HERE, "libddf_oracle.so")


def build(force=False):
    """gcc -O2, OpenMP, no fast-math, no FMA contraction."""
    if (not force and os.path.exists(_LIB)
            and os.path.getmtime(_LIB) >= max(os.path.getmtime(f) for f in _SRCS + _HDRS)):
        return _LIB
    subprocess.check_call(["gcc", "-O2", "-Wall", "-ffp-contract=off", "-fopenmp", "-fPIC", "-shared",
                           "-o", _LIB] + _SRCS + ["-lm"])
    return _LIB


class OrcLayout(C.Structure):
    _fields_ = [(k, C.c_int32) for k in ("input_kind", "n_freq_origin", "n_freq_dir", "n_hidden",
                                         "width", "skip_layer", "n_out", "weight_dtype")]


class OrcHashLayout(C.Structure):
    _fields_ = [("n_levels", C.c_int32), ("n_features", C.c_int32), ("log2_table", C.c_int32),
                ("base_res", C.c_int32), ("growth", C.c_double), ("box_min", C.c_float * 3),
                ("box_max", C.c_float * 3), ("n_freq_dir", C.c_int32), ("n_hidden", C.c_int32),
                ("width", C.c_int32), ("n_out", C.c_int32), ("table_dtype", C.c_int32),
                ("mlp_dtype", C.c_int32)]


class OrcTrainParams(C.Structure):
    _fields_ = [("lr0", C.c_double), ("lr_final_frac", C.c_double), ("total_steps", C.c_int32),
                ("beta1", C.c_double), ("beta2", C.c_double), ("adam_eps", C.c_double),
                ("dist_clamp", C.c_double), ("ce_weight", C.c_double)]


class OrcCamera(C.Structure):
    _fields_ = [("pos", C.c_double * 3), ("look_at", C.c_double * 3), ("fov_deg", C.c_double)]


class OrcScene(C.Structure):
    _fields_ = [("sphere_c", C.c_double * 3), ("sphere_r", C.c_double),
                ("box_min", C.c_double * 3), ("box_max", C.c_double * 3)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.orc_softplus.restype = C.c_double
        _lib.orc_softplus.argtypes = [C.c_double]
        _lib.orc_sigmoid.restype = C.c_double
        _lib.orc_sigmoid.argtypes = [C.c_double]
        _lib.orc_round_bf16.restype = C.c_double
        _lib.orc_round_bf16.argtypes = [C.c_double]
        _lib.orc_mix64.restype = C.c_uint64
        _lib.orc_mix64.argtypes = [C.c_uint64]
        _lib.orc_u64_at.restype = C.c_uint64
        _lib.orc_u64_at.argtypes = [C.c_uint64] * 3
        _lib.orc_uniform01.restype = C.c_double
        _lib.orc_uniform01.argtypes = [C.c_uint64] * 3
        _lib.orc_hash_table_entries.restype = C.c_int64
        _lib.orc_hash_mlp_params.restype = C.c_int64
        _lib.orc_hash_index.restype = C.c_int64
        _lib.orc_gen_shadow_from_hits.restype = C.c_int64
        _lib.orc_hit_normals.restype = C.c_int64
        _lib.orc_hash_loss_grads.restype = C.c_double
        _lib.orc_lr_at.restype = C.c_double
        _lib.orc_solid_scene_raycast.restype = C.c_double
        _lib.orc_ray_sphere.restype = C.c_double
        _lib.orc_ray_box_exit.restype = C.c_double
    return _lib


def _layout(lay):
    return OrcLayout(lay.input_kind, lay.n_freq_origin, lay.n_freq_dir, lay.n_hidden, lay.width,
                     lay.skip_layer, lay.n_out, lay.weight_dtype)


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def _blob(lay, blob):
    want = np.uint16 if lay.weight_dtype == 1 else np.float32
    b = np.ascontiguousarray(blob)
    assert b.dtype == want, (b.dtype, want)
    return b


def default_threads():
    return len(os.sched_getaffinity(0))


def softplus(z):
    return lib().orc_softplus(float(z))


def sigmoid(z):
    return lib().orc_sigmoid(float(z))


def round_bf16(x):
    return lib().orc_round_bf16(float(x))


def mix64(z):
    return lib().orc_mix64(C.c_uint64(int(z)))


def uniform01(seed, stream, idx):
    return lib().orc_uniform01(C.c_uint64(int(seed)), C.c_uint64(int(stream)), C.c_uint64(int(idx)))


def enc_dim(lay):
    L = _layout(lay)
    return lib().orc_enc_dim(C.byref(L))


def encode(lay, o, d=None):
    o = _f32(o)
    n = o.shape[0]
    L = _layout(lay)
    g = np.empty((n, enc_dim(lay)), dtype=np.float64)
    dd = _f32(d) if d is not None else None
    lib().orc_encode(C.byref(L), _p(o), _p(dd) if dd is not None else None, C.c_int64(n), _p(g))
    return g


def forward(lay, blob, o, d=None, mode=0, nthreads=0):
    """Returns (z[n][n_out], dist[n], vis[n]) in float64; vis is None for n_out == 1."""
    o = _f32(o)
    n = o.shape[0]
    dd = _f32(d) if d is not None else None
    L = _layout(lay)
    b = _blob(lay, blob)
    z = np.zeros((n, lay.n_out), dtype=np.float64)
    dist = np.zeros(n, dtype=np.float64)
    vis = np.zeros(n, dtype=np.float64) if lay.n_out == 2 else None
    rc = lib().orc_forward(C.byref(L), _p(b), _p(o), _p(dd) if dd is not None else None, C.c_int64(n),
                           C.c_int(mode), _p(z), _p(dist), _p(vis) if vis is not None else None,
                           C.c_int(nthreads))
    if rc != 0:
        raise ValueError("oracle: bad layout")
    return z, dist, vis


def _v3(v):
    return (C.c_double * 3)(*[float(x) for x in v])


def ray_sphere(o, d, c, r):
    return lib().orc_ray_sphere(_v3(o), _v3(d), _v3(c), C.c_double(r))


def ray_box_exit(o, d, bmin, bmax):
    face = C.c_int(-1)
    t = lib().orc_ray_box_exit(_v3(o), _v3(d), _v3(bmin), _v3(bmax), C.byref(face))
    return t, face.value


def dir_from_u(u1, u2):
    out = (C.c_double * 3)()
    lib().orc_dir_from_u(C.c_double(u1), C.c_double(u2), out)
    return np.array(list(out))


def camera_from_seed(seed, stream, radius=2.5):
    cam = OrcCamera()
    lib().orc_camera_from_seed(C.c_uint64(int(seed)), C.c_uint64(int(stream)), C.c_double(radius), C.byref(cam))
    return cam


def make_camera(pos, look_at=(0.0, 0.0, 0.0), fov_deg=50.0):
    return OrcCamera(_v3(pos), _v3(look_at), float(fov_deg))


def make_scene(sphere_c=(0.0, 0.0, 0.0), sphere_r=0.6, box_min=(-3.0, -3.0, -3.0), box_max=(3.0, 3.0, 3.0)):
    return OrcScene(_v3(sphere_c), float(sphere_r), _v3(box_min), _v3(box_max))


def gen_camera(cam, width, height):
    n = width * height
    o = np.empty((n, 3), np.float32)
    d = np.empty((n, 3), np.float32)
    lib().orc_gen_camera(C.byref(cam), C.c_int(width), C.c_int(height), _p(o), _p(d))
    return o, d


def gen_sphere_points(seed, stream, n, radius=1.0):
    p = np.empty((n, 3), np.float32)
    nrm = np.empty((n, 3), np.float32)
    lib().orc_gen_sphere_points(C.c_uint64(int(seed)), C.c_uint64(int(stream)), C.c_int64(n),
                                C.c_double(radius), _p(p), _p(nrm))
    return p, nrm


def gen_shadow(p, nrm, light=(3.0, 3.0, 3.0), eps=1e-3):
    p, nrm = _f32(p), _f32(nrm)
    n = p.shape[0]
    o = np.empty((n, 3), np.float32)
    d = np.empty((n, 3), np.float32)
    tmax = np.empty(n, np.float32)
    lib().orc_gen_shadow(_p(p), _p(nrm), C.c_int64(n), _v3(light), C.c_double(eps), _p(o), _p(d), _p(tmax))
    return o, d, tmax


def gen_gbuffer(cam, scene, width, height):
    n = width * height
    p = np.empty((n, 3), np.float32)
    nrm = np.empty((n, 3), np.float32)
    t = np.empty(n, np.float32)
    lib().orc_gen_gbuffer(C.byref(cam), C.byref(scene), C.c_int(width), C.c_int(height), _p(p), _p(nrm), _p(t))
    return p, nrm, t


def gen_ao(p, nrm, spp, seed, stream, eps=1e-3):
    p, nrm = _f32(p), _f32(nrm)
    n = p.shape[0]
    o = np.empty((n * spp, 3), np.float32)
    d = np.empty((n * spp, 3), np.float32)
    lib().orc_gen_ao(_p(p), _p(nrm), C.c_int64(n), C.c_int(spp), C.c_uint64(int(seed)),
                     C.c_uint64(int(stream)), C.c_double(eps), _p(o), _p(d))
    return o, d


def ao_reduce(vis, dist, spp, ao_radius=float("inf")):
    vis, dist = _f32(vis), _f32(dist)
    n = vis.shape[0] // spp
    ao = np.empty(n, np.float32)
    lib().orc_ao_reduce(_p(vis), _p(dist), C.c_int64(n), C.c_int(spp), C.c_double(ao_radius), _p(ao))
    return ao


def sdf_eval(lay, blob, p, base_radius=1.0, alpha=0.05, mode=0, nthreads=0):
    p = _f32(p)
    n = p.shape[0]
    L = _layout(lay)
    b = _blob(lay, blob)
    s = np.empty(n, np.float64)
    rc = lib().orc_sdf_eval(C.byref(L), _p(b), _p(p), C.c_int64(n), C.c_float(base_radius),
                            C.c_float(alpha), C.c_int(mode), _p(s), C.c_int(nthreads))
    if rc != 0:
        raise ValueError("oracle: bad SDF layout")
    return s


def sphere_trace(lay, blob, o, d, max_steps=64, eps=1e-3, t_max=6.0, base_radius=1.0, alpha=0.05,
                 mode=0, want_trace=False, nthreads=0, omega=1.0):
    o, d = _f32(o), _f32(d)
    n = o.shape[0]
    L = _layout(lay)
    b = _blob(lay, blob)
    t = np.empty(n, np.float32)
    hit = np.empty(n, np.uint8)
    steps = np.empty(n, np.int32)
    tp = np.empty((n, max_steps, 3), np.float32) if want_trace else None
    ts = np.empty((n, max_steps), np.float32) if want_trace else None
    rc = lib().orc_sphere_trace_relaxed(C.byref(L), _p(b), _p(o), _p(d), C.c_int64(n), C.c_int(max_steps),
                                C.c_float(eps), C.c_float(t_max), C.c_float(base_radius),
                                C.c_float(alpha), C.c_float(omega), C.c_int(mode), _p(t), _p(hit), _p(steps),
                                _p(tp) if want_trace else None, _p(ts) if want_trace else None,
                                C.c_int(nthreads))
    if rc != 0:
        raise ValueError("oracle: bad SDF layout")
    return (t, hit, steps, tp, ts) if want_trace else (t, hit, steps)


# ------------------------------------------------------------------ hash-grid DDF (ddf_hash_oracle.h)

def _hlayout(lay):
    return OrcHashLayout(lay.n_levels, lay.n_features, lay.log2_table, lay.base_res, float(lay.growth),
                         (C.c_float * 3)(*lay.box_min), (C.c_float * 3)(*lay.box_max), lay.n_freq_dir,
                         lay.n_hidden, lay.width, lay.n_out, lay.table_dtype, lay.mlp_dtype)


def hash_level(lay, level):
    """(resolution N_l, stored entries, entry offset, hashed?) of one level."""
    L = _hlayout(lay)
    res, ent, off, hs = C.c_int64(), C.c_int64(), C.c_int64(), C.c_int()
    rc = lib().orc_hash_level(C.byref(L), C.c_int(level), C.byref(res), C.byref(ent), C.byref(off), C.byref(hs))
    if rc != 0:
        raise ValueError("oracle: bad hash layout / level")
    return res.value, ent.value, off.value, bool(hs.value)


def hash_table_entries(lay):
    L = _hlayout(lay)
    return lib().orc_hash_table_entries(C.byref(L))


def hash_mlp_in(lay):
    L = _hlayout(lay)
    return lib().orc_hash_mlp_in(C.byref(L))


def hash_mlp_params(lay):
    L = _hlayout(lay)
    return lib().orc_hash_mlp_params(C.byref(L))


def hash_index(lay, level, ix, iy, iz):
    L = _hlayout(lay)
    return lib().orc_hash_index(C.byref(L), C.c_int(level), C.c_uint32(ix), C.c_uint32(iy), C.c_uint32(iz))


def _table(lay, table):
    t = np.ascontiguousarray(table)
    assert t.dtype == (np.uint16 if lay.table_dtype == 2 else np.float32), t.dtype
    return t


def hash_encode(lay, table, x):
    x = _f32(x)
    n = x.shape[0]
    L = _hlayout(lay)
    t = _table(lay, table)
    feat = np.zeros((n, lay.n_levels * lay.n_features), dtype=np.float64)
    rc = lib().orc_hash_encode(C.byref(L), _p(t), _p(x), C.c_int64(n), _p(feat))
    if rc != 0:
        raise ValueError("oracle: bad hash layout")
    return feat


def hash_forward(lay, table, mlp, o, d, mode=0, nthreads=0):
    """Returns (z[n][n_out], dist[n], vis[n]) in float64."""
    o, d = _f32(o), _f32(d)
    n = o.shape[0]
    L = _hlayout(lay)
    t = _table(lay, table)
    m = np.ascontiguousarray(mlp)
    assert m.dtype == (np.uint16 if lay.mlp_dtype == 1 else np.float32), m.dtype
    z = np.zeros((n, lay.n_out), dtype=np.float64)
    dist = np.zeros(n, dtype=np.float64)
    vis = np.zeros(n, dtype=np.float64) if lay.n_out == 2 else None
    rc = lib().orc_hash_forward(C.byref(L), _p(t), _p(m), _p(o), _p(d), C.c_int64(n), C.c_int(mode),
                                _p(z), _p(dist), _p(vis) if vis is not None else None, C.c_int(nthreads))
    if rc != 0:
        raise ValueError("oracle: bad hash layout")
    return z, dist, vis


# ------------------------------------------------------------------ wavefront secondary rays

def gen_shadow_from_hits(o, d, dist, vis, light=(3.0, 3.0, 3.0), eps=1e-3):
    """Returns (o2, d2, tmax, index) of the compacted shadow-ray batch."""
    o, d, dist, vis = _f32(o), _f32(d), _f32(dist), _f32(vis)
    n = o.shape[0]
    o2 = np.empty((n, 3), np.float32); d2 = np.empty((n, 3), np.float32)
    tmax = np.empty(n, np.float32); index = np.empty(n, np.int32)
    k = lib().orc_gen_shadow_from_hits(_p(o), _p(d), _p(dist), _p(vis), C.c_int64(n), _v3(light), C.c_float(eps),
                                       _p(o2), _p(d2), _p(tmax), _p(index))
    return o2[:k].copy(), d2[:k].copy(), tmax[:k].copy(), index[:k].copy()


def shadow_lit(vis2, dist2, tmax, index, n):
    vis2, dist2, tmax = _f32(vis2), _f32(dist2), _f32(tmax)
    index = np.ascontiguousarray(index, dtype=np.int32)
    lit = np.empty(n, np.uint8)
    lib().orc_shadow_lit(_p(vis2), _p(dist2), _p(tmax), _p(index), C.c_int64(len(index)), C.c_int64(n), _p(lit))
    return lit


def hit_normals(o, d, dist, vis, width, height):
    """Returns (p, nrm, index) of the hits of a width x height primary batch (reading W5)."""
    o, d, dist, vis = _f32(o), _f32(d), _f32(dist), _f32(vis)
    n = width * height
    assert o.shape[0] == n
    p = np.empty((n, 3), np.float32); nrm = np.empty((n, 3), np.float32); index = np.empty(n, np.int32)
    k = lib().orc_hit_normals(_p(o), _p(d), _p(dist), _p(vis), C.c_int(width), C.c_int(height), _p(p), _p(nrm), _p(index))
    return p[:k].copy(), nrm[:k].copy(), index[:k].copy()


# ------------------------------------------------------------------ training (ddf_hash_oracle.h, T1-T5)

def train_params(lr0=3e-3, lr_final_frac=0.05, total_steps=30000, beta1=0.9, beta2=0.999, adam_eps=1e-8,
                 dist_clamp=6.0, ce_weight=0.3):
    return OrcTrainParams(lr0, lr_final_frac, total_steps, beta1, beta2, adam_eps, dist_clamp, ce_weight)


def hash_loss_grads(lay, table, mlp, o, d, t, hit, P, want_grads=True):
    """(loss, grad_table[entries*F], grad_mlp) in float64; table and mlp are float32 master copies."""
    o, d, t = _f32(o), _f32(d), _f32(t)
    hit = np.ascontiguousarray(hit, dtype=np.uint8)
    table, mlp = _f32(table), _f32(mlp)
    n = o.shape[0]
    L = _hlayout(lay)
    gt = np.zeros(table.shape[0], np.float64) if want_grads else None
    gm = np.zeros(mlp.shape[0], np.float64) if want_grads else None
    loss = lib().orc_hash_loss_grads(C.byref(L), _p(table), _p(mlp), _p(o), _p(d), _p(t), _p(hit), C.c_int64(n),
                                     C.byref(P), _p(gt) if want_grads else None, _p(gm) if want_grads else None)
    return loss, gt, gm


def hash_relu_margin(lay, table, mlp, o, d):
    """min |pre-activation| over the hidden units, per ray (float64): the distance from a ReLU kink."""
    o, d = _f32(o), _f32(d)
    table, mlp = _f32(table), _f32(mlp)
    L = _hlayout(lay)
    out = np.empty(o.shape[0], np.float64)
    rc = lib().orc_hash_relu_margin(C.byref(L), _p(table), _p(mlp), _p(o), _p(d), C.c_int64(o.shape[0]), _p(out))
    assert rc == 0
    return out


def lr_at(P, step):
    return lib().orc_lr_at(C.byref(P), C.c_int64(step))


def adam_step(p, g, m, v, step, lr, P):
    """in place on p (float32), m, v (float64)"""
    assert p.dtype == np.float32 and m.dtype == np.float64 and v.dtype == np.float64
    g = np.ascontiguousarray(g, dtype=np.float64)
    lib().orc_adam_step(_p(p), _p(g), _p(m), _p(v), C.c_int64(p.shape[0]), C.c_int64(step), C.c_double(lr), C.byref(P))


def solid_scene_raycast(o, d, sphere_c=(0.0, 0.0, 0.0), sphere_r=0.5, bmin=(-0.9, -0.9, -0.9), bmax=(0.9, 0.9, -0.6)):
    return lib().orc_solid_scene_raycast(_v3(o), _v3(d), _v3(sphere_c), C.c_double(sphere_r), _v3(bmin), _v3(bmax))


TRAIN_SCENE = dict(sphere_c=(0.0, 0.0, 0.0), sphere_r=0.5, bmin=(-0.9, -0.9, -0.9), bmax=(0.9, 0.9, -0.6))


def gen_train_batch(seed, stream, step, n, sample_half=2.0, scene=None):
    sc = scene or TRAIN_SCENE
    o = np.empty((n, 3), np.float32); d = np.empty((n, 3), np.float32)
    t = np.empty(n, np.float32); hit = np.empty(n, np.uint8)
    lib().orc_gen_train_batch(_v3(sc["sphere_c"]), C.c_double(sc["sphere_r"]), _v3(sc["bmin"]), _v3(sc["bmax"]),
                              C.c_uint64(int(seed)), C.c_uint64(int(stream)), C.c_int64(step), C.c_int64(n),
                              C.c_double(sample_half), _p(o), _p(d), _p(t), _p(hit))
    return o, d, t, hit
