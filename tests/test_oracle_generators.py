"""Pins for the oracle's generators, AO reducer and sphere tracer.

Closed forms and invariants only: pinhole geometry, textbook ray-sphere / ray-slab results on
hand-placed rays, the analytic occluded fraction of the shadow batch, cosine-weighted moments.
"""
import math

import numpy as np
import pytest

from ddf_inputs import MASTER_SEED, STREAMS, Layout, layout_sdf, make_weights, mix64, uniform01

TAN25 = 0.4663076581549986


def test_rng_matches_shared_spec(orc):
    """A8: the oracle's C mixer and the numpy one in ddf_inputs are the same function."""
    assert orc.mix64(0) == 0xE220A8397B1DCDAF          # SplitMix64's first output for seed 0
    for z in (1, 12345, 2 ** 63 + 17):
        assert orc.mix64(z) == int(mix64(np.uint64(z)))
    for idx in (0, 1, 999, 2 ** 40 + 3):
        assert orc.uniform01(MASTER_SEED, 5, idx) == float(uniform01(MASTER_SEED, 5, [idx])[0])
    u = uniform01(MASTER_SEED, 6, np.arange(200000))
    assert abs(u.mean() - 0.5) < 3e-3 and abs(u.var() - 1 / 12) < 2e-3 and u.min() >= 0 and u.max() < 1


# ------------------------------------------------------------------ P9: camera, intersections

def test_ray_sphere_and_box_textbook(orc):
    assert orc.ray_sphere([0, 0, -3], [0, 0, 1], [0, 0, 0], 1.0) == pytest.approx(2.0, abs=1e-15)
    assert orc.ray_sphere([0, 0, 0], [0, 0, 1], [0, 0, 0], 1.0) == pytest.approx(1.0)    # from inside
    assert orc.ray_sphere([0, 2, -3], [0, 0, 1], [0, 0, 0], 1.0) == -1.0                 # miss
    assert orc.ray_sphere([0, 0, 3], [0, 0, 1], [0, 0, 0], 1.0) == -1.0                  # behind
    # grazing offset b: t = sqrt(9 - b^2) - sqrt(1 - b^2) measured from z=-3... use pythagoras
    b = 0.6
    assert orc.ray_sphere([b, 0, -3], [0, 0, 1], [0, 0, 0], 1.0) == pytest.approx(3.0 - math.sqrt(1 - b * b))
    t, face = orc.ray_box_exit([0, 0, 0], [1, 0, 0], [-3, -3, -3], [3, 3, 3])
    assert (t, face) == (3.0, 1)
    t, face = orc.ray_box_exit([1, 1, 1], [0, -1, 0], [-3, -3, -3], [3, 3, 3])
    assert (t, face) == (4.0, 2)
    d = np.array([1.0, 2.0, -2.0]) / 3.0
    t, face = orc.ray_box_exit([0, 0, 0], d, [-3, -3, -3], [3, 3, 3])
    assert t == pytest.approx(4.5) and face in (3, 4)        # y and z faces tie at t = 4.5


def test_camera_pinhole_geometry(orc):
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    c = np.array(list(cam.pos))
    assert np.linalg.norm(c) == pytest.approx(2.5, rel=1e-12)
    W = H = 64
    o, d = orc.gen_camera(cam, W, H)
    assert o.shape == (W * H, 3) and np.all(o == c.astype(np.float32))
    assert np.allclose(np.linalg.norm(d.astype(np.float64), axis=1), 1.0, atol=2e-7)
    d = d.reshape(H, W, 3).astype(np.float64)
    f = -c / np.linalg.norm(c)
    centre = d[H // 2 - 1:H // 2 + 1, W // 2 - 1:W // 2 + 1].reshape(-1, 3).mean(0)
    assert np.allclose(centre / np.linalg.norm(centre), f, atol=1e-6)
    # a pixel centre at normalised offset (u, v) makes tan(angle to axis) = sqrt(u^2+v^2) * tan 25
    for (row, col) in [(0, 0), (10, 50), (63, 31)]:
        u = (2 * (col + 0.5) / W - 1); v = (1 - 2 * (row + 0.5) / H)
        cosang = d[row, col] @ f
        assert math.tan(math.acos(cosang)) == pytest.approx(math.hypot(u, v) * TAN25, rel=1e-5)
    # image orientation: rows go down (v decreases), columns go right; world up is +z
    right = np.cross(f, [0, 0, 1.0]); right /= np.linalg.norm(right)
    up2 = np.cross(right, f)
    assert (d[0, W // 2] - d[H - 1, W // 2]) @ up2 > 0
    assert (d[H // 2, W - 1] - d[H // 2, 0]) @ right > 0
    # full 50 degree field of view between the image borders (extrapolate half a pixel)
    cam2 = orc.make_camera([0, -2.5, 0], fov_deg=50.0)
    o2, d2 = orc.gen_camera(cam2, 2, 2)
    # 2x2 image: pixel centres sit at +-0.5 of the half-extent
    assert abs(d2[0, 0] / d2[0, 1]) == pytest.approx(0.5 * TAN25, rel=1e-6)
    assert abs(d2[0, 2] / d2[0, 1]) == pytest.approx(0.5 * TAN25, rel=1e-6)


def test_camera_up_fallback(orc):
    cam = orc.make_camera([0, 0, 2.5])
    o, d = orc.gen_camera(cam, 4, 4)
    assert np.all(np.isfinite(d)) and np.allclose(np.linalg.norm(d, axis=1), 1.0, atol=1e-6)


def test_gbuffer_points_lie_on_scene(orc):
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    sc = orc.make_scene()
    W = H = 96
    p, nrm, t = orc.gen_gbuffer(cam, sc, W, H)
    o, d = orc.gen_camera(cam, W, H)
    assert np.allclose(p, o + t[:, None] * d, atol=1e-5)
    r = np.linalg.norm(p.astype(np.float64), axis=1)
    on_sphere = np.abs(r - 0.6) < 1e-5
    on_wall = np.isclose(np.abs(p).max(axis=1), 3.0, atol=1e-5)
    assert np.all(on_sphere | on_wall) and on_sphere.sum() > 100 and on_wall.sum() > 100
    assert np.allclose(np.linalg.norm(nrm, axis=1), 1.0, atol=1e-6)
    assert np.allclose(nrm[on_sphere], p[on_sphere] / 0.6, atol=1e-5)
    # wall normals point inward: n . p = -3
    assert np.allclose((nrm[on_wall] * p[on_wall]).sum(1), -3.0, atol=1e-5)
    # analytic sphere silhouette: a ray hits iff its angle to the axis is below asin(0.6/2.5)
    c = np.array(list(cam.pos)); f = -c / 2.5
    ang = np.arccos(np.clip(d.astype(np.float64) @ f, -1, 1))
    lim = math.asin(0.6 / 2.5)
    clear = np.abs(ang - lim) > 1e-4
    assert np.array_equal(on_sphere[clear], (ang < lim)[clear])
    # independent distances: sphere hits obey the closed form along the axis ray
    i = np.argmin(ang)
    assert t[i] == pytest.approx(2.5 * math.cos(ang[i]) - math.sqrt(0.36 - (2.5 * math.sin(ang[i])) ** 2), rel=1e-5)


# ------------------------------------------------------------------ P10: shadow batch

def test_shadow_batch_closed_form_fraction(orc):
    n = 1 << 18
    p, nrm = orc.gen_sphere_points(MASTER_SEED, STREAMS["shadow_points"], n, 1.0)
    assert np.array_equal(p, nrm)
    assert np.allclose(np.linalg.norm(p.astype(np.float64), axis=1), 1.0, atol=2e-7)
    assert np.allclose(p.mean(0), 0.0, atol=5e-3) and np.allclose((p.astype(np.float64) ** 2).mean(0), 1 / 3, atol=3e-3)
    L = np.array([3.0, 3.0, 3.0])
    o, d, tmax = orc.gen_shadow(p, nrm, L, 1e-3)
    o64, d64 = o.astype(np.float64), d.astype(np.float64)
    assert np.allclose(np.linalg.norm(o64, axis=1), 1.001, atol=3e-7)
    assert np.allclose(np.linalg.norm(d64, axis=1), 1.0, atol=2e-7)
    assert np.allclose(tmax, np.linalg.norm(L - o64, axis=1), rtol=1e-6)
    assert np.allclose(np.cross(d64, L - o64), 0.0, atol=1e-6)
    # occluded by the unit sphere (textbook discriminant, written here independently)
    b = (o64 * d64).sum(1)
    occl = (b < 0) & (b * b - ((o64 * o64).sum(1) - 1.0) >= 0)
    D = math.sqrt(27.0)
    theta_t = math.acos(1 / D) + math.acos(1 / 1.001)
    want = (1 + math.cos(theta_t)) / 2
    assert want == pytest.approx(0.574203, abs=1e-6)
    assert occl.mean() == pytest.approx(want, abs=4 * math.sqrt(0.25 / n))
    assert abs(occl.mean() - 0.596225) > 0.015          # the value a missing offset would give


# ------------------------------------------------------------------ P11: AO

def test_ao_samples_are_cosine_weighted(orc):
    rng = np.random.default_rng(1)
    nrm = rng.standard_normal((2000, 3)); nrm /= np.linalg.norm(nrm, axis=1, keepdims=True)
    nrm[:6] = [[1, 0, 0], [-1, 0, 0], [0, 1, 0], [0, -1, 0], [0, 0, 1], [0, 0, -1]]
    p = rng.standard_normal((2000, 3)).astype(np.float32)
    spp = 16
    o, d = orc.gen_ao(p, nrm, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3)
    assert o.shape == (2000 * spp, 3)
    nn = np.repeat(nrm.astype(np.float32).astype(np.float64), spp, axis=0)
    assert np.allclose(o, np.repeat(p, spp, axis=0) + 1e-3 * nn, atol=1e-6)
    assert np.allclose(np.linalg.norm(d.astype(np.float64), axis=1), 1.0, atol=2e-7)
    c = (d.astype(np.float64) * nn).sum(1)
    assert c.min() >= -1e-7
    m = len(c)
    assert c.mean() == pytest.approx(2 / 3, abs=4 * math.sqrt(1 / 18 / m))        # var = 1/2 - 4/9
    assert (c * c).mean() == pytest.approx(0.5, abs=4 * math.sqrt(1 / 12 / m))
    # azimuth is uniform: the tangential part has zero mean
    tang = d.astype(np.float64) - c[:, None] * nn
    assert np.allclose(tang[:spp * 6].reshape(6, spp, 3).mean(1), 0, atol=0.5)
    assert np.allclose(tang.mean(0), 0, atol=0.02)


def test_ao_reduce_rules_and_sphere_over_floor(orc):
    spp = 16
    vis = np.array([0.9] * 16 + [0.1] * 16 + [0.9] * 4 + [0.5] * 12, np.float32)     # 0.5 is a miss (A10)
    dist = np.ones(48, np.float32)
    assert orc.ao_reduce(vis, dist, spp).tolist() == [0.0, 1.0, 0.75]
    assert orc.ao_reduce(vis, dist, spp, ao_radius=0.5).tolist() == [1.0, 1.0, 1.0]
    # cosine-weighted occlusion of a sphere (radius r, centre at height h) seen from the floor
    # point below it is (r/h)^2: substitute the analytic hit test for the MLP
    npts, r, h = 4096, 0.6, 1.5
    p = np.zeros((npts, 3), np.float32); nrm = np.tile(np.array([0, 0, 1], np.float32), (npts, 1))
    o, d = orc.gen_ao(p, nrm, spp, 77, STREAMS["ao_samples"], 0.0)
    hit = np.array([orc.ray_sphere(o[i], d[i], [0, 0, h], r) > 0 for i in range(0, npts * spp, 1)])
    ao = orc.ao_reduce(hit.astype(np.float32), np.ones(npts * spp, np.float32), spp)
    assert set(np.unique(ao * 16).tolist()) <= set(range(17))
    pocc = (r / h) ** 2
    assert 1 - ao.mean() == pytest.approx(pocc, abs=4 * math.sqrt(pocc * (1 - pocc) / (npts * spp)))


# ------------------------------------------------------------------ P12: sphere tracer

def test_sphere_trace_alpha0_reaches_analytic_distance(orc):
    lay = Layout(1, 2, 0, 1, 4, -1, 1, 1)
    blob = make_weights(lay)
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 48, 48)
    # widen the fan so that some rays miss the unit sphere
    t, hit, steps, tp, ts = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0, want_trace=True)
    want = np.array([orc.ray_sphere(o[i], d[i], [0, 0, 0], 1.0) for i in range(len(o))])
    ang = np.arccos(np.clip(d.astype(np.float64) @ (-np.array(list(cam.pos)) / 2.5), -1, 1))
    lim = math.asin(1 / 2.5)
    # grazing rays converge slowly and may stop within eps *outside* the sphere: exclude a band
    sure_hit, sure_miss = ang < lim - 0.02, ang > lim + 0.02
    assert sure_hit.sum() > 500 and sure_miss.sum() > 100
    assert np.all(hit[sure_hit] == 1) and np.all(hit[sure_miss] == 0)
    # at a hit the remaining gap along the ray is bounded by eps / cos(incidence); cos >= 0.19 here
    gap = want[sure_hit] - t[sure_hit]
    assert np.all(gap > -1e-5) and np.all(gap < 1e-3 / 0.19)
    assert np.all(t[sure_miss] > 6.0) and np.all(steps[sure_miss] < 64)
    # first step: s_0 = |o| - 1 = 1.5 for every ray; the trace visits p_k = o + t_k d
    assert np.allclose(ts[:, 0], 1.5, atol=1e-6)
    assert np.allclose(tp[:, 1], o + 1.5 * d, atol=1e-6)
    assert np.all(steps >= 2) and np.all(np.isnan(ts[np.arange(len(o)), np.minimum(steps, 63)]) | (steps == 64))


def test_over_relaxed_sphere_trace_is_safe_and_shorter(orc):
    """reading A19': with the exact SDF of the unit sphere, steps of omega * s reach
    the same hits at the analytic distance and fall back when a relaxed step jumps the surface (the
    spheres at t_prev and t no longer touch); omega = 1 is the plain tracer bit for bit.  On this
    scene relaxation only pays for omega = 1.1: from the camera the first step is 1.5 and almost
    normal to the surface, so omega >= 1.2 overshoots, falls back and costs one evaluation more per
    ray - which is why the CUDA tracer does not implement it."""
    lay = Layout(1, 2, 0, 1, 4, -1, 1, 1)
    blob = make_weights(lay)
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 48, 48)
    t1, h1, s1 = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0)
    ta, ha, sa = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0, omega=1.0)
    assert np.array_equal(t1, ta) and np.array_equal(h1, ha) and np.array_equal(s1, sa)
    want = np.array([orc.ray_sphere(o[i], d[i], [0, 0, 0], 1.0) for i in range(len(o))])
    ang = np.arccos(np.clip(d.astype(np.float64) @ (-np.array(list(cam.pos)) / 2.5), -1, 1))
    lim = math.asin(1 / 2.5)
    sure_hit, sure_miss = ang < lim - 0.02, ang > lim + 0.02
    for om in (1.1, 1.2, 1.6, 1.9):
        t, hit, steps, tp, ts = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0, want_trace=True, omega=om)
        assert np.all(hit[sure_hit] == 1) and np.all(hit[sure_miss] == 0)
        gap = want[sure_hit] - t[sure_hit]
        assert np.all(np.abs(gap) < 1e-3 / 0.19 + 1e-5)               # stops within eps of the surface, on either side
        assert (steps.sum() < s1.sum()) == (om < 1.15), (om, steps.sum(), s1.sum())
        # a ray through the centre: s_0 = 1.5, the relaxed step lands at t = 1.5 om; for om = 1.9 that is past the
        # far side reach: |s_1| + |s_0| < 1.5 om  =>  fall back to t = 1.5 (the plain position)
        c = int(np.argmin(ang))
        if om == 1.9:
            assert abs(ts[c, 0] - 1.5) < 1e-3 and abs(np.linalg.norm(tp[c, 2] - (o[c] + 1.5 * d[c]))) < 2e-3
        assert np.all(t[sure_miss] > 6.0)


def test_sphere_trace_mlp_term_is_orc_forward(orc):
    """s(p) = (|p| - R) + alpha * MLP(p): the MLP part is exactly the (pinned) forward pass."""
    lay = Layout(1, 3, 0, 2, 8, 1, 1, 1)
    blob = make_weights(lay, seed=4, bias_scale=0.2)
    p = np.random.default_rng(3).uniform(-1.5, 1.5, (40, 3)).astype(np.float32)
    z, _, _ = orc.forward(lay, blob, p, None)
    s = orc.sdf_eval(lay, blob, p, 1.0, 0.05)
    want = (np.linalg.norm(p.astype(np.float64), axis=1) - 1.0) + 0.05 * z[:, 0]
    assert np.allclose(s, want, atol=5e-7)                  # fp32 state arithmetic
    t, hit, steps, tp, ts = orc.sphere_trace(lay, blob, p * 0 + [0, 0, -2.5], np.tile([0, 0, 1.0], (40, 1)),
                                             8, 1e-3, 6.0, 1.0, 0.05, want_trace=True)
    s0 = orc.sdf_eval(lay, blob, tp[:, 0], 1.0, 0.05)
    assert np.allclose(ts[:, 0], s0, atol=1e-7)
