"""Pins of the training oracle (oracle/ddf_hash_oracle.c, readings T1-T5): CPU only.
Gradients are pinned by central finite differences of the oracle's own LOSS (a different code path:
forward only), Adam and the schedule by their published closed forms, the supervision by textbook
ray-sphere / ray-box values."""
import math

import numpy as np

from ddf_inputs import HashLayout, make_hash_table, make_hash_mlp, random_rays


def _small():
    return HashLayout(n_levels=3, n_features=2, log2_table=9, base_res=3, growth=2.0,
                      box_min=(-1.0, -1.0, -1.0), box_max=(1.0, 1.0, 1.0), n_freq_dir=2, n_hidden=2, width=8)


def _batch(orc, lay, n=40):
    o, d = random_rays(n)
    rng = np.random.default_rng(3)
    t = rng.uniform(0.2, 3.0, n).astype(np.float32)
    hit = (rng.uniform(size=n) < 0.6).astype(np.uint8)
    table = make_hash_table(lay, orc.hash_table_entries(lay), scale=0.5)
    mlp = make_hash_mlp(lay, bias_scale=0.3)
    return o, d, t, hit, table, mlp


def test_gradients_match_finite_differences(orc):
    lay = _small()
    o, d, t, hit, table, mlp = _batch(orc, lay)
    P = orc.train_params(dist_clamp=2.0)                  # some rays sit beyond the clamp: zero distance gradient there
    loss, gt, gm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, P)
    assert np.isfinite(loss) and np.abs(gt).max() > 0 and np.abs(gm).max() > 0
    rng = np.random.default_rng(0)
    h = 1e-3                                              # fp32 master copies: the step must survive the cast
    touched = np.nonzero(gt)[0]
    for arr, g, picks in ((table, gt, rng.choice(touched, 25, replace=False)), (mlp, gm, rng.choice(len(mlp), 40, replace=False))):
        for i in picks:
            a = arr.copy(); b = arr.copy()
            a[i] += h; b[i] -= h
            step = float(a[i]) - float(b[i])
            la = orc.hash_loss_grads(lay, a if arr is table else table, a if arr is mlp else mlp, o, d, t, hit, P, want_grads=False)[0]
            lb = orc.hash_loss_grads(lay, b if arr is table else table, b if arr is mlp else mlp, o, d, t, hit, P, want_grads=False)[0]
            fd = (la - lb) / step
            assert abs(fd - g[i]) <= 2e-4 * max(1.0, abs(g[i])) + 2e-5, (i, fd, g[i])
    # entries no ray touches have exactly zero gradient
    assert np.count_nonzero(gt) < len(gt)


def test_relu_margin_is_the_smallest_hidden_pre_activation(orc):
    """orc.hash_relu_margin against numpy matrix products on the (separately pinned) encoder's features, and
    its meaning: a ray with margin m keeps every ReLU on its side under any perturbation of a
    pre-activation below m, so nudging a bias by less than the batch's margin leaves the gradient's
    zero pattern (the ReLU masks) of the first layer's bias untouched."""
    lay = _small()
    o, d, t, hit, table, mlp = _batch(orc, lay, n=200)
    feat = orc.hash_encode(lay, table, o)
    gam = [d.astype(np.float64)]
    for k in range(lay.n_freq_dir):
        gam += [np.sin(np.pi * d.astype(np.float64) * 2.0 ** k), np.cos(np.pi * d.astype(np.float64) * 2.0 ** k)]
    x = np.concatenate([feat] + gam, axis=1)
    E, W = x.shape[1], lay.width
    w = mlp.astype(np.float64)
    W0, b0 = w[:W * E].reshape(W, E), w[W * E:W * E + W]
    o1 = W * E + W
    W1, b1 = w[o1:o1 + W * W].reshape(W, W), w[o1 + W * W:o1 + W * W + W]
    z0 = x @ W0.T + b0
    z1 = np.maximum(z0, 0.0) @ W1.T + b1
    want = np.minimum(np.abs(z0).min(axis=1), np.abs(z1).min(axis=1))
    got = orc.hash_relu_margin(lay, table, mlp, o, d)
    assert np.allclose(got, want, rtol=1e-12, atol=1e-15) and got.min() > 0 and got.max() < 1.0


def test_loss_closed_forms(orc):
    """zero MLP: softplus(b0) = ln 2 + ..., CE = ln 2; clamp; misses carry no distance term (T1, T2)"""
    lay = _small()
    o, d, t, hit, table, mlp = _batch(orc, lay, n=10)
    mlp = np.zeros_like(mlp)
    P = orc.train_params(dist_clamp=0.5, ce_weight=0.3)
    hit[:] = 1; t[:] = math.log(2.0) + 0.25
    loss, _, gm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, P)
    assert abs(loss - (0.25 + 0.3 * math.log(2.0))) < 1e-7          # |ln2 - t| = 0.25 < clamp
    t[:] = 5.0
    loss, _, gm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, P)
    assert abs(loss - (0.5 + 0.3 * math.log(2.0))) < 1e-7           # clamped at 0.5 ...
    assert gm[-2] == 0.0 and abs(gm[-1] - 0.3 * (0.5 - 1.0)) < 1e-12  # ... and flat there; d CE / d z1 = w (xi - hit)
    hit[:] = 0
    loss, _, gm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, P)
    assert abs(loss - 0.3 * math.log(2.0)) < 1e-12 and gm[-2] == 0.0 and abs(gm[-1] - 0.15) < 1e-12


def test_adam_and_schedule_closed_forms(orc):
    P = orc.train_params(lr0=3e-3, lr_final_frac=0.05, total_steps=30000, adam_eps=1e-12)
    assert abs(orc.lr_at(P, 0) - 3e-3) < 1e-15 and abs(orc.lr_at(P, 30000) - 1.5e-4) < 1e-15     # "decayed by cosine to five percent"
    assert abs(orc.lr_at(P, 15000) - 3e-3 * 0.525) < 1e-15 and orc.lr_at(P, 99999) == orc.lr_at(P, 30000)
    g = np.array([0.5, -2.0, 1e-3, -7e-5]); p = np.array([1.0, 1.0, 1.0, 1.0], np.float32)
    m = np.zeros(4); v = np.zeros(4)
    orc.adam_step(p, g, m, v, 1, 0.01, P)
    assert np.allclose(p, 1.0 - 0.01 * np.sign(g), atol=1e-6)        # first step: -lr sign(g)
    for s in range(2, 11):
        orc.adam_step(p, g, m, v, s, 0.01, P)
    assert np.allclose(p, 1.0 - 0.1 * np.sign(g), atol=1e-5)         # constant gradient: every step is -lr sign(g)
    assert np.allclose(m, (1 - 0.9 ** 10) * g) and np.allclose(v, (1 - 0.999 ** 10) * g * g)
    # zero gradient after a history: the moments decay, the parameter keeps moving the same way
    p0 = p.copy(); orc.adam_step(p, np.zeros(4), m, v, 11, 0.01, P)
    assert np.all(np.sign(p - p0) == -np.sign(g))


def test_supervision_raycast_textbook(orc):
    c, r, bmin, bmax = (0.0, 0.0, 0.0), 0.5, (-0.9, -0.9, -0.9), (0.9, 0.9, -0.6)
    rc = lambda o, d: orc.solid_scene_raycast(o, d, c, r, bmin, bmax)
    assert abs(rc((0, 0, 3), (0, 0, -1)) - 2.5) < 1e-12                 # sphere from outside
    assert abs(rc((0, 0, 0), (0, 0, 1)) - 0.5) < 1e-12                  # from inside: where the ray leaves
    assert abs(rc((0.8, 0.8, 3), (0, 0, -1)) - 3.6) < 1e-12             # misses the sphere, lands on the slab's top face
    assert abs(rc((0.8, 0, -0.75), (1, 0, 0)) - 0.1) < 1e-12            # inside the slab: exit face
    assert rc((2, 2, 2), (0, 0, 1)) == -1.0 and rc((0, 2, 0), (1, 0, 0)) == -1.0     # misses
    assert abs(rc((0, 0, -3), (0, 0, 1)) - 2.1) < 1e-12                 # slab bottom before the sphere
    s = 1 / math.sqrt(2)
    assert abs(rc((-2, 0, -2.75), (s, 0, s)) - (1.85 / s)) < 1e-9       # oblique: x is inside the slab from t = 1.1/s, z only from 1.85/s (at x = -0.15)


# ---- orc_gen_train_batch (reading T6; "Rays that start on the surface and point in all directions ... a point
# moved forward by s should report distance t-s", "We replace 30 percent of each batch with the ray-march
# shifted points").  The pin shares nothing with the generator's ray casts: each ray's random draws are recomputed with
# the numpy counter generator (ddf_inputs/rng.py), which says what SHOULD have happened to it (anchored iff u6 >= 0.5 and
# the camera ray hit; shifted iff the emitted ray hits and u9 < 0.3), and the geometry is judged by implicit surface
# functions and brute-force sampling along the ray, never by a ray-surface formula.
def _unsigned_surface_distance(p, sc):
    c = np.array(sc["sphere_c"]); r = sc["sphere_r"]
    ds = np.abs(np.linalg.norm(p - c, axis=1) - r)
    bmin, bmax = np.array(sc["bmin"]), np.array(sc["bmax"])
    q = np.abs(p - 0.5 * (bmin + bmax)) - 0.5 * (bmax - bmin)              # textbook signed distance of a box
    sd = np.linalg.norm(np.maximum(q, 0.0), axis=1) + np.minimum(q.max(axis=1), 0.0)
    return np.minimum(ds, np.abs(sd))


def _depth_inside(p, sc):
    """> 0: how deep p is inside the sphere or the box (0 outside)."""
    c = np.array(sc["sphere_c"]); r = sc["sphere_r"]
    bmin, bmax = np.array(sc["bmin"]), np.array(sc["bmax"])
    q = np.abs(p - 0.5 * (bmin + bmax)) - 0.5 * (bmax - bmin)
    return np.maximum(np.maximum(r - np.linalg.norm(p - c, axis=-1), -q.max(axis=-1)), 0.0)


def test_train_batch_generator_pins(orc):
    from ddf_inputs.rng import MASTER_SEED, STREAMS, uniform01
    sc = orc.TRAIN_SCENE
    n, step, half = 1 << 18, 3, 2.0
    o, d, t, hit = orc.gen_train_batch(MASTER_SEED, STREAMS["train_rays"], step, n, half)
    o64, d64, t64, hit = o.astype(np.float64), d.astype(np.float64), t.astype(np.float64), hit.astype(bool)
    base = (np.uint64(step) * np.uint64(n) + np.arange(n, dtype=np.uint64)) * np.uint64(16)
    u = np.stack([uniform01(MASTER_SEED, STREAMS["train_rays"], base + np.uint64(j)) for j in range(11)], axis=1)
    oo = (2.0 * u[:, 0:3] - 1.0) * half                                    # camera origin, uniform in the sampling cube
    q = (2.0 * u[:, 3:6] - 1.0) - oo                                       # toward a point of the unit cube
    dcam = q / np.linalg.norm(q, axis=1, keepdims=True)
    moved = np.any(o != oo.astype(np.float32), axis=1)
    A = u[:, 6] >= 0.5                                                     # the anchor draw
    ok10 = u[:, 10] > 0                                                    # a zero shift moves nothing (probability 2^-24)

    # every ray: unit direction; a miss has target 0; a hit's target ends ON the surface
    assert np.abs(np.linalg.norm(d64, axis=1) - 1.0).max() < 1e-6
    assert np.all(t[~hit] == 0.0) and np.all(t[hit] > 0.0)
    assert _unsigned_surface_distance(o64[hit] + t64[hit, None] * d64[hit], sc).max() < 2e-5
    assert 0.3 < hit.mean() < 0.95

    # ... and it is the FIRST surface: nothing solid strictly before it, and a miss never runs deep through a solid
    outside = _depth_inside(o64, sc) == 0.0
    f = (np.arange(64) + 0.5) / 64
    sel = np.nonzero(hit & outside)[0][:20000]
    pts = o64[sel, None, :] + (f[None, :, None] * (t64[sel, None, None] - 1e-4)) * d64[sel, None, :]
    assert _depth_inside(pts, sc).max() < 1e-5
    sel = np.nonzero(~hit)[0][:20000]
    s = (np.arange(512) + 0.5) / 512 * 7.5
    pts = o64[sel, None, :] + s[None, :, None] * d64[sel, None, :]
    assert _depth_inside(pts, sc).max() < 0.02

    # camera half (u6 < 0.5): never anchored - the direction is the camera's, and the origin moves iff the ray hits and
    # u9 < 0.3 (the shift fraction, exactly), by s = u10 * (distance before the shift) along the ray: target t - s
    C_ = ~A
    assert np.abs(d64[C_] - dcam[C_]).max() < 1e-6
    assert np.array_equal(moved[C_ & ok10], (hit & (u[:, 9] < 0.3))[C_ & ok10])
    sh = C_ & moved
    s_ = np.linalg.norm(o64[sh] - oo[sh], axis=1)
    assert np.abs(np.cross(o64[sh] - oo[sh], dcam[sh])).max() < 1e-5       # moved along the ray
    assert np.abs(s_ - u[sh, 10] * (s_ + t64[sh])).max() < 5e-6           # s = u10 * t_before, target = t_before - s (fp32 outputs)
    assert abs(moved[C_ & hit].mean() - 0.3) < 4 * math.sqrt(0.21 / (C_ & hit).sum())

    # anchor half (u6 >= 0.5): anchored iff the camera ray hit, with the camera half's hit rate (two samples of one
    # Bernoulli, 4 sigma); an anchored ray starts 1e-3 BEFORE the camera ray's surface point, pointing where the
    # sphere sample of (u7, u8) points (reading A9)
    p_cam = hit[C_].mean()
    anchored = A & moved
    sig = math.sqrt(p_cam * (1 - p_cam) * (1.0 / A.sum() + 1.0 / C_.sum()))
    assert abs(anchored[A].mean() - p_cam) < 4 * sig, (anchored[A].mean(), p_cam, sig)
    assert abs(anchored.mean() - 0.5 * p_cam) < 4 * sig
    z = 2.0 * u[:, 7] - 1.0; phi = 2.0 * np.pi * u[:, 8]; rr = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    dsph = np.stack([rr * np.cos(phi), rr * np.sin(phi), z], axis=1)
    assert np.abs(d64[anchored] - dsph[anchored]).max() < 1e-6
    assert np.all(~moved[A & ~anchored] & ~hit[A & ~anchored])             # camera miss: emitted as it is
    shifted = anchored & hit & (u[:, 9] < 0.3)
    s_ = np.where(shifted, t64 * u[:, 10] / (1.0 - u[:, 10]), 0.0)         # undo the shift: s = u10 * t_before
    o_pre = o64 - s_[:, None] * d64
    assert np.abs(np.cross(o_pre[anchored] - oo[anchored], dcam[anchored])).max() < 2e-5   # on the camera ray
    res = _unsigned_surface_distance(o_pre[anchored] + 1e-3 * dcam[anchored], sc)
    assert res.max() < 5e-5, res.max()                                     # 1e-3 before the surface, not on or beyond it
    assert (anchored & ~shifted).sum() > 10000 and shifted.sum() > 10000
