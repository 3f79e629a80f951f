"""Wavefront secondary rays: CPU pins of the oracle twin,
then the CUDA path (compaction + second query + lit flags) against it through the C ABI."""
import math

import numpy as np
import pytest

from ddf_inputs import MASTER_SEED, STREAMS, layout_c1, layout_hash_paper, make_weights, make_hash_table, make_hash_mlp, random_rays


# ------------------------------------------------------------------ CPU: the twin against geometry

def test_twin_on_an_analytic_sphere(orc):
    """Feed the twin the EXACT field of a unit sphere (dist = ray-sphere distance, vis = hit): the
    secondary origins lie eps inside the ray from the surface, directions are unit and aim at the
    light, tmax is the light distance, the index list is the increasing list of hits."""
    ocam = orc.make_camera((0.0, -2.5, 0.0))
    o, d = orc.gen_camera(ocam, 64, 64)
    t = np.array([orc.ray_sphere(o[i], d[i], (0, 0, 0), 1.0) for i in range(len(o))])
    vis = (t > 0).astype(np.float32); dist = np.where(t > 0, t, 0.0).astype(np.float32)
    L = np.array([3.0, 3.0, 3.0])
    o2, d2, tmax, idx = orc.gen_shadow_from_hits(o, d, dist, vis, L, 1e-3)
    assert np.array_equal(idx, np.nonzero(vis > 0.5)[0]) and 0 < len(idx) < len(o)
    hit = o[idx].astype(np.float64) + dist[idx, None].astype(np.float64) * d[idx]
    assert np.allclose(np.linalg.norm(hit, axis=1), 1.0, atol=1e-5)
    assert np.allclose(np.linalg.norm(o2 - hit, axis=1), 1e-3, atol=2e-6)          # stepped back by eps ...
    assert np.all(np.einsum("ij,ij->i", o2 - hit, d[idx]) < 0)                      # ... against the ray
    assert np.allclose(np.linalg.norm(d2, axis=1), 1.0, atol=1e-6)
    assert np.allclose(o2 + tmax[:, None] * d2, L[None, :], atol=1e-5)
    # lit flags with the exact field again: a point of the sphere is lit iff its shadow ray leaves the sphere
    t2 = np.array([orc.ray_sphere(o2[k], d2[k], (0, 0, 0), 1.0) for k in range(len(idx))])
    vis2 = (t2 > 0).astype(np.float32); dist2 = np.where(t2 > 0, t2, 0).astype(np.float32)
    lit = orc.shadow_lit(vis2, dist2, tmax, idx, len(o))
    facing = np.einsum("ij,ij->i", hit, L[None, :] - hit) > 0                       # n . (L - p) > 0
    inside_margin = np.abs(np.einsum("ij,ij->i", hit, L[None, :] - hit)) > 0.3      # away from the terminator (the eps offset lifts grazing rays over the horizon)
    assert np.array_equal(lit[idx][inside_margin].astype(bool), facing[inside_margin])
    assert lit[np.nonzero(vis < 0.5)[0]].sum() == 0                                 # primary misses are never lit


def _plane_t(o, d, z0):
    """distance of rays to the plane z = z0 (inf where they do not reach it)"""
    with np.errstate(divide="ignore", invalid="ignore"):
        t = (z0 - o[:, 2].astype(np.float64)) / d[:, 2].astype(np.float64)
    return np.where(np.isfinite(t) & (t > 0), t, np.inf)


def test_hit_normals_on_exact_fields(orc):
    """Reading W5 against geometry.  Exact plane field: every normal is the plane's, facing the camera.
    Exact sphere field: normals are P / |P| up to the finite-difference error of one pixel.
    Sphere in front of a plane: plane pixels beside the silhouette keep the plane normal, because the
    difference goes to the neighbour with the smaller distance jump (an always-forward rule fails)."""
    W, H = 96, 80
    ocam = orc.make_camera((0.3, -0.4, 2.5))
    o, d = orc.gen_camera(ocam, W, H)
    tp = _plane_t(o, d, -1.0)
    assert np.all(np.isfinite(tp))
    vis = np.ones(W * H, np.float32)
    p, nrm, idx = orc.hit_normals(o, d, tp.astype(np.float32), vis, W, H)
    assert np.array_equal(idx, np.arange(W * H))
    assert np.allclose(p[:, 2], -1.0, atol=1e-5)
    assert np.allclose(nrm, np.array([0.0, 0.0, 1.0])[None, :], atol=2e-3)          # fp32 distances: ~1e-7 / pixel footprint
    # sphere alone
    ts = np.array([orc.ray_sphere(o[i], d[i], (0, 0, 0), 1.0) for i in range(W * H)])
    vis = (ts > 0).astype(np.float32); dist = np.where(ts > 0, ts, 0.0).astype(np.float32)
    p, nrm, idx = orc.hit_normals(o, d, dist, vis, W, H)
    assert np.array_equal(idx, np.nonzero(vis > 0.5)[0]) and 0 < len(idx) < W * H
    assert np.allclose(np.linalg.norm(nrm, axis=1), 1.0, atol=1e-6)
    assert np.all(np.einsum("ij,ij->i", nrm, d[idx]) <= 1e-6)                       # faces the camera
    true_n = p / np.linalg.norm(p, axis=1, keepdims=True)
    front = -np.einsum("ij,ij->i", true_n, d[idx]) > 0.4                            # away from the silhouette
    cosang = np.einsum("ij,ij->i", nrm, true_n)[front]
    assert front.sum() > 500 and np.degrees(np.arccos(np.clip(cosang, -1, 1))).max() < 2.5
    # sphere in front of the plane
    both = np.minimum(np.where(ts > 0, ts, np.inf), tp)
    on_plane = ~(ts > 0)
    p, nrm, idx = orc.hit_normals(o, d, both.astype(np.float32), np.ones(W * H, np.float32), W, H)
    img = nrm.reshape(H, W, 3); pl = on_plane.reshape(H, W)
    nb_x = np.zeros_like(pl); nb_x[:, 1:] |= pl[:, :-1]; nb_x[:, :-1] |= pl[:, 1:]  # a plane neighbour on each axis
    nb_y = np.zeros_like(pl); nb_y[1:, :] |= pl[:-1, :]; nb_y[:-1, :] |= pl[1:, :]
    sel = pl & nb_x & nb_y
    beside = sel.copy(); beside[:, :-1] &= ~pl[:, 1:]                               # forward x-neighbour is on the sphere
    assert beside[:, :-1].sum() > 10
    assert np.allclose(img[sel], np.array([0.0, 0.0, 1.0])[None, :], atol=2e-3)


def test_hit_normals_hand_cases(orc):
    """Ties go forward, an axis without a hit neighbour falls back to -d, misses are skipped."""
    a = 0.25
    xs, ys = np.meshgrid(np.arange(3.0), np.arange(3.0))                            # 3 x 3 parallel rays along +z
    o = np.stack([xs.ravel(), ys.ravel(), np.zeros(9)], 1).astype(np.float32)
    d = np.tile(np.array([0.0, 0.0, 1.0], np.float32), (9, 1))
    dist = (1.0 + a * np.abs(xs.ravel() - 1.0)).astype(np.float32)                  # a V-shaped valley along x = 1
    vis = np.ones(9, np.float32)
    p, nrm, idx = orc.hit_normals(o, d, dist, vis, 3, 3)
    s = math.sqrt(1 + a * a)
    # centre pixel: |dt| ties, forward: du = (1, 0, a), dv = (0, 1, 0): du x dv = (-a, 0, 1), turned against d
    assert np.allclose(nrm[4], [a / s, 0.0, -1.0 / s], atol=1e-6)
    # left column has only a forward x-neighbour: du = (1, 0, -a) -> (a, 0, 1) -> turned: (-a, 0, -1) / s
    assert np.allclose(nrm[3], [-a / s, 0.0, -1.0 / s], atol=1e-6)
    # an isolated hit and a one-row image: no y-neighbour -> -d
    vis1 = np.zeros(9, np.float32); vis1[4] = 1.0
    p, nrm, idx = orc.hit_normals(o, d, dist, vis1, 3, 3)
    assert list(idx) == [4] and np.allclose(nrm[0], [0, 0, -1]) and np.allclose(p[0], [1, 1, 1])
    p, nrm, idx = orc.hit_normals(o[:3], d[:3], dist[:3], vis[:3], 3, 1)
    assert len(idx) == 3 and np.allclose(nrm, [[0, 0, -1]] * 3)
    # the smaller jump wins: make the forward neighbour of the centre far away
    dist2 = dist.copy(); dist2[5] = 5.0
    p, nrm, idx = orc.hit_normals(o, d, dist2, vis, 3, 3)
    assert np.allclose(nrm[4], [-a / s, 0.0, -1.0 / s], atol=1e-6)                  # backward: du = (1, 0, -a)
    # threshold: vis exactly 0.5 is a miss
    vis2 = vis.copy(); vis2[0] = 0.5
    assert 0 not in orc.hit_normals(o, d, dist, vis2, 3, 3)[2]


def test_twin_threshold_and_order(orc):
    o = np.zeros((6, 3), np.float32); d = np.tile(np.array([[0, 0, 1]], np.float32), (6, 1))
    dist = np.arange(1, 7, dtype=np.float32)
    vis = np.array([0.5, 0.50001, 0.2, 1.0, 0.4999, 0.9], np.float32)               # ties (0.5) are misses (A10)
    o2, d2, tmax, idx = orc.gen_shadow_from_hits(o, d, dist, vis, (0, 0, 10), 0.25)
    assert list(idx) == [1, 3, 5]
    assert np.allclose(o2[:, 2], [1.75, 3.75, 5.75]) and np.allclose(tmax, [8.25, 6.25, 4.25])
    lit = orc.shadow_lit(np.array([0.9, 0.9, 0.1], np.float32), np.array([1.0, 7.0, 1.0], np.float32), tmax, idx, 6)
    assert list(lit) == [0, 0, 0, 1, 0, 1]                                          # occluded only if dist2 < tmax


# ------------------------------------------------------------------ GPU

def _models(ddf):
    """both model kinds, with the visibility-head bias raised to 1 so that hits and occlusions are
    common (the seeded random fields otherwise answer xi ~ 0.3 almost everywhere)"""
    lay = layout_c1()
    blob = make_weights(lay).copy()
    blob[-1] = 0x3F80                                         # bf16 bits of 1.0: bias of the visibility logit
    yield "dense", ddf.ddf_create(blob, lay), lambda orc, o, d: orc.forward(lay, blob, o, d)
    hl = layout_hash_paper()
    n = ddf.ddf_hashgrid_table_entries(hl)
    tab, mlp = make_hash_table(hl, n), make_hash_mlp(hl).copy()
    mlp[-1] = 1.0
    yield "hash", ddf.ddf_create_hashgrid(tab, mlp, hl), lambda orc, o, d: orc.hash_forward(hl, tab, mlp, o, d)


@pytest.mark.gpu
def test_gpu_wavefront_against_twin(orc):
    import torch
    import paper_2606_00817_b200 as ddf
    ddf.build()
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    W = H = 384; n = W * H
    light = (3.0, 3.0, 3.0)
    for name, m, oracle_fwd in _models(ddf):
        o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
        ddf.ddf_gen_camera(cam, W, H, o, d)
        # spread the origins so that hits and misses mix (with one shared origin the seeded random
        # fields answer nearly the same xi for every direction)
        o += torch.from_numpy(random_rays(n)[0]).cuda() * 0.4
        dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
        lit = torch.full((n,), 7, dtype=torch.uint8, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
        ddf.ddf_query_shadowed(m, o, d, n, light, 1e-3, dist, vis, lit, cnt)
        torch.cuda.synchronize()
        k = int(cnt.item())
        # primary results are exactly ddf_query's
        d1 = torch.empty(n, device="cuda"); v1 = torch.empty(n, device="cuda")
        ddf.ddf_query(m, o, d, n, d1, v1)
        assert torch.equal(d1, dist) and torch.equal(v1, vis)
        assert k == int((vis > 0.5).sum().item()) and 0 < k < n, (name, k)
        # compaction against the twin on the GPU's own primary results: indices bit-exact, rays to 1e-5
        o2 = torch.empty((n, 3), device="cuda"); d2 = torch.empty((n, 3), device="cuda")
        tmax = torch.empty(n, device="cuda"); idx = torch.empty(n, dtype=torch.int32, device="cuda"); c2 = torch.zeros(1, dtype=torch.int64, device="cuda")
        ddf.ddf_gen_shadow_from_hits(m, o, d, dist, vis, n, light, 1e-3, o2, d2, tmax, idx, c2)
        assert int(c2.item()) == k
        ro2, rd2, rt, ridx = orc.gen_shadow_from_hits(o.cpu().numpy(), d.cpu().numpy(), dist.cpu().numpy(), vis.cpu().numpy(), light, 1e-3)
        assert np.array_equal(idx[:k].cpu().numpy(), ridx)
        assert np.allclose(o2[:k].cpu().numpy(), ro2, atol=2e-6) and np.allclose(d2[:k].cpu().numpy(), rd2, atol=1e-5)
        assert np.allclose(tmax[:k].cpu().numpy(), rt, rtol=1e-6)
        # lit flags = the decision rule applied to a plain second query of the compacted batch
        dist2 = torch.empty(k, device="cuda"); vis2 = torch.empty(k, device="cuda")
        ddf.ddf_query(m, o2[:k].contiguous(), d2[:k].contiguous(), k, dist2, vis2)
        want = orc.shadow_lit(vis2.cpu().numpy(), dist2.cpu().numpy(), tmax[:k].cpu().numpy(), ridx, n)
        assert np.array_equal(lit.cpu().numpy(), want), name
        assert 0 < int(lit.sum().item()) < k                 # both outcomes occur
        # ... and against the oracle end to end on a sample of hit rays, away from the two thresholds
        sel = np.arange(0, k, max(1, k // 400))[:400]
        z, t2, xi2 = oracle_fwd(orc, ro2[sel], rd2[sel])
        safe = (np.abs(xi2 - 0.5) > 1e-2) & (np.abs(t2 - rt[sel]) > 1e-2 * (1 + np.abs(t2)))
        ref = ~((xi2 > 0.5) & (t2 < rt[sel]))
        got = lit.cpu().numpy()[ridx[sel]].astype(bool)
        assert np.array_equal(got[safe], ref[safe]) and safe.mean() > 0.5, name
        # several lights: bit j of the mask is the single-light answer for light j (verified above for the first),
        # the primary results are the same, every hit is traced once per light
        lights = [light, (-3.0, 2.0, 1.0), (0.5, -4.0, 2.5)]
        mask = torch.full((n,), 0xAA, dtype=torch.uint8, device="cuda"); c3 = torch.zeros(1, dtype=torch.int64, device="cuda")
        dm = torch.empty(n, device="cuda"); vm = torch.empty(n, device="cuda")
        ddf.ddf_query_shadowed_lights(m, o, d, n, lights, 1e-3, dm, vm, mask, c3)
        assert int(c3.item()) == 3 * k and torch.equal(dm, dist) and torch.equal(vm, vis)
        assert int(mask.max().item()) < 8
        for j, lj in enumerate(lights):
            one = torch.empty(n, dtype=torch.uint8, device="cuda")
            ddf.ddf_query_shadowed(m, o, d, n, lj, 1e-3, dist, vis, one, None)
            assert torch.equal((mask >> j) & 1, one), (name, j)
            if j:                                            # the other lights against the oracle too, on a sample
                qo2, qd2, qt, qidx = orc.gen_shadow_from_hits(o.cpu().numpy(), d.cpu().numpy(), dist.cpu().numpy(), vis.cpu().numpy(), lj, 1e-3)
                z, t2, xi2 = oracle_fwd(orc, qo2[sel], qd2[sel])
                safe = (np.abs(xi2 - 0.5) > 1e-2) & (np.abs(t2 - qt[sel]) > 1e-2 * (1 + np.abs(t2)))
                ref = ~((xi2 > 0.5) & (t2 < qt[sel]))
                got = one.cpu().numpy()[qidx[sel]].astype(bool)
                assert np.array_equal(got[safe], ref[safe]) and safe.mean() > 0.5, (name, j)
        assert len(set(int(x) for x in mask.unique().cpu())) > 2          # the lights disagree somewhere
        # n = 0 and determinism
        ddf.ddf_query_shadowed(m, o, d, 0, light, 1e-3, dist, vis, lit, cnt)
        assert int(cnt.item()) == 0
        lit2 = torch.empty(n, dtype=torch.uint8, device="cuda")
        ddf.ddf_query_shadowed(m, o, d, n, light, 1e-3, dist, vis, lit2, None)
        assert torch.equal(lit2, torch.from_numpy(want).cuda())
        ddf.ddf_destroy(m)


@pytest.mark.gpu
def test_gpu_compaction_edge_cases(orc):
    """all hits, no hits, one hit at the end, sizes around the 256-ray scan block and a 2^22 batch"""
    import torch
    import paper_2606_00817_b200 as ddf
    from ddf_inputs import layout_c0
    ddf.build()
    m = ddf.ddf_create(make_weights(layout_c0()), layout_c0())
    g = torch.Generator(device="cuda").manual_seed(3)
    for n, mode in [(1, "all"), (255, "none"), (256, "all"), (257, "last"), (1000, "rand"), (65537, "rand"), (1 << 22, "rand")]:
        o = torch.rand((n, 3), device="cuda", generator=g); d = torch.nn.functional.normalize(torch.randn((n, 3), device="cuda", generator=g), dim=1)
        dist = torch.rand(n, device="cuda", generator=g) + 0.5
        vis = {"all": torch.ones(n, device="cuda"), "none": torch.zeros(n, device="cuda"),
               "last": torch.zeros(n, device="cuda"), "rand": torch.rand(n, device="cuda", generator=g)}[mode]
        if mode == "last": vis[-1] = 1.0
        o2 = torch.empty((n, 3), device="cuda"); d2 = torch.empty((n, 3), device="cuda"); tmax = torch.empty(n, device="cuda")
        idx = torch.full((n,), -1, dtype=torch.int32, device="cuda"); cnt = torch.full((1,), -5, dtype=torch.int64, device="cuda")
        ddf.ddf_gen_shadow_from_hits(m, o, d, dist, vis, n, (1.0, 2.0, 3.0), 1e-2, o2, d2, tmax, idx, cnt)
        want = torch.nonzero(vis > 0.5).flatten().to(torch.int32)
        k = int(cnt.item())
        assert k == len(want) and torch.equal(idx[:k], want), (n, mode)
        assert bool((idx[k:] == -1).all())
        if k:
            p = o[want.long()] + (dist[want.long()] - 1e-2)[:, None] * d[want.long()]
            assert torch.allclose(o2[:k], p, atol=1e-6)
    ddf.ddf_destroy(m)


@pytest.mark.gpu
def test_gpu_hit_normals_on_an_exact_sphere_field(orc):
    """ddf_gen_ao_from_hits fed the exact field of a unit sphere in front of a plane: the compacted index is
    the oracle's, hit points and normals agree with it (smooth data: no sign or neighbour ambiguity), and the
    rays are the oracle's generator run on them."""
    import torch
    import paper_2606_00817_b200 as ddf
    from ddf_inputs import layout_c0
    ddf.build()
    m = ddf.ddf_create(make_weights(layout_c0()), layout_c0())
    for (W, H) in [(96, 80), (257, 3), (1, 1), (5, 1), (1, 300)]:
        ocam = orc.make_camera((0.3, -0.4, 2.5))
        o, d = orc.gen_camera(ocam, W, H)
        ts = np.array([orc.ray_sphere(o[i], d[i], (0, 0, 0), 1.0) for i in range(W * H)])
        tp = _plane_t(o, d, -1.0)
        dist = np.minimum(np.where(ts > 0, ts, np.inf), tp).astype(np.float32)
        vis = np.ones(W * H, np.float32); vis[::7] = 0.0                                # holes: one-sided differences
        rp, rn, ridx = orc.hit_normals(o, d, dist, vis, W, H)
        n = W * H; spp = 4
        og, dg, tg, vg = (torch.from_numpy(x).cuda() for x in (o, d, dist, vis))
        p_c = torch.empty((n, 3), device="cuda"); n_c = torch.empty((n, 3), device="cuda")
        idx = torch.full((n,), -1, dtype=torch.int32, device="cuda"); cnt = torch.full((1,), -5, dtype=torch.int64, device="cuda")
        o2 = torch.full((n * spp, 3), float("nan"), device="cuda"); d2 = torch.full((n * spp, 3), float("nan"), device="cuda")
        ddf.ddf_gen_ao_from_hits(m, og, dg, tg, vg, W, H, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3, p_c, n_c, idx, o2, d2, cnt)
        torch.cuda.synchronize()
        k = int(cnt.item())
        assert k == len(ridx) and np.array_equal(idx[:k].cpu().numpy(), ridx) and bool((idx[k:] == -1).all()), (W, H)
        assert np.allclose(p_c[:k].cpu().numpy(), rp, atol=2e-6)
        # fp32 differences of neighbouring hit points: 1e-7 against a pixel footprint of ~1e-2 .. 3e-2
        assert np.allclose(n_c[:k].cpu().numpy(), rn, atol=5e-4), (W, H, np.abs(n_c[:k].cpu().numpy() - rn).max())
        ro2, rd2 = orc.gen_ao(p_c[:k].cpu().numpy(), n_c[:k].cpu().numpy(), spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3)
        assert np.allclose(o2[:k * spp].cpu().numpy(), ro2, atol=1e-5) and np.allclose(d2[:k * spp].cpu().numpy(), rd2, atol=2e-5)
        assert bool(torch.isnan(o2[k * spp:]).all())                                     # nothing past the count
        # normals only
        ddf.ddf_gen_ao_from_hits(m, og, dg, tg, vg, W, H, spp, 0, 0, 1e-3, p_c, n_c, idx, None, None, cnt)
        assert int(cnt.item()) == k and ddf.ddf_get_info(m, 1) == 3
    # no hits at all, empty image
    z = torch.zeros(64, device="cuda")
    ddf.ddf_gen_ao_from_hits(m, og[:64].contiguous(), dg[:64].contiguous(), tg[:64].contiguous(), z, 8, 8, 4, 1, 2, 1e-3,
                             p_c, n_c, idx, o2, d2, cnt)
    assert int(cnt.item()) == 0
    cnt.fill_(9)
    ddf.ddf_gen_ao_from_hits(m, None, None, None, None, 0, 5, 4, 1, 2, 1e-3, None, None, None, None, None, cnt)
    assert int(cnt.item()) == 0
    ddf.ddf_destroy(m)


@pytest.mark.gpu
def test_gpu_ao_wavefront_against_twin(orc):
    """ddf_query_ao_wavefront: primary results are ddf_query's; hits, hit points, normals and rays follow the twin
    on the GPU's own primary results; the AO image is the decision rule applied to a plain second query of the
    compacted rays (bit for bit) and agrees with the oracle evaluated end to end on sampled pixels."""
    import torch
    import paper_2606_00817_b200 as ddf
    ddf.build()
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    for name, m, oracle_fwd in _models(ddf):
        for (W, H, spp, radius) in [(256, 192, 16, 1.5), (61, 47, 5, float("inf"))]:   # fused reduce / host-counted path
            n = W * H
            o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
            ddf.ddf_gen_camera(cam, W, H, o, d)
            o += torch.from_numpy(random_rays(n)[0]).cuda() * 0.4
            dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda"); nrm = torch.full((n, 3), 9.0, device="cuda")
            ao = torch.full((n,), float("nan"), device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
            seed, stream = MASTER_SEED, STREAMS["ao_samples"]
            ddf.ddf_query_ao_wavefront(m, o, d, W, H, spp, seed, stream, 1e-3, radius, dist, vis, nrm, ao, cnt)
            torch.cuda.synchronize()
            d1 = torch.empty(n, device="cuda"); v1 = torch.empty(n, device="cuda")
            ddf.ddf_query(m, o, d, n, d1, v1)
            assert torch.equal(d1, dist) and torch.equal(v1, vis)
            k = int((vis > 0.5).sum().item())
            assert int(cnt.item()) == k * spp and 0 < k < n, (name, k)
            # the twin on the GPU's primary results
            on, dn, tn, vn = o.cpu().numpy(), d.cpu().numpy(), dist.cpu().numpy(), vis.cpu().numpy()
            rp, rn, ridx = orc.hit_normals(on, dn, tn, vn, W, H)
            p_c = torch.empty((n, 3), device="cuda"); n_c = torch.empty((n, 3), device="cuda"); idx = torch.empty(n, dtype=torch.int32, device="cuda")
            o2 = torch.empty((n * spp, 3), device="cuda"); d2 = torch.empty((n * spp, 3), device="cuda"); c2 = torch.zeros(1, dtype=torch.int64, device="cuda")
            ddf.ddf_gen_ao_from_hits(m, o, d, dist, vis, W, H, spp, seed, stream, 1e-3, p_c, n_c, idx, o2, d2, c2)
            assert int(c2.item()) == k and np.array_equal(idx[:k].cpu().numpy(), ridx)
            assert np.allclose(p_c[:k].cpu().numpy(), rp, atol=4e-6)
            ng = n_c[:k].cpu().numpy()
            grazing = np.abs(np.einsum("ij,ij->i", rn, dn[ridx])) < 1e-3                 # the turn against the ray may flip
            err = np.minimum(np.abs(ng - rn).max(1), np.where(grazing, np.abs(ng + rn).max(1), np.inf))
            assert (err < 1e-3).mean() > 0.999 and grazing.mean() < 0.01, (name, err.max())
            assert np.allclose(np.linalg.norm(ng, axis=1), 1.0, atol=1e-5)
            img = nrm.cpu().numpy()
            assert np.array_equal(img[ridx], ng) and not img[vn <= 0.5].any()             # per-pixel copy, 0 on misses
            ro2, rd2 = orc.gen_ao(p_c[:k].cpu().numpy(), ng, spp, seed, stream, 1e-3)
            assert np.allclose(o2[:k * spp].cpu().numpy(), ro2, atol=1e-5) and np.allclose(d2[:k * spp].cpu().numpy(), rd2, atol=2e-5)
            # AO = the rule on a plain second query of those rays, scattered back; misses = 1
            dist2 = torch.empty(k * spp, device="cuda"); vis2 = torch.empty(k * spp, device="cuda")
            ddf.ddf_query(m, o2[:k * spp].contiguous(), d2[:k * spp].contiguous(), k * spp, dist2, vis2)
            want = np.ones(n, np.float32)
            want[ridx] = orc.ao_reduce(vis2.cpu().numpy(), dist2.cpu().numpy(), spp, radius)
            if spp & (spp - 1) == 0: assert np.array_equal(ao.cpu().numpy(), want), (name, W, spp)
            else: assert np.allclose(ao.cpu().numpy(), want, atol=1e-6, rtol=0), (name, W, spp)   # hits / spp rounds in fp32 on the GPU, fp64 in the oracle
            assert 0.0 < want[ridx].mean() < 1.0
            # the oracle end to end on sampled pixels
            sel = np.arange(0, k, max(1, k // 100))[:100]
            rows = (sel[:, None] * spp + np.arange(spp)[None, :]).reshape(-1)
            z, t2, xi2 = oracle_fwd(orc, ro2[rows], rd2[rows])
            ref = orc.ao_reduce(xi2.astype(np.float32), t2.astype(np.float32), spp, radius)
            near = ((np.abs(xi2 - 0.5) < 1e-2) | (np.abs(t2 - radius) < 1e-2 * (1 + np.abs(t2)))).reshape(-1, spp).sum(1)
            assert np.all(np.abs(want[ridx[sel]] - ref) <= near / spp + 1e-6), name
            # determinism
            ao_b = torch.empty(n, device="cuda")
            ddf.ddf_query_ao_wavefront(m, o, d, W, H, spp, seed, stream, 1e-3, radius, dist, vis, None, ao_b, None)
            assert torch.equal(ao_b, ao)
        ddf.ddf_query_ao_wavefront(m, o, d, 0, 7, 4, 1, 2, 1e-3, 1.0, dist, vis, None, ao, cnt)
        assert int(cnt.item()) == 0
        ddf.ddf_destroy(m)


@pytest.mark.gpu
def test_gpu_shaded_frame_is_the_two_loops_on_one_primary_query(orc):
    """ddf_query_shaded = ddf_query + the shadow loop + the AO loop on the same primary results: every output
    bit for bit what ddf_query_shadowed_lights and ddf_query_ao_wavefront return, one primary query fewer."""
    import torch
    import paper_2606_00817_b200 as ddf
    ddf.build()
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    W, H, spp = 200, 160, 8; n = W * H
    lights = [(3.0, 3.0, 3.0), (-3.0, 2.0, 1.0)]
    for name, m, _ in _models(ddf):
        o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
        ddf.ddf_gen_camera(cam, W, H, o, d)
        o += torch.from_numpy(random_rays(n)[0]).cuda() * 0.4
        new = lambda *s, dt=torch.float32, v=0: torch.full(s, v, dtype=dt, device="cuda")
        dist_a, vis_a, mask_a, c_a = new(n), new(n), new(n, dt=torch.uint8), new(1, dt=torch.int64)
        ddf.ddf_query_shadowed_lights(m, o, d, n, lights, 1e-3, dist_a, vis_a, mask_a, c_a)
        l_a = ddf.ddf_get_info(m, 1)
        dist_b, vis_b, nrm_b, ao_b, c_b = new(n), new(n), new(n, 3), new(n), new(1, dt=torch.int64)
        ddf.ddf_query_ao_wavefront(m, o, d, W, H, spp, 5, 6, 1e-3, 2.0, dist_b, vis_b, nrm_b, ao_b, c_b)
        l_b = ddf.ddf_get_info(m, 1)
        ddf.ddf_query(m, o, d, n, dist_b, vis_b)
        l_q = ddf.ddf_get_info(m, 1)
        dist, vis, mask, nrm, ao, cs = new(n, v=7), new(n, v=7), new(n, dt=torch.uint8, v=0xFF), new(n, 3, v=7), new(n, v=7), new(2, dt=torch.int64, v=-1)
        ddf.ddf_query_shaded(m, o, d, W, H, lights, spp, 5, 6, 1e-3, 2.0, dist, vis, mask, nrm, ao, cs)
        torch.cuda.synchronize()
        assert ddf.ddf_get_info(m, 1) == l_a + l_b - l_q, name
        assert torch.equal(dist, dist_a) and torch.equal(vis, vis_a) and torch.equal(mask, mask_a), name
        assert torch.equal(nrm, nrm_b) and torch.equal(ao, ao_b), name
        assert cs.tolist() == [int(c_a.item()), int(c_b.item())] and cs[0] > 0 and cs[1] > 0
        # one loop only
        mask2, cs2 = new(n, dt=torch.uint8, v=0xFF), new(2, dt=torch.int64, v=-1)
        ddf.ddf_query_shaded(m, o, d, W, H, lights, 0, 0, 0, 1e-3, 2.0, dist, vis, mask2, None, None, cs2)
        assert torch.equal(mask2, mask_a) and cs2.tolist() == [int(c_a.item()), 0]
        ao2, cs3 = new(n, v=7), new(2, dt=torch.int64, v=-1)
        ddf.ddf_query_shaded(m, o, d, W, H, [], spp, 5, 6, 1e-3, 2.0, dist, vis, None, None, ao2, cs3)
        assert torch.equal(ao2, ao_b) and cs3.tolist() == [0, int(c_b.item())]
        ddf.ddf_query_shaded(m, o, d, 0, 0, lights, spp, 5, 6, 1e-3, 2.0, dist, vis, mask, nrm, ao, cs)
        assert cs.tolist() == [0, 0]
        with pytest.raises(ddf.DdfError):
            ddf.ddf_query_shaded(m, o, d, W, H, lights, spp, 5, 6, 1e-3, 2.0, dist, vis, None, nrm, ao, cs)
        ddf.ddf_destroy(m)


@pytest.mark.gpu
@pytest.mark.parametrize("path", [0, 1])                 # narrow tcgen05 kernel (count stays on the device) / CUDA-core path (host-counted)
def test_gpu_ao_wavefront_on_the_narrow_and_cuda_core_paths(orc, path):
    import torch
    import paper_2606_00817_b200 as ddf
    from ddf_inputs import layout_c0
    ddf.build()
    m = ddf.ddf_create(make_weights(layout_c0()), layout_c0())
    ddf.ddf_set_path(m, path)
    W, H, spp = 64, 48, 8; n = W * H
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o = torch.empty((n, 3), device="cuda"); d = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, W, H, o, d)
    o += torch.from_numpy(random_rays(n)[0]).cuda() * 0.4
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda"); ao = torch.full((n,), float("nan"), device="cuda")
    cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    ddf.ddf_query_ao_wavefront(m, o, d, W, H, spp, 3, 4, 1e-3, 1.0, dist, vis, None, ao, cnt)
    torch.cuda.synchronize()
    k = int((vis > 0.5).sum().item())
    assert int(cnt.item()) == k * spp and 0 < k < n
    p_c = torch.empty((n, 3), device="cuda"); n_c = torch.empty((n, 3), device="cuda"); idx = torch.empty(n, dtype=torch.int32, device="cuda")
    o2 = torch.empty((n * spp, 3), device="cuda"); d2 = torch.empty((n * spp, 3), device="cuda"); c2 = torch.zeros(1, dtype=torch.int64, device="cuda")
    ddf.ddf_gen_ao_from_hits(m, o, d, dist, vis, W, H, spp, 3, 4, 1e-3, p_c, n_c, idx, o2, d2, c2)
    rp, rn, ridx = orc.hit_normals(o.cpu().numpy(), d.cpu().numpy(), dist.cpu().numpy(), vis.cpu().numpy(), W, H)
    assert int(c2.item()) == k and np.array_equal(idx[:k].cpu().numpy(), ridx)
    dist2 = torch.empty(k * spp, device="cuda"); vis2 = torch.empty(k * spp, device="cuda")
    ddf.ddf_query(m, o2[:k * spp].contiguous(), d2[:k * spp].contiguous(), k * spp, dist2, vis2)
    want = np.ones(n, np.float32)
    want[ridx] = orc.ao_reduce(vis2.cpu().numpy(), dist2.cpu().numpy(), spp, 1.0)
    assert np.array_equal(ao.cpu().numpy(), want) and 0.0 < want[ridx].mean() < 1.0
    ddf.ddf_destroy(m)
