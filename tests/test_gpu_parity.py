"""GPU parity: the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.

Tolerances (BASELINE.json north_star), against the EXACT fp64 oracle:
    |dd| <= 1e-2 (1 + |d|),   |dv| <= 1e-2,   hit/miss (xi > 0.5) agreement >= 99.9 % outside
    the band |xi - 0.5| < 1e-2.
Second, tighter comparison against the oracle's QUANTISED mode (bf16 rounding at the GPU's
rounding points, A11): |dz| <= 4e-2 on the logits and a mean below 3e-3 - bf16
rounding flips caused by fp32-vs-fp64 accumulation keep it from being exact, but a dropped
K block, a leaking pad lane or a mis-ordered skip is O(0.1 - 1).
"""
import math

import numpy as np
import pytest
import torch

from ddf_inputs import (MASTER_SEED, STREAMS, Layout, layout_c0, layout_c1, layout_sdf, make_weights,
                        random_rays, blob_layer_shapes, blob_num_elements)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ddf():
    import paper_2606_00817_b200 as pkg
    pkg.build()
    assert torch.cuda.is_available()
    return pkg


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _query(ddf, model, o, d, logits=False):
    n = o.shape[0]
    od, dd = _cuda(o), (_cuda(d) if d is not None else None)
    if logits:
        z = torch.full((n, model.layout.n_out), float("nan"), device="cuda")
        ddf.ddf_query_logits(model, od, dd, n, z)
        torch.cuda.synchronize()
        return z.cpu().numpy()
    dist = torch.full((n,), float("nan"), device="cuda")
    vis = torch.full((n,), float("nan"), device="cuda")
    ddf.ddf_query(model, od, dd, n, dist, vis)
    torch.cuda.synchronize()
    return dist.cpu().numpy(), vis.cpu().numpy()


def check_parity(dist, vis, t_ref, xi_ref, what=""):
    """north_star tolerances against the exact oracle; returns the statistics."""
    ed = np.abs(dist - t_ref) / (1.0 + np.abs(t_ref))
    ev = np.abs(vis - xi_ref)
    band = np.abs(xi_ref - 0.5) < 1e-2
    agree = ((vis > 0.5) == (xi_ref > 0.5))[~band].mean() if (~band).any() else 1.0
    stats = dict(max_d=float(ed.max()), max_v=float(ev.max()), p999_d=float(np.quantile(ed, 0.999)),
                 agree=float(agree), band_frac=float(band.mean()))
    assert np.all(np.isfinite(dist)) and np.all(np.isfinite(vis)), what
    assert ed.max() <= 1e-2, (what, stats)
    assert ev.max() <= 1e-2, (what, stats)
    assert agree >= 0.999, (what, stats)
    assert band.mean() < 0.2, (what, stats)          # logits are O(1), not collapsed (reading A7)
    return stats


def check_quantised(z_gpu, z_q, what="", max_tol=4.5e-2, mean_tol=2e-3):
    """Second gate: logits against the oracle's quantised mode (same bf16 rounding points, fp64 sums).  Most logits agree
    to ~1e-6; the tail comes from hidden activations that sit on a bf16 rounding boundary and round the other way under
    the kernel's fp32 summation order - one flip moves one activation by 2^-8 of its value and the remaining layers
    carry it to the logit.  Bounds are ~2x what the committed kernels measure (printed below on every run):
    the defaults are for the 8 x 1280 network on >= 8,192 rays (measured max 2.1e-2, mean 9.6e-4), shallower or narrower
    networks pass their own."""
    e = np.abs(z_gpu - z_q)
    print("QUANT %-40s n=%6d max %.3e mean %.3e rays above 1e-3: %d" % (what, e.shape[0], float(e.max()), float(e.mean()),
                                                                        int((e.reshape(e.shape[0], -1).max(1) > 1e-3).sum())))
    assert e.max() <= max_tol and e.mean() <= mean_tol, (what, float(e.max()), float(e.mean()), max_tol, mean_tol)


# ------------------------------------------------------------------ configs[0]: all 4096 rays

@pytest.fixture(scope="module")
def c0(ddf):
    lay = layout_c0()
    blob = make_weights(lay)
    m = ddf.ddf_create(blob, lay)
    yield lay, blob, m
    ddf.ddf_destroy(m)


def test_config0_all_rays(ddf, orc, c0):
    lay, blob, m = c0
    o, d = random_rays(4096)
    dist, vis = _query(ddf, m, o, d)
    z, t, xi = orc.forward(lay, blob, o, d, mode=0)
    check_parity(dist, vis, t, xi, "C0")
    zq, _, _ = orc.forward(lay, blob, o, d, mode=1)
    check_quantised(_query(ddf, m, o, d, logits=True), zq, "C0 quantised", max_tol=5e-3, mean_tol=2e-6)   # measured 2.2e-3 / 4.5e-7


# ------------------------------------------------------------------ paper-scale network

@pytest.fixture(scope="module")
def c1(ddf):
    lay = layout_c1()
    blob = make_weights(lay)
    m = ddf.ddf_create(blob, lay)
    assert ddf.ddf_get_info(m, 0) == 1, "the tcgen05 path must serve configs[1]"
    yield lay, blob, m
    ddf.ddf_destroy(m)


def _sample(n, k=8192):
    """the first and last tile, every tile boundary +-1 of the first 64 tiles, whole tiles from the second
    and later waves of the persistent grid (74 CTA pairs: tiles 74 and 147 are the second tiles of the first and last pair,
    148 opens the third wave), a tile in the middle, and a stride sample filling up to k rays in total."""
    idx = [np.arange(0, min(n, 260)), np.arange(max(0, n - 260), n)]
    for b in range(256, min(n, 256 * 65), 256):
        idx.append(np.array([b - 1, b, b + 1]))
    tiles = (n + 255) // 256
    for t in (74, 147, 148, tiles // 2):
        if 0 < t < tiles:
            idx.append(np.arange(t * 256, min(n, t * 256 + 256)))
    fixed = np.unique(np.concatenate(idx)); fixed = fixed[fixed < n]
    rest = max(0, k - len(fixed))
    if rest == 0 or n <= k:
        return fixed if n > k else np.arange(n)
    return np.unique(np.concatenate([fixed, np.linspace(0, n - 1, rest + 256).astype(np.int64)]))


def _paper_scale_parity(ddf, orc, c1, od, dd, n, what):
    lay, blob, m = c1
    dist = torch.full((n,), float("nan"), device="cuda")
    vis = torch.full((n,), float("nan"), device="cuda")
    ddf.ddf_query(m, od, dd, n, dist, vis)
    torch.cuda.synchronize()
    assert ddf.ddf_get_info(m, 1) == 1                      # one launch: the fused kernel
    assert bool(torch.isfinite(dist).all()) and bool(torch.isfinite(vis).all())
    idx = _sample(n)
    it = torch.from_numpy(idx).cuda()
    o, d = od[it].cpu().numpy(), dd[it].cpu().numpy()
    z, t, xi = orc.forward(lay, blob, o, d, mode=0)
    stats = check_parity(dist[it].cpu().numpy(), vis[it].cpu().numpy(), t, xi, what)
    zg = torch.empty((len(idx), 2), device="cuda")
    ddf.ddf_query_logits(m, od[it].contiguous(), dd[it].contiguous(), len(idx), zg)
    zq, _, _ = orc.forward(lay, blob, o, d, mode=1)
    check_quantised(zg.cpu().numpy(), zq, what + " quantised")
    # a ray's result does not depend on the batch it is in
    d2 = torch.empty(len(idx), device="cuda"); v2 = torch.empty(len(idx), device="cuda")
    ddf.ddf_query(m, od[it].contiguous(), dd[it].contiguous(), len(idx), d2, v2)
    assert torch.equal(d2, dist[it]) and torch.equal(v2, vis[it])
    print("%s: %d rays against the exact oracle: %s" % (what, len(idx), stats))
    return stats


def test_sample_meets_the_survey_size():
    for n in (1 << 20, 1 << 22, 1 << 24):
        idx = _sample(n)
        assert len(idx) >= 8192 and len(np.unique(idx)) == len(idx) and idx.max() < n
        for b in range(256, 256 * 65, 256):
            assert b - 1 in idx and b in idx and b + 1 in idx
        assert 74 * 256 + 100 in idx and 148 * 256 in idx and n - 1 in idx and 0 in idx


def test_config1_camera_full_batch(ddf, orc, c1):
    """configs[1]: 2^20 primary rays of a 1024x1024 pinhole camera, full batch on the GPU."""
    W = H = 1024
    n = W * H
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    od = torch.empty((n, 3), device="cuda"); dd = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, W, H, od, dd)
    ocam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o_ref, d_ref = orc.gen_camera(ocam, W, H)
    assert np.allclose(od.cpu().numpy(), o_ref, atol=1e-6) and np.allclose(dd.cpu().numpy(), d_ref, atol=1e-5)
    _paper_scale_parity(ddf, orc, c1, od, dd, n, "C1 camera")


def test_config1_tail_statistics_on_65536_rays(ddf, orc, c1):
    """"Report max, 99.9th percentile and pass fraction, not just pass/fail" - every 16th ray of
    the configs[1] camera batch (65,536 rays, ~30 s of oracle) answered inside the full 2^20-ray launch; the printed
    statistics are the ones DESIGN.md 5 quotes."""
    lay, blob, m = c1
    W = H = 1024
    n = W * H
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    od = torch.empty((n, 3), device="cuda"); dd = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, W, H, od, dd)
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    ddf.ddf_query(m, od, dd, n, dist, vis)
    torch.cuda.synchronize()
    idx = np.arange(5, n, 16)                                   # 65,536 rays, every tile of the launch touched
    it = torch.from_numpy(idx).cuda()
    z, t, xi = orc.forward(lay, blob, od[it].cpu().numpy(), dd[it].cpu().numpy(), mode=0)
    g_d, g_v = dist[it].cpu().numpy(), vis[it].cpu().numpy()
    ed = np.abs(g_d - t) / (1.0 + np.abs(t)); ev = np.abs(g_v - xi)
    band = np.abs(xi - 0.5) < 1e-2
    agree = ((g_v > 0.5) == (xi > 0.5))[~band].mean()
    print("C1 tail, %d rays: |dd|/(1+|d|) max %.3e p99.9 %.3e rms %.3e | |dv| max %.3e p99.9 %.3e rms %.3e | "
          "hit/miss agreement outside the band %.5f, band fraction %.4f, pass fraction %.5f"
          % (len(idx), ed.max(), np.quantile(ed, 0.999), np.sqrt((ed ** 2).mean()), ev.max(), np.quantile(ev, 0.999),
             np.sqrt((ev ** 2).mean()), agree, band.mean(), ((ed <= 1e-2) & (ev <= 1e-2)).mean()))
    assert ed.max() <= 1e-2 and ev.max() <= 1e-2 and agree >= 0.999 and band.mean() < 0.2


def test_config2_shadow_full_batch(ddf, orc, c1):
    """configs[2]: 2^22 shadow rays from the unit sphere toward the light at (3,3,3)."""
    n = 1 << 22
    p = torch.empty((n, 3), device="cuda"); nrm = torch.empty((n, 3), device="cuda")
    od = torch.empty((n, 3), device="cuda"); dd = torch.empty((n, 3), device="cuda"); tmax = torch.empty(n, device="cuda")
    ddf.ddf_gen_sphere_points(MASTER_SEED, STREAMS["shadow_points"], n, 1.0, p, nrm)
    ddf.ddf_gen_shadow(p, nrm, n, (3.0, 3.0, 3.0), 1e-3, od, dd, tmax)
    k = 1 << 16
    p_ref, n_ref = orc.gen_sphere_points(MASTER_SEED, STREAMS["shadow_points"], k, 1.0)
    o_ref, d_ref, t_ref = orc.gen_shadow(p_ref, n_ref, (3.0, 3.0, 3.0), 1e-3)
    assert np.allclose(p[:k].cpu().numpy(), p_ref, atol=1e-5)
    assert np.allclose(od[:k].cpu().numpy(), o_ref, atol=1e-5) and np.allclose(dd[:k].cpu().numpy(), d_ref, atol=1e-5)
    assert np.allclose(tmax[:k].cpu().numpy(), t_ref, rtol=1e-5)
    # property at full size (pin P10): occluded fraction of the analytic unit sphere = 0.574203
    b = (od.double() * dd.double()).sum(1)
    occl = (b < 0) & (b * b - ((od.double() ** 2).sum(1) - 1.0) >= 0)
    assert abs(float(occl.double().mean()) - 0.574203) < 4 * math.sqrt(0.25 / n)
    _paper_scale_parity(ddf, orc, c1, od, dd, n, "C2 shadow")
    # the shadow decision on the GPU results
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda"); sh = torch.empty(n, dtype=torch.uint8, device="cuda")
    lay, blob, m = c1
    ddf.ddf_query(m, od, dd, n, dist, vis)
    ddf.ddf_shadow_test(vis, dist, tmax, n, sh)
    assert torch.equal(sh.bool(), (vis > 0.5) & (dist < tmax))


def test_config3_ao_full_batch(ddf, orc, c1):
    """configs[3]: 1024x1024 G-buffer x 16 cosine samples = 16.7M rays, AO reduced on the GPU."""
    lay, blob, m = c1
    W = H = 1024
    npts, spp = W * H, 16
    n = npts * spp
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    sc = ddf.DdfScene((0.0, 0.0, 0.0), 0.6, (-3.0, -3.0, -3.0), (3.0, 3.0, 3.0))
    p = torch.empty((npts, 3), device="cuda"); nrm = torch.empty((npts, 3), device="cuda"); th = torch.empty(npts, device="cuda")
    ddf.ddf_gen_gbuffer(cam, sc, W, H, p, nrm, th)
    od = torch.empty((n, 3), device="cuda"); dd = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_ao(p, nrm, npts, spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3, od, dd)
    # generator twins on a band of rows through the middle of the image (sphere + walls)
    ocam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    p_ref, n_ref, t_ref = orc.gen_gbuffer(ocam, orc.make_scene(), W, H)
    pg, ng = p.cpu().numpy(), nrm.cpu().numpy()
    on_s_g = np.abs(np.linalg.norm(pg, axis=1) - 0.6) < 1e-4
    on_s_r = np.abs(np.linalg.norm(p_ref, axis=1) - 0.6) < 1e-4
    same_surface = (on_s_g & on_s_r) | (~on_s_g & ~on_s_r & np.all(ng == n_ref, axis=1))
    assert same_surface.mean() > 0.9999                       # silhouette pixels may flip sphere/wall
    perr = np.abs(pg - p_ref).max(axis=1)[same_surface]
    assert (perr < 2e-5).mean() > 0.9995 and perr.max() < 5e-3   # grazing sphere hits amplify fp32 rounding
    assert np.allclose(ng[same_surface], n_ref[same_surface], atol=1e-2)
    assert (np.abs(ng - n_ref).max(axis=1)[same_surface] < 5e-5).mean() > 0.9995
    assert np.allclose(th.cpu().numpy()[same_surface], t_ref[same_surface], atol=5e-3)
    # the twin draws sample k = pixel*spp + s: a prefix of the image shares the GPU's indices
    o_ref, d_ref = orc.gen_ao(pg[:8192], ng[:8192], spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3)
    assert np.allclose(od[:8192 * spp].cpu().numpy(), o_ref, atol=1e-5)
    assert np.allclose(dd[:8192 * spp].cpu().numpy(), d_ref, atol=2e-5)
    rows = slice(500 * W, 504 * W)
    o_ref, d_ref = orc.gen_ao(pg[rows], ng[rows], spp, MASTER_SEED, STREAMS["ao_samples"], 1e-3)
    o_all, d_all = od.view(npts, spp, 3)[500 * W:504 * W].reshape(-1, 3).cpu().numpy(), dd.view(npts, spp, 3)[500 * W:504 * W].reshape(-1, 3).cpu().numpy()
    assert np.allclose(o_all, o_ref, atol=1e-5)               # origins do not depend on the sample index
    nn = np.repeat(ng[rows], spp, axis=0)
    assert np.allclose(np.linalg.norm(d_all, axis=1), 1.0, atol=1e-5) and ((d_all * nn).sum(1) >= -1e-5).all()
    c = (dd * nrm.repeat_interleave(spp, dim=0)).sum(1).double()
    assert abs(float(c.mean()) - 2 / 3) < 1e-3 and abs(float((c * c).mean()) - 0.5) < 1e-3     # pin P11 at full size
    # per-ray parity on samples + fused AO against the reducer on the GPU's own per-ray outputs
    _paper_scale_parity(ddf, orc, c1, od, dd, n, "C3 AO")
    ao = torch.full((npts,), float("nan"), device="cuda")
    ddf.ddf_query_ao(m, od, dd, npts, spp, float("inf"), ao)
    torch.cuda.synchronize()
    assert ddf.ddf_get_info(m, 1) == 1                         # fused: query + reduce in one launch
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda"); ao2 = torch.empty(npts, device="cuda")
    ddf.ddf_query(m, od, dd, n, dist, vis)
    ddf.ddf_ao_reduce(vis, dist, npts, spp, float("inf"), ao2)
    assert torch.equal(ao, ao2)
    k = 4096
    assert np.array_equal(orc.ao_reduce(vis[:k * spp].cpu().numpy(), dist[:k * spp].cpu().numpy(), spp), ao2[:k].cpu().numpy())
    # AO image against the oracle evaluated end to end on whole pixels
    pix = np.arange(0, npts, npts // 256)[:256]                # AO parity on >= 256 whole pixels
    ridx = (pix[:, None] * spp + np.arange(spp)[None, :]).reshape(-1)
    it = torch.from_numpy(ridx).cuda()
    z, t, xi = orc.forward(lay, blob, od[it].cpu().numpy(), dd[it].cpu().numpy(), mode=0)
    ao_ref = orc.ao_reduce(xi.astype(np.float32), t.astype(np.float32), spp)
    near = (np.abs(xi - 0.5) < 1e-2).reshape(-1, spp).sum(1)   # rays that may legitimately flip
    assert np.all(np.abs(ao[torch.from_numpy(pix).cuda()].cpu().numpy() - ao_ref) <= near / spp + 1e-6)
