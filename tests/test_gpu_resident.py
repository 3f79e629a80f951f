"""GPU tests of the activation-resident kernel (ddf_set_path 5; csrc/ddf_tc_res.cuh): the same forward pass as the
persistent kernel with the layer hand-off in shared / tensor memory.  Parity against the oracle with the north_star
tolerances (exact mode) and the tighter quantised comparison, the closed forms P1 / P4 / P5 through this kernel, and the
contract: results independent of n and of the ray's position, every output mode, device-side count."""
import math

import numpy as np
import pytest
import torch

from ddf_inputs import (MASTER_SEED, STREAMS, Layout, layout_c1, layout_sdf, make_weights, random_rays,
                        blob_layer_shapes, blob_num_elements)
from test_gpu_parity import check_parity, check_quantised, _sample

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ddf():
    import paper_2606_00817_b200 as pkg
    pkg.build()
    assert torch.cuda.is_available()
    return pkg


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _logits(ddf, m, o, d, n):
    z = torch.full((n, m.layout.n_out), float("nan"), device="cuda")
    ddf.ddf_query_logits(m, o, d, n, z)
    torch.cuda.synchronize()
    return z


# 256x1: one hidden layer is outside what the resident kernel serves (its head-partial buffer relies on the layer-0
# hand-over of a second layer); path 5 must answer it with the persistent kernel, still in one launch
# name, layout, (max, mean) bound of the quantised gate: ~2x the measured values (max over the ten batch sizes, 300 rays each)
LAYOUTS = [("256x1 falls back", Layout(0, 10, 4, 1, 256, -1, 2, 0), (1e-5, 1e-6)),                     # measured 8.1e-7 / 1.5e-7
           ("256x2", Layout(0, 10, 4, 2, 256, -1, 2, 0), (1e-5, 1e-6)),                                # 4.2e-6 / 1.5e-7
           ("256x3 skip 1", Layout(0, 10, 4, 3, 256, 1, 2, 0), (5e-4, 5e-6)),                          # 2.2e-4 / 9.7e-7
           ("512x3 skip 2, no direction bands", Layout(0, 6, 0, 3, 512, 2, 2, 0), (2e-3, 2e-5)),       # 9.1e-4 / 4.2e-6
           ("768x2 one output", Layout(0, 4, 4, 2, 768, -1, 1, 0), (1e-5, 1e-6)),                      # 1.6e-6 / 2.9e-7
           ("1024x4 skip 3", Layout(0, 10, 4, 4, 1024, 3, 2, 0), (1e-2, 1e-4)),                        # 4.2e-3 / 4.2e-5
           ("configs[1]", layout_c1(), (2.5e-2, 2.5e-3)),                                              # 9.6e-3 / 8.9e-4
           ("SDF network", layout_sdf(), (2.5e-2, 2.5e-3))]                                            # 9.1e-3 / 1.1e-3


@pytest.mark.parametrize("name,lay,qtol", LAYOUTS, ids=[l[0] for l in LAYOUTS])
def test_resident_kernel_matches_the_oracle_and_the_persistent_kernel(ddf, orc, name, lay, qtol):
    blob = make_weights(lay, bias_scale=0.2)
    m = ddf.ddf_create(blob, lay)
    for n in (1, 63, 64, 65, 127, 128, 129, 1000, 128 * 74 + 1, 20011):
        o_np, d_np = random_rays(n)
        o = _cuda(o_np); d = _cuda(d_np) if lay.input_kind == 0 else None
        ddf.ddf_set_path(m, 3); z3 = _logits(ddf, m, o, d, n)
        ddf.ddf_set_path(m, 5); z5 = _logits(ddf, m, o, d, n)
        assert ddf.ddf_get_info(m, 1) == 1                                  # one launch
        assert bool(torch.isfinite(z5).all())
        idx = np.unique(np.linspace(0, n - 1, min(n, 300)).astype(np.int64))
        zq = orc.forward(lay, blob, o_np[idx], d_np[idx] if lay.input_kind == 0 else None, mode=1)[0]
        check_quantised(z5.cpu().numpy()[idx], zq, "%s n=%d" % (name, n), max_tol=qtol[0], mean_tol=qtol[1])
        # the two kernels add the same products in a different order: equal up to bf16 rounding flips along the layers
        assert float((z3 - z5).abs().max()) <= 4e-2 and float((z3 - z5).abs().mean()) <= 3e-3
        if lay.n_hidden < 2:
            assert torch.equal(z3, z5)                                      # the same kernel answered both
    ddf.ddf_destroy(m)


def test_resident_kernel_full_camera_batch_parity_and_contract(ddf, orc):
    """configs[1], 2^20 camera rays in one launch of the resident kernel: north_star tolerances on >= 8192 sampled rays,
    results independent of the batch (bit for bit), AO reduce fused in the kernel = reducer on its per-ray outputs,
    device-side ray count, no write past n."""
    lay = layout_c1(); blob = make_weights(lay)
    m = ddf.ddf_create(blob, lay)
    ddf.ddf_set_path(m, 5)
    W = H = 1024; n = W * H
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    od = torch.empty((n, 3), device="cuda"); dd = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_camera(cam, W, H, od, dd)
    dist = torch.full((n,), float("nan"), device="cuda"); vis = torch.full((n,), float("nan"), device="cuda")
    ddf.ddf_query(m, od, dd, n, dist, vis)
    torch.cuda.synchronize()
    assert ddf.ddf_get_info(m, 1) == 1
    assert bool(torch.isfinite(dist).all()) and bool(torch.isfinite(vis).all())
    idx = _sample(n); it = torch.from_numpy(idx).cuda()
    o, d = od[it].cpu().numpy(), dd[it].cpu().numpy()
    z, t, xi = orc.forward(lay, blob, o, d, mode=0)
    stats = check_parity(dist[it].cpu().numpy(), vis[it].cpu().numpy(), t, xi, "resident C1 camera")
    print("resident kernel, C1 camera: %d rays against the exact oracle: %s" % (len(idx), stats))
    # the hand-over protocol (asynchronous peer stores, relay, parked chunks) has no run-to-run freedom: twelve more
    # launches of the full batch return the same bits
    for _ in range(12):
        da = torch.empty(n, device="cuda"); va = torch.empty(n, device="cuda")
        ddf.ddf_query(m, od, dd, n, da, va)
        assert torch.equal(da, dist) and torch.equal(va, vis)
    # a ray's result does not depend on the batch it is in, nor on its position
    d2 = torch.empty(len(idx), device="cuda"); v2 = torch.empty(len(idx), device="cuda")
    ddf.ddf_query(m, od[it].contiguous(), dd[it].contiguous(), len(idx), d2, v2)
    assert torch.equal(d2, dist[it]) and torch.equal(v2, vis[it])
    N = 128 * 148 + 77
    o_np, d_np = random_rays(N); oN, dN = _cuda(o_np), _cuda(d_np)
    fd = torch.empty(N, device="cuda"); fv = torch.empty(N, device="cuda")
    ddf.ddf_query(m, oN, dN, N, fd, fv)
    perm = torch.randperm(N, device="cuda", generator=torch.Generator(device="cuda").manual_seed(3))
    pd = torch.empty(N, device="cuda"); pv = torch.empty(N, device="cuda")
    ddf.ddf_query(m, oN[perm].contiguous(), dN[perm].contiguous(), N, pd, pv)
    assert torch.equal(pd, fd[perm]) and torch.equal(pv, fv[perm])
    for k in (0, 1, 127, 129, 1009):
        a = torch.full((max(k, 1) + 8,), -7.0, device="cuda"); b = torch.full((max(k, 1) + 8,), -7.0, device="cuda")
        ddf.ddf_query(m, oN, dN, k, a, b)
        torch.cuda.synchronize()
        assert torch.equal(a[:k], fd[:k]) and torch.equal(b[:k], fv[:k]) and bool((a[k:] == -7.0).all()) and bool((b[k:] == -7.0).all())
    # fused AO reduce (16 rays per pixel) = the reducer on the per-ray outputs; visibility bias 1 so hits and misses mix
    blob2 = blob.copy(); blob2[-1] = 0x3F80
    m2 = ddf.ddf_create(blob2, lay); ddf.ddf_set_path(m2, 5)
    npts, spp = 4001, 16                                                   # 64,016 rays: a ragged last tile
    o2, d2n = random_rays(npts * spp); o2, d2n = _cuda(o2), _cuda(d2n)
    rd = torch.empty(npts * spp, device="cuda"); rv = torch.empty(npts * spp, device="cuda")
    ddf.ddf_query(m2, o2, d2n, npts * spp, rd, rv)
    ao = torch.full((npts,), float("nan"), device="cuda"); ao2 = torch.empty(npts, device="cuda")
    ddf.ddf_query_ao(m2, o2, d2n, npts, spp, float("inf"), ao)
    assert ddf.ddf_get_info(m2, 1) == 1
    ddf.ddf_ao_reduce(rv, rd, npts, spp, float("inf"), ao2)
    hf = float((rv > 0.5).float().mean())
    assert torch.equal(ao, ao2) and 0.05 < hf < 0.95, hf
    ddf.ddf_destroy(m2)
    ddf.ddf_destroy(m)


def test_resident_kernel_closed_forms(ddf, orc):
    """P1 (zero weights: heads of the bias), P4 shape (all-ones first layer exposes the K padding 90 -> 96) and P5 (selector
    layers pass gamma through, also through the skip only) on the resident kernel."""
    o, d = random_rays(700)
    od, dd = _cuda(o), _cuda(d)
    lay = Layout(0, 4, 4, 3, 256, 1, 2, 0)
    blob = np.zeros(blob_num_elements(lay), np.float32); blob[-2:] = [1.25, -0.5]
    m = ddf.ddf_create(blob, lay); ddf.ddf_set_path(m, 5)
    dist = torch.empty(700, device="cuda"); vis = torch.empty(700, device="cuda")
    ddf.ddf_query(m, od, dd, 700, dist, vis); torch.cuda.synchronize()
    assert np.allclose(dist.cpu().numpy(), 1.25 + math.log1p(math.exp(-1.25)), rtol=2e-7)
    assert np.allclose(vis.cpu().numpy(), 1.0 / (1.0 + math.exp(0.5)), rtol=2e-7)
    ddf.ddf_destroy(m)

    def blob_of(lay, layers):
        parts = []
        for (Wm, b), (oo, ii) in zip(layers, blob_layer_shapes(lay)):
            Wm = np.asarray(Wm, np.float64); assert Wm.shape == (oo, ii)
            parts += [Wm.reshape(-1), np.asarray(b, np.float64).reshape(oo)]
        return np.concatenate(parts).astype(np.float32)

    width = 256
    lay = Layout(0, 10, 4, 1, width, -1, 2, 0)
    head = np.zeros((2, width)); head[0, :] = 1.0 / width; head[1, 0] = -0.25
    m = ddf.ddf_create(blob_of(lay, [(np.ones((width, 90)), np.zeros(width)), (head, [0, 1])]), lay); ddf.ddf_set_path(m, 5)
    z = _logits(ddf, m, od, dd, 700).cpu().numpy()
    gq = np.vectorize(orc.round_bf16)(orc.encode(lay, o, d))
    s = np.maximum(gq.sum(1), 0.0)
    assert np.allclose(z[:, 0], s, atol=2e-5, rtol=1e-5) and np.allclose(z[:, 1], 1.0 - 0.25 * s, atol=2e-5, rtol=1e-5)
    ddf.ddf_destroy(m)

    for through_skip in (False, True):
        lay = Layout(0, 10, 4, 3, 256, 1, 2, 0)
        E, Wd = 90, 256
        rng = np.random.default_rng(5)
        c = [np.vectorize(orc.round_bf16)(rng.standard_normal(E)) for _ in range(2)]
        sel = np.zeros((Wd, E)); sel[:E] = np.eye(E); sel[E:2 * E] = -np.eye(E)
        ident = np.zeros((Wd, Wd)); ident[:2 * E, :2 * E] = np.eye(2 * E)
        layers = []
        for l in range(3):
            nin = E if l == 0 else (Wd + E if l == 1 else Wd)
            Wl = np.zeros((Wd, nin))
            if through_skip:
                if l == 1: Wl[:, Wd:] = sel
                elif l == 2: Wl[:, :Wd] = ident
            else:
                if l == 0: Wl[:, :E] = sel
                else: Wl[:, :Wd] = ident
            layers.append((Wl, np.zeros(Wd)))
        head = np.zeros((2, Wd))
        for j in range(2):
            head[j, :E] = c[j]; head[j, E:2 * E] = -c[j]
        layers.append((head, np.zeros(2)))
        m = ddf.ddf_create(blob_of(lay, layers), lay); ddf.ddf_set_path(m, 5)
        z = _logits(ddf, m, od, dd, 700).cpu().numpy()
        gq = np.vectorize(orc.round_bf16)(orc.encode(lay, o, d))
        assert np.allclose(z[:, 0], gq @ c[0], atol=3e-5) and np.allclose(z[:, 1], gq @ c[1], atol=3e-5), through_skip
        ddf.ddf_destroy(m)


def test_sphere_tracer_on_the_resident_kernel(ddf, orc):
    """The tracer's per-step evaluation with the live-ray count read on the device (n_dev): with the MLP term off the
    result is the step rule alone - bit-identical to the CPU tracer whichever kernel evaluates the (unused) network."""
    lay = layout_sdf(); blob = make_weights(lay)
    m = ddf.ddf_create(blob, lay); ddf.ddf_set_path(m, 5)
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 200, 150)                                  # 30,000 rays: the persistent-size path (resident kernel)
    n = len(o)
    t = torch.empty(n, device="cuda"); hit = torch.empty(n, dtype=torch.uint8, device="cuda")
    st = torch.empty(n, dtype=torch.int32, device="cuda"); tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    ddf.sdf_sphere_trace(m, _cuda(o), _cuda(d), n, ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.0, 1), t, hit, st, None, None, tot)
    torch.cuda.synchronize()
    rt, rhit, rsteps = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0)
    assert np.array_equal(t.cpu().numpy(), rt) and np.array_equal(hit.cpu().numpy(), rhit) and np.array_equal(st.cpu().numpy(), rsteps)
    # with the MLP on: same statistics as the persistent kernel's trace of the same rays
    prm = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 1)
    ddf.sdf_sphere_trace(m, _cuda(o), _cuda(d), n, prm, t, hit, st, None, None, tot); torch.cuda.synchronize()
    h5, s5 = float(hit.float().mean()), float(st.float().mean())
    ddf.ddf_set_path(m, 3)
    ddf.sdf_sphere_trace(m, _cuda(o), _cuda(d), n, prm, t, hit, st, None, None, tot); torch.cuda.synchronize()
    h3, s3 = float(hit.float().mean()), float(st.float().mean())
    assert abs(h5 - h3) < 3.0 * math.sqrt(2 * h3 * (1 - h3) / n) and abs(s5 - s3) < 1.0
    ddf.ddf_destroy(m)
