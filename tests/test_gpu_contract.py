"""GPU tests: closed forms through the kernels (pins P1, P4, P5), the API contract (T4), the two
kernel paths against each other, the host-buffer entry point, and the sphere tracer (P12)."""
import math

import numpy as np
import pytest
import torch

from ddf_inputs import (MASTER_SEED, STREAMS, Layout, layout_c0, layout_c1, layout_sdf, make_weights,
                        random_rays, blob_layer_shapes, blob_num_elements, f32_to_bf16_bits)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ddf():
    import paper_2606_00817_b200 as pkg
    pkg.build()
    return pkg


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _logits(ddf, m, o, d):
    n = o.shape[0]
    z = torch.full((n, m.layout.n_out), float("nan"), device="cuda")
    ddf.ddf_query_logits(m, _cuda(o), _cuda(d) if d is not None else None, n, z)
    torch.cuda.synchronize()
    return z.cpu().numpy()


def _heads(ddf, m, o, d):
    n = o.shape[0]
    dist = torch.full((n,), float("nan"), device="cuda"); vis = torch.full((n,), float("nan"), device="cuda")
    ddf.ddf_query(m, _cuda(o), _cuda(d), n, dist, vis)
    torch.cuda.synchronize()
    return dist.cpu().numpy(), vis.cpu().numpy()


def _blob(lay, layers):
    parts = []
    for (W, b), (o, i) in zip(layers, blob_layer_shapes(lay)):
        W = np.asarray(W, np.float64); assert W.shape == (o, i)
        parts += [W.reshape(-1), np.asarray(b, np.float64).reshape(o)]
    return np.concatenate(parts).astype(np.float32)


# ------------------------------------------------------------------ closed forms on the GPU

@pytest.mark.parametrize("path", [0, 1])                # the fused kernel that serves the layout / the CUDA-core path
@pytest.mark.parametrize("width", [32, 64, 128, 256])   # padded to 64 / narrow tcgen05 x2 / wide tcgen05 kernel
def test_zero_weights_give_head_of_bias(ddf, width, path):
    lay = Layout(0, 4, 4, 3, width, 1, 2, 0)
    blob = np.zeros(blob_num_elements(lay), np.float32)
    blob[-2:] = [1.25, -0.5]
    m = ddf.ddf_create(blob, lay)
    ddf.ddf_set_path(m, path)
    o, d = random_rays(300)
    dist, vis = _heads(ddf, m, o, d)
    assert np.allclose(dist, 1.25 + math.log1p(math.exp(-1.25)), rtol=2e-7)
    assert np.allclose(vis, 1.0 / (1.0 + math.exp(0.5)), rtol=2e-7)
    blob[-2:] = 0
    m2 = ddf.ddf_create(blob, lay)
    dist, vis = _heads(ddf, m2, o, d)
    assert np.allclose(dist, math.log(2.0), rtol=2e-7) and np.all(vis == 0.5)


@pytest.mark.parametrize("path", [0, 1])
@pytest.mark.parametrize("width", [32, 64, 128, 256])
def test_all_ones_layer_exposes_pad_lanes(ddf, orc, width, path):
    """P4 shape: W0 = all ones => every hidden unit = ReLU(sum gamma); K = 90 is padded to 128 on
    the GPU, so any pad lane that is not zero changes the sum."""
    lay = Layout(0, 10, 4, 1, width, -1, 2, 0)
    head = np.zeros((2, width)); head[0, :] = 1.0 / width; head[1, 0] = -0.25
    blob = _blob(lay, [(np.ones((width, 90)), np.zeros(width)), (head, [0, 1])])
    m = ddf.ddf_create(blob, lay)
    ddf.ddf_set_path(m, path)
    o, d = random_rays(513)
    z = _logits(ddf, m, o, d)
    g = orc.encode(lay, o, d)
    gq = np.vectorize(orc.round_bf16)(g)
    s = np.maximum(gq.sum(1), 0.0)
    assert np.allclose(z[:, 0], s, atol=2e-5, rtol=1e-5)
    assert np.allclose(z[:, 1], 1.0 - 0.25 * s, atol=2e-5, rtol=1e-5)


@pytest.mark.parametrize("through_skip", [False, True])
def test_selector_layers_pass_encoding_through(ddf, orc, through_skip):
    """P5 on the tcgen05 path: width 256 >= 2E (E = 90); z = c . gamma (bf16-rounded gamma)."""
    lay = Layout(0, 10, 4, 3, 256, 1, 2, 0)
    E, W = 90, 256
    rng = np.random.default_rng(5)
    c = [np.vectorize(orc.round_bf16)(rng.standard_normal(E)) for _ in range(2)]
    sel = np.zeros((W, E)); sel[:E] = np.eye(E); sel[E:2 * E] = -np.eye(E)
    ident = np.zeros((W, W)); ident[:2 * E, :2 * E] = np.eye(2 * E)
    layers = []
    for l in range(3):
        nin = E if l == 0 else (W + E if l == 1 else W)
        Wl = np.zeros((W, nin))
        if through_skip:
            if l == 1: Wl[:, W:] = sel
            elif l == 2: Wl[:, :W] = ident
        else:
            if l == 0: Wl[:, :E] = sel
            else: Wl[:, :W] = ident
        layers.append((Wl, np.zeros(W)))
    head = np.zeros((2, W))
    for j in range(2):
        head[j, :E] = c[j]; head[j, E:2 * E] = -c[j]
    layers.append((head, np.zeros(2)))
    m = ddf.ddf_create(_blob(lay, layers), lay)
    assert ddf.ddf_get_info(m, 0) == 1
    o, d = random_rays(700)
    z = _logits(ddf, m, o, d)
    gq = np.vectorize(orc.round_bf16)(orc.encode(lay, o, d))
    assert np.allclose(z[:, 0], gq @ c[0], atol=3e-5) and np.allclose(z[:, 1], gq @ c[1], atol=3e-5)


def test_encoding_on_gpu_matches_definition(ddf, orc):
    """gamma read back through an identity-selector network, including origins at radius 2.5 where
    the top band's phase is ~4000 rad (exact power-of-two scaling)."""
    lay = Layout(0, 10, 4, 1, 256, -1, 2, 0)
    E, W = 90, 256
    o, d = random_rays(256)
    o = (o * 2.5).astype(np.float32)
    g = orc.encode(lay, o, d)
    for k in range(0, E, 2):
        W0 = np.zeros((W, E)); W0[0, k] = 1; W0[1, k] = -1; W0[2, k + 1] = 1; W0[3, k + 1] = -1
        head = np.zeros((2, W)); head[0, 0] = 1; head[0, 1] = -1; head[1, 2] = 1; head[1, 3] = -1
        m = ddf.ddf_create(_blob(lay, [(W0, np.zeros(W)), (head, [0, 0])]), lay)
        z = _logits(ddf, m, o, d)
        ddf.ddf_destroy(m)
        assert np.allclose(z, np.vectorize(orc.round_bf16)(g[:, k:k + 2]), atol=1e-6), k


# ------------------------------------------------------------------ API contract

@pytest.fixture(scope="module")
def c1(ddf):
    lay = layout_c1()
    m = ddf.ddf_create(make_weights(lay), lay)
    yield lay, m
    ddf.ddf_destroy(m)


def test_edge_sizes_permutation_determinism(ddf, c1):
    lay, m = c1
    N = 256 * 148 + 257
    o, d = random_rays(N)
    od, dd = _cuda(o), _cuda(d)
    full_d = torch.empty(N, device="cuda"); full_v = torch.empty(N, device="cuda")
    ddf.ddf_query(m, od, dd, N, full_d, full_v)
    again_d = torch.empty(N, device="cuda"); again_v = torch.empty(N, device="cuda")
    ddf.ddf_query(m, od, dd, N, again_d, again_v)
    assert torch.equal(full_d, again_d) and torch.equal(full_v, again_v)          # bit-reproducible
    for n in (0, 1, 127, 128, 129, 255, 256, 257, 1009):
        dist = torch.full((max(n, 1) + 8,), -7.0, device="cuda"); vis = torch.full((max(n, 1) + 8,), -7.0, device="cuda")
        ddf.ddf_query(m, od, dd, n, dist, vis)
        torch.cuda.synchronize()
        assert torch.equal(dist[:n], full_d[:n]) and torch.equal(vis[:n], full_v[:n]), n
        assert bool((dist[n:] == -7.0).all()) and bool((vis[n:] == -7.0).all()), n    # no write past n
    perm = torch.randperm(N, device="cuda", generator=torch.Generator(device="cuda").manual_seed(1))
    pd = torch.empty(N, device="cuda"); pv = torch.empty(N, device="cuda")
    ddf.ddf_query(m, od[perm].contiguous(), dd[perm].contiguous(), N, pd, pv)
    assert torch.equal(pd, full_d[perm]) and torch.equal(pv, full_v[perm])
    # out_vis may be NULL
    only_d = torch.empty(N, device="cuda")
    ddf.ddf_query(m, od, dd, N, only_d, None)
    assert torch.equal(only_d, full_d)
    # unaligned (4-byte aligned only) buffers
    ou = torch.empty(3 * 1001 + 1, device="cuda")[1:].view(1001, 3); ou.copy_(od[:1001])
    du = torch.empty(3 * 1001 + 1, device="cuda")[1:].view(1001, 3); du.copy_(dd[:1001])
    outu = torch.empty(1002, device="cuda")[1:]
    from paper_2606_00817_b200.binding import lib, _stream
    import ctypes as C
    rc = lib().ddf_query(m.handle, C.c_void_p(ou.data_ptr()), C.c_void_p(du.data_ptr()), C.c_int64(1001),
                         C.c_void_p(outu.data_ptr()), None, _stream(None))
    assert rc == 0
    assert torch.equal(outu, full_d[:1001])


def test_column_split_path_is_bit_identical_to_the_persistent_kernel(ddf, c1, sdf):
    """Batches of at most 40 tiles are answered one launch per layer with a layer's output columns
    split over the CTA pairs (ddf_set_path 4 forces it up to 74 tiles, 3 forbids it): heads, logits,
    the AO reduction and the sphere tracer's device-side ray count must give the persistent kernel's bits."""
    lay, m = c1
    N = 256 * 74 + 300
    o, d = random_rays(N, seed=21)
    od, dd = _cuda(o), _cuda(d)

    def run(path, n, mode):
        ddf.ddf_set_path(m, path)
        if mode == "heads":
            out = torch.full((2, n + 8), -7.0, device="cuda")
            ddf.ddf_query(m, od, dd, n, out[0], out[1])
        elif mode == "logits":
            out = torch.full((n + 8, 2), -7.0, device="cuda")
            ddf.ddf_query_logits(m, od, dd, n, out)
        else:
            out = torch.full((n // 16 + 8,), -7.0, device="cuda")
            ddf.ddf_query_ao(m, od, dd, n // 16, 16, 0.7, out)
        torch.cuda.synchronize()
        return out, ddf.ddf_get_info(m, 1)

    try:
        for n in (1, 255, 256, 257, 1000, 4099, 40 * 256, 40 * 256 + 16, 74 * 256):
            for mode in ("heads", "logits", "ao"):
                if mode == "ao" and n < 16:
                    continue
                a, la = run(3, n, mode)
                b, lb = run(4, n, mode)
                c, lc = run(0, n, mode)
                assert la == 1 and lb == lay.n_hidden + 2, (n, mode, la, lb)
                assert lc == (lb if n <= 40 * 256 else la), (n, mode, lc)        # the automatic choice
                assert torch.equal(a, b) and torch.equal(a, c), (n, mode)
                assert bool(torch.isfinite(a).all())                             # includes the -7 guard past n
                if mode == "heads":
                    assert bool((a[:, n:] == -7.0).all()) and bool((a[:, :n] != -7.0).all())
        # more tiles than the scratch has rows for: path 4 falls back to the persistent kernel
        a, la = run(4, N, "heads")
        assert la == 1
    finally:
        ddf.ddf_set_path(m, 0)
    # sphere tracer (device-side live-ray count, early exit) on a batch small enough to be split
    slay, sblob, sm = sdf
    oo, ddd = random_rays(3000, seed=22)
    oo = (oo * 2.5 / np.linalg.norm(oo, axis=1, keepdims=True)).astype(np.float32)
    ddd = (-oo / np.linalg.norm(oo, axis=1, keepdims=True)).astype(np.float32)
    res = []
    try:
        for path in (3, 4):
            ddf.ddf_set_path(sm, path)
            res.append(_trace(ddf, sm, oo, ddd, ddf.SdfTraceParams(32, 1e-3, 6.0, 1.0, 0.05, 1)))
    finally:
        ddf.ddf_set_path(sm, 0)
    for x, y in zip(res[0], res[1]):
        assert np.array_equal(x, y)
    assert res[0][3] > 3000                                                      # more than one step was taken


def test_bad_arguments(ddf, c1):
    lay, m = c1
    from paper_2606_00817_b200.binding import lib, _stream
    import ctypes as C
    x = torch.zeros((4, 3), device="cuda"); y = torch.zeros(4, device="cuda")
    p = lambda t: C.c_void_p(t.data_ptr())
    assert lib().ddf_query(m.handle, p(x), p(x), C.c_int64(-1), p(y), p(y), _stream(None)) == -1
    assert lib().ddf_query(m.handle, None, p(x), C.c_int64(4), p(y), p(y), _stream(None)) == -1
    assert lib().ddf_query(m.handle, p(x), None, C.c_int64(4), p(y), p(y), _stream(None)) == -1
    assert lib().ddf_query(m.handle, p(x), p(x), C.c_int64(4), None, p(y), _stream(None)) == -1
    assert lib().ddf_query(m.handle, None, None, C.c_int64(0), None, None, _stream(None)) == 0
    bad = Layout(0, 10, 4, 8, 1280, 4, 2, 1)
    with pytest.raises(ddf.DdfError):
        wbig = Layout(0, 4, 4, 1, 2100, -1, 2, 0)
        ddf.ddf_set_path(ddf.ddf_create(make_weights(wbig), wbig), 2)   # width 2100: beyond the padded tilings, CUDA-core path only
    prm = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 0)
    t = torch.zeros(4, device="cuda"); h = torch.zeros(4, dtype=torch.uint8, device="cuda"); s = torch.zeros(4, dtype=torch.int32, device="cuda")
    with pytest.raises(ddf.DdfError):
        ddf.sdf_sphere_trace(m, x, x, 4, prm, t, h, s)         # a DDF model is not an SDF model
    slay = layout_sdf()
    sm = ddf.ddf_create(make_weights(slay), slay)
    for omega in (2.0, 2.5, -0.5, float("nan")):               # the relaxation factor must lie in [0, 2)
        with pytest.raises(ddf.DdfError, match="invalid argument"):
            ddf.sdf_sphere_trace(sm, x, x, 4, ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 0, omega), t, h, s)
    ddf.sdf_sphere_trace(sm, x, x, 4, ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 0, 1.999), t, h, s)
    torch.cuda.synchronize()
    ddf.ddf_destroy(sm)


@pytest.mark.parametrize("lay", [Layout(0, 6, 3, 4, 512, 2, 2, 1), Layout(0, 6, 3, 4, 128, 2, 2, 0), Layout(0, 4, 4, 3, 64, -1, 2, 1),
                                 Layout(1, 10, 0, 5, 128, 3, 1, 1),
                                 # widths the kernels do not tile are zero-padded at create (96 -> 128, 200 -> 256, 384 -> 512, 24 -> 64)
                                 Layout(0, 6, 3, 3, 96, 1, 2, 0), Layout(0, 4, 4, 2, 200, -1, 2, 0), Layout(0, 10, 4, 4, 384, 2, 2, 1),
                                 Layout(0, 2, 2, 2, 24, 1, 2, 0),
                                 # narrow but too deep for shared memory (12 x 128, skip): padded to 256, wide kernel
                                 Layout(0, 10, 4, 12, 128, 5, 2, 1)])
def test_simt_and_tcgen05_paths_agree(ddf, orc, lay):
    """wide tcgen05 kernel, narrow tcgen05 kernel (width 128 with skip / width 64 / point input with
    one linear output) against the plain CUDA-core path and both oracle modes"""
    blob = make_weights(lay, seed=17, bias_scale=0.2)
    m = ddf.ddf_create(blob, lay)
    assert ddf.ddf_get_info(m, 0) == 1
    o, d = random_rays(2000, seed=5)
    if lay.input_kind == 1:
        d = None
    ddf.ddf_set_path(m, 2); z_tc = _logits(ddf, m, o, d)
    # one fused launch, or (wide kernel, a batch this small) encode + one launch per layer + heads
    assert ddf.ddf_get_info(m, 1) == (lay.n_hidden + 2 if ddf.ddf_get_info(m, 3) == 256 else 1)
    ddf.ddf_set_path(m, 1); z_si = _logits(ddf, m, o, d); assert ddf.ddf_get_info(m, 1) > 1
    zq, _, _ = orc.forward(lay, blob, o, d, mode=1)
    ze, _, _ = orc.forward(lay, blob, o, d, mode=0)
    assert np.abs(z_tc - z_si).max() < 4e-2 and np.abs(z_tc - z_si).mean() < 3e-3
    for z in (z_tc, z_si):
        assert np.abs(z - zq).max() < 4e-2 and np.abs(z - zq).mean() < 3e-3
        assert np.abs(z - ze).max() < 4e-2


@pytest.mark.parametrize("n", [5000, (1 << 18) + 77, (1 << 21) + 5])     # one pass / 4 chunks / 8 chunks, ragged tails
def test_query_host_matches_device_query(ddf, c1, n):
    """host-buffer entry: uploads, answers and downloads are pipelined in tile-aligned chunks on three
    streams for large batches; the results must be the device query's, bit for bit"""
    lay, m = c1
    o, d = random_rays(min(n, 1 << 16))
    reps = (n + len(o) - 1) // len(o)
    o = np.tile(o, (reps, 1))[:n].copy(); d = np.tile(d, (reps, 1))[:n].copy()
    oh, dh = torch.from_numpy(o).pin_memory(), torch.from_numpy(d).pin_memory()
    dist_h = torch.full((n,), float("nan")).pin_memory(); vis_h = torch.full((n,), float("nan")).pin_memory()
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        ddf.ddf_query_host(m, oh, dh, n, dist_h, vis_h, stream=st)       # synchronises inside the call
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    ddf.ddf_query(m, oh.cuda(), dh.cuda(), n, dist, vis)
    assert torch.equal(dist.cpu(), dist_h) and torch.equal(vis.cpu(), vis_h)
    ddf.ddf_query_host(m, oh, dh, n, dist_h, None)                        # default stream, no visibility output
    assert torch.equal(dist.cpu(), dist_h)


def test_model_from_device_fp32_blob(ddf, orc):
    lay = Layout(0, 4, 4, 2, 256, -1, 2, 0)
    blob = make_weights(lay, bias_scale=0.1)
    m_host = ddf.ddf_create(blob, lay)
    m_dev = ddf.ddf_create(torch.from_numpy(blob).cuda(), lay)
    o, d = random_rays(300)
    assert np.array_equal(_logits(ddf, m_host, o, d), _logits(ddf, m_dev, o, d))
    zq, _, _ = orc.forward(lay, blob, o, d, mode=1)
    assert np.abs(_logits(ddf, m_host, o, d) - zq).max() < 1e-3


# ------------------------------------------------------------------ sphere tracer

@pytest.fixture(scope="module")
def sdf(ddf):
    lay = layout_sdf()
    blob = make_weights(lay)
    m = ddf.ddf_create(blob, lay)
    yield lay, blob, m
    ddf.ddf_destroy(m)


def _trace(ddf, m, o, d, prm, want_trace=False):
    n = o.shape[0]
    t = torch.empty(n, device="cuda"); hit = torch.empty(n, dtype=torch.uint8, device="cuda")
    steps = torch.empty(n, dtype=torch.int32, device="cuda"); tot = torch.zeros(1, dtype=torch.int64, device="cuda")
    tp = torch.empty((n, prm.max_steps, 3), device="cuda") if want_trace else None
    ts = torch.empty((n, prm.max_steps), device="cuda") if want_trace else None
    ddf.sdf_sphere_trace(m, _cuda(o), _cuda(d), n, prm, t, hit, steps, tp, ts, tot)
    torch.cuda.synchronize()
    out = [t.cpu().numpy(), hit.cpu().numpy(), steps.cpu().numpy(), int(tot.item())]
    if want_trace:
        out += [tp.cpu().numpy(), ts.cpu().numpy()]
    return out


def test_sphere_trace_alpha0_is_bit_identical_to_the_cpu_tracer(ddf, orc, sdf):
    """P12: with the MLP term off the step rule alone decides everything: t, hit and steps must
    equal the CPU tracer's exactly (both carry the ray state in fp32 with the same fma order),
    and t reaches the analytic ray-sphere distance."""
    lay, blob, m = sdf
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 64, 64)
    for early in (0, 1):
        prm = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.0, early)
        t, hit, steps, tot = _trace(ddf, m, o, d, prm)
        rt, rhit, rsteps = orc.sphere_trace(lay, blob, o, d, 64, 1e-3, 6.0, 1.0, 0.0)
        assert np.array_equal(hit, rhit) and np.array_equal(steps, rsteps) and np.array_equal(t, rt)
        assert tot == (64 * len(o) if not early else int(steps.sum()))
    want = np.array([orc.ray_sphere(o[i], d[i], [0, 0, 0], 1.0) for i in range(len(o))])
    h = hit == 1
    assert h.sum() > 1000 and np.all(want[h] > 0) and np.all(np.abs(want[h] - t[h]) < 1e-3 / 0.05)


def _replay_step_rule(s_row, omega, eps, t_max, max_steps=64):
    """the (over-relaxed) step rule of include/ddf.h in fp32, fed with the values the kernel itself saw"""
    f = np.float32
    tt = f(0.0); tp = f(0.0); sp = f(np.nan); om = f(max(omega, 1.0)); h = 0; k = 0
    for k in range(max_steps):
        s = f(s_row[k])
        if om > 1 and f(abs(s) + abs(sp)) < f(tt - tp):
            tt = f(tp + sp); om = f(1.0); sp = f(np.nan)
            if tt > t_max or tt < 0: break
            continue
        if abs(s) < eps: h = 1; break
        tp, sp = tt, s
        tt = f(np.float64(om) * np.float64(s) + np.float64(tt))      # one rounding, like fmaf (the product is exact in fp64)
        if tt > t_max or tt < 0: break
    return h, k + 1, tt


@pytest.mark.parametrize("eps", [1e-2, 1e-3, 1e-4])
@pytest.mark.parametrize("omega", [0.0, 1.0, 1.1, 1.5, 1.9])
def test_over_relaxed_sphere_trace_and_thresholds_alpha0_bit_identical_to_the_cpu_tracer(ddf, orc, sdf, omega, eps):
    """SURVEY.md 8(f) f4, PAPER.md:112 ("across convergence thresholds"): with the MLP term off, the CUDA tracer with
    over-relaxed steps (fall-back included) and at every hit threshold returns the CPU tracer's t, hit and steps
    exactly, in both modes; omega 0 and 1 are the plain rule; large omega does fall back on this view."""
    lay, blob, m = sdf
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 48, 48)
    rt, rhit, rsteps, _, rs = orc.sphere_trace(lay, blob, o, d, 64, eps, 6.0, 1.0, 0.0, want_trace=True, omega=max(omega, 1.0))
    for early in (0, 1):
        prm = ddf.SdfTraceParams(64, eps, 6.0, 1.0, 0.0, early, omega)
        t, hit, steps, tot = _trace(ddf, m, o, d, prm)
        assert np.array_equal(hit, rhit) and np.array_equal(steps, rsteps) and np.array_equal(t, rt)
        assert tot == (64 * len(o) if not early else int(steps.sum()))
    assert 500 < rhit.sum() < len(o)
    if omega <= 1.0:
        pt, phit, psteps = orc.sphere_trace(lay, blob, o, d, 64, eps, 6.0, 1.0, 0.0)
        assert np.array_equal(pt, rt) and np.array_equal(psteps, rsteps)
    if omega >= 1.5:
        # a fall-back shows as a step whose t went backwards: the point after it is closer to the origin of the ray
        assert (rsteps[rhit == 1] >= 3).any()


@pytest.mark.parametrize("omega,eps", [(1.3, 1e-3), (1.0, 1e-2), (1.0, 1e-4), (1.6, 1e-2)])
def test_over_relaxed_sphere_trace_teacher_forcing_with_the_mlp_on(ddf, orc, sdf, omega, eps):
    """MLP on (alpha 0.05): both modes agree bit for bit, the values at the visited points match the oracle's SDF, and the
    rule of ddf.h replayed on the kernel's own values reproduces every decision, at other thresholds and with omega > 1."""
    lay, blob, m = sdf
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 24, 24)
    t, hit, steps, tot, tp, ts = _trace(ddf, m, o, d, ddf.SdfTraceParams(64, eps, 6.0, 1.0, 0.05, 0, omega), want_trace=True)
    t1, hit1, steps1, tot1, tp1, ts1 = _trace(ddf, m, o, d, ddf.SdfTraceParams(64, eps, 6.0, 1.0, 0.05, 1, omega), want_trace=True)
    assert np.array_equal(t, t1) and np.array_equal(hit, hit1) and np.array_equal(steps, steps1)
    assert np.array_equal(np.nan_to_num(ts, nan=-9.0), np.nan_to_num(ts1, nan=-9.0))
    assert tot == 64 * len(o) and tot1 == int(steps.sum())
    visited = ~np.isnan(ts)
    assert np.array_equal(visited.sum(1), steps)
    rows, cols = np.nonzero(visited)
    pick = np.random.default_rng(0).choice(len(rows), 600, replace=False)
    s_ref = orc.sdf_eval(lay, blob, tp[rows[pick], cols[pick]], 1.0, 0.05, mode=0)
    assert np.abs(ts[rows[pick], cols[pick]] - s_ref).max() < 0.05 * 4e-2 + 1e-6
    for i in range(len(o)):
        assert _replay_step_rule(ts[i], omega, eps, 6.0) == (hit[i], steps[i], t[i]), i
    assert 0.1 < hit.mean() < 0.95


def test_sphere_trace_teacher_forcing(ddf, orc, sdf):
    """MLP on: trajectories are chaotic under bf16, so the oracle re-evaluates s at the kernel's
    own visited points (same tolerance per step); end results are compared statistically."""
    lay, blob, m = sdf
    cam = orc.camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    o, d = orc.gen_camera(cam, 24, 24)
    prm = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 0)
    t, hit, steps, tot, tp, ts = _trace(ddf, m, o, d, prm, want_trace=True)
    prm1 = ddf.SdfTraceParams(64, 1e-3, 6.0, 1.0, 0.05, 1)
    t1, hit1, steps1, tot1, tp1, ts1 = _trace(ddf, m, o, d, prm1, want_trace=True)
    assert np.array_equal(t, t1) and np.array_equal(hit, hit1) and np.array_equal(steps, steps1)
    assert np.array_equal(np.nan_to_num(ts, nan=-9.0), np.nan_to_num(ts1, nan=-9.0))
    assert tot == 64 * len(o) and tot1 == int(steps.sum())
    visited = ~np.isnan(ts)
    assert np.array_equal(visited.sum(1), steps)
    rows, cols = np.nonzero(visited)
    pick = np.random.default_rng(0).choice(len(rows), 1200, replace=False)
    pts = tp[rows[pick], cols[pick]]
    s_ref = orc.sdf_eval(lay, blob, pts, 1.0, 0.05, mode=0)
    assert np.abs(ts[rows[pick], cols[pick]] - s_ref).max() < 0.05 * 4e-2 + 1e-6      # alpha * logit tolerance
    # the step rule applied to the kernel's own s reproduces its decisions
    for i in np.random.default_rng(1).choice(len(o), 64, replace=False):
        tt = np.float32(0.0); h = 0; k = 0
        for k in range(64):
            s = ts[i, k]
            if abs(s) < 1e-3: h = 1; break
            tt = np.float32(tt + s)
            if tt > 6.0 or tt < 0: break
        assert (h, k + 1, tt) == (hit[i], steps[i], t[i])
    # Statistics against the CPU tracer run end to end, on a 40 x 40 view (N = 1600 rays).  Per ray the two traces
    # diverge (bf16 vs fp64 values of a function with Lipschitz constant >> 1 feed back into the next point), so
    # the comparison is of two samples of one distribution.  Bound = 3 sigma of the difference of two INDEPENDENT
    # samples of size N - sqrt(2 p (1 - p) / N) for the hit rate, sqrt((var_gpu + var_cpu) / N) for the mean step
    # count - which over-estimates the spread of these paired samples (rays that converge quickly agree exactly).
    o2, d2 = orc.gen_camera(cam, 40, 40)
    t2, hit2, steps2, _ = _trace(ddf, m, o2, d2, prm1, want_trace=False)
    rt, rhit, rsteps = orc.sphere_trace(lay, blob, o2, d2, 64, 1e-3, 6.0, 1.0, 0.05)
    N = len(o2); ph = 0.5 * (hit2.mean() + rhit.mean())
    b_hit = 3.0 * math.sqrt(2.0 * ph * (1.0 - ph) / N)
    b_steps = 3.0 * math.sqrt((steps2.var() + rsteps.var()) / N)
    print("sphere trace, %d rays: hit rate %.4f vs %.4f (bound %.4f), mean steps %.2f vs %.2f (bound %.2f)"
          % (N, hit2.mean(), rhit.mean(), b_hit, steps2.mean(), rsteps.mean(), b_steps))
    assert 0.2 < ph < 0.9 and abs(hit2.mean() - rhit.mean()) < b_hit and abs(steps2.mean() - rsteps.mean()) < b_steps


def test_maximum_batch_2pow24_and_side_stream(ddf, orc, c1):
    """The largest batch BASELINE.json names (2^24 rays, 403 MB of ray data) in one call on a
    non-default stream: finite everywhere, sampled rays within tolerance, prefix-consistent with a
    smaller call (results do not depend on n)."""
    lay, m = c1
    n = 1 << 24
    o, d = random_rays(1 << 16)
    od = _cuda(o).repeat(n >> 16, 1); dd = _cuda(d).repeat(n >> 16, 1)
    dist = torch.full((n,), float("nan"), device="cuda"); vis = torch.full((n,), float("nan"), device="cuda")
    st = torch.cuda.Stream()
    st.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(st):
        ddf.ddf_query(m, od, dd, n, dist, vis, stream=st)
    st.synchronize()
    assert bool(torch.isfinite(dist).all()) and bool(torch.isfinite(vis).all())
    # the batch repeats a 2^16 block: every repetition must give the same bits
    assert torch.equal(dist.view(-1, 1 << 16)[0], dist.view(-1, 1 << 16)[-1])
    assert torch.equal(dist.view(-1, 1 << 16).min(0).values, dist.view(-1, 1 << 16).max(0).values)
    small_d = torch.empty(1 << 16, device="cuda"); small_v = torch.empty(1 << 16, device="cuda")
    ddf.ddf_query(m, od, dd, 1 << 16, small_d, small_v)
    assert torch.equal(small_d, dist[:1 << 16]) and torch.equal(small_v, vis[:1 << 16])
    from ddf_inputs import make_weights
    idx = np.arange(0, 1 << 16, 97)
    z, t, xi = orc.forward(lay, make_weights(lay), o[idx], d[idx], mode=0)
    g = dist[-(1 << 16):].cpu().numpy()[idx]
    assert (np.abs(g - t) / (1 + np.abs(t))).max() <= 1e-2


def test_reserved_calls_do_not_allocate(ddf, c1, sdf):
    """ddf_reserve sizes the per-batch workspaces; afterwards ddf_query_host, ddf_query_camera and sdf_sphere_trace
    leave the device's free memory where it was (no allocation in the query calls), also for a
    batch larger than any seen before."""
    lay, m = c1
    n = 300_000
    o, d = random_rays(n)
    oh, dh = torch.from_numpy(o).pin_memory(), torch.from_numpy(d).pin_memory()
    dist_h, vis_h = torch.empty(n).pin_memory(), torch.empty(n).pin_memory()
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    ddf.ddf_reserve(m, ddf.RESERVE_HOST | ddf.RESERVE_RAYS, n)
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ddf.ddf_query_host(m, oh, dh, n, dist_h, vis_h)
    cam = ddf.ddf_camera_from_seed(MASTER_SEED, STREAMS["camera_pos"], 2.5)
    ddf.ddf_query_camera(m, cam, 500, 600, dist, vis)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free0
    ddf.ddf_query(m, _cuda(o), _cuda(d), n, dist, vis)
    torch.cuda.synchronize()
    assert torch.equal(dist.cpu(), dist_h) and torch.equal(vis.cpu(), vis_h)
    slay, sblob, sm = sdf
    k = 50_000
    ddf.ddf_reserve(sm, ddf.RESERVE_TRACE, k)
    t = torch.empty(k, device="cuda"); hit = torch.empty(k, dtype=torch.uint8, device="cuda"); steps = torch.empty(k, dtype=torch.int32, device="cuda")
    oc, dc = _cuda(o[:k] * 2.0), _cuda(d[:k])
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    ddf.sdf_sphere_trace(sm, oc, dc, k, ddf.SdfTraceParams(8, 1e-3, 6.0, 1.0, 0.05, 1), t, hit, steps, None, None, None)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1


def test_reserve_on_the_cuda_core_path_is_bounded_and_covers_queries_and_wavefront_calls(ddf):
    """A model forced to the CUDA-core path answers a batch in passes of 16,384 rays, so ddf_reserve for 2^22 rays must
    size its activation workspace for 16,384 rows (about 172 MB at width 1280), not for 2^22 (44 GB); after the
    reservation a query larger than one pass and a wavefront call leave the free memory where it was.  ddf_query_ao
    with an spp that does not divide 32 keeps per-ray results: RESERVE_RAYS with that spp covers them on a fused model."""
    lay = layout_c1()
    m = ddf.ddf_create(make_weights(lay), lay)
    ddf.ddf_set_path(m, 1)
    n = 40_000                                                   # three passes, the last one ragged
    o, d = random_rays(n)
    oc, dc = _cuda(o), _cuda(d)
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    lit = torch.empty(n, dtype=torch.uint8, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ddf.ddf_reserve(m, ddf.RESERVE_WAVE, 1 << 22, 0)
    torch.cuda.synchronize()
    free1 = torch.cuda.mem_get_info()[0]
    wave_bytes = 40 * (1 << 22)
    assert free0 - free1 < wave_bytes + 256 * 1024 * 1024, (free0 - free1)      # 168 MB wavefront + ~172 MB activations
    ddf.ddf_query(m, oc, dc, n, dist, vis)
    ddf.ddf_query_shadowed(m, oc, dc, n, (3.0, 3.0, 3.0), 1e-3, dist, vis, lit, cnt)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free1
    assert 0 < int(cnt.item()) < n
    # same bits as the fused kernel's batch-size-independent answer on the first pass boundary
    ddf.ddf_set_path(m, 0)
    d0 = torch.empty(n, device="cuda"); v0 = torch.empty(n, device="cuda")
    ddf.ddf_query(m, oc, dc, n, d0, v0)
    torch.cuda.synchronize()
    assert float((d0 - dist).abs().max()) <= 1e-2 * (1 + float(d0.abs().max())) and float((v0 - vis).abs().max()) <= 1e-2
    # fused model, spp = 12: the unfused reduce's per-ray results come from the reservation
    n_pts, spp = 2_000, 12
    ao = torch.empty(n_pts, device="cuda")
    ddf.ddf_reserve(m, ddf.RESERVE_RAYS, n_pts * spp, spp)
    torch.cuda.synchronize()
    free2 = torch.cuda.mem_get_info()[0]
    ddf.ddf_query_ao(m, oc[:n_pts * spp], dc[:n_pts * spp], n_pts, spp, 2.0, ao)
    torch.cuda.synchronize()
    assert torch.cuda.mem_get_info()[0] == free2
    assert bool(((ao >= 0) & (ao <= 1)).all())
    ddf.ddf_destroy(m)


def test_a_model_belongs_to_the_device_it_was_created_on(ddf, c1):
    """ddf_get_info(model, 4) is the creating device; with another device current every call is refused (needs two GPUs
    for the refusal itself; on a one-GPU box only the ownership record and the pass-through are checked)."""
    lay, m = c1
    assert ddf.ddf_get_info(m, 4) == torch.cuda.current_device()
    if torch.cuda.device_count() < 2:
        return
    home = torch.cuda.current_device()
    o, d = random_rays(64)
    oc, dc = _cuda(o), _cuda(d)
    dist = torch.empty(64, device="cuda"); vis = torch.empty(64, device="cuda")
    try:
        torch.cuda.set_device((home + 1) % torch.cuda.device_count())
        with pytest.raises(ddf.DdfError, match="invalid argument"):
            ddf.ddf_query(m, oc, dc, 64, dist, vis)
        with pytest.raises(ddf.DdfError, match="invalid argument"):
            ddf.ddf_reserve(m, ddf.RESERVE_HOST, 64)
    finally:
        torch.cuda.set_device(home)
    ddf.ddf_query(m, oc, dc, 64, dist, vis)
    torch.cuda.synchronize()
    assert bool(torch.isfinite(dist).all())
