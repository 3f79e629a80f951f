"""Stream capture (CUDA graphs) of library calls: a call whose workspaces already exist issues only
stream-ordered work (kernels, memsets, device-to-device copies; no allocation, no synchronisation), so it
can be captured once and replayed.  The wavefront loop - six launches whose secondary batch size never
leaves the device - and the training pass with its dependent-launch chain are the launch-bound cases."""
import numpy as np
import pytest
import torch

from ddf_inputs import (MASTER_SEED, STREAMS, HashLayout, layout_c1, layout_hash_paper, make_weights, make_hash_table,
                        make_hash_mlp, random_rays)

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ddf():
    import paper_2606_00817_b200 as pkg
    pkg.build()
    assert torch.cuda.is_available()
    return pkg


def _capture(fn):
    g = torch.cuda.CUDAGraph()
    s = torch.cuda.Stream()
    s.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(s):
        g.capture_begin()
        try:
            fn(s.cuda_stream)
        finally:
            g.capture_end()
    torch.cuda.synchronize()
    return g


@pytest.mark.parametrize("kind", ["hash", "dense"])
def test_wavefront_call_replays_from_a_graph(ddf, kind):
    if kind == "hash":
        hl = layout_hash_paper(); mlp = make_hash_mlp(hl).copy(); mlp[-1] = 1.0
        m = ddf.ddf_create_hashgrid(make_hash_table(hl, ddf.ddf_hashgrid_table_entries(hl)), mlp, hl)
        n = 50000
    else:
        lay = layout_c1(); blob = make_weights(lay).copy(); blob[-1] = 0x3F80
        m = ddf.ddf_create(blob, lay)
        n = 5000
    o_np, d_np = random_rays(n)
    o = torch.from_numpy(o_np).cuda(); d = torch.from_numpy(d_np).cuda()
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda")
    mask = torch.empty(n, dtype=torch.uint8, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    lights = [(3.0, 3.0, 3.0), (-3.0, 2.0, 1.0)]
    ddf.ddf_query_shadowed_lights(m, o, d, n, lights, 1e-3, dist, vis, mask, cnt)         # eager: creates the workspaces
    torch.cuda.synchronize()
    want = (dist.clone(), vis.clone(), mask.clone(), int(cnt.item()))
    assert 0 < want[3] < 2 * n
    g = _capture(lambda st: ddf.ddf_query_shadowed_lights(m, o, d, n, lights, 1e-3, dist, vis, mask, cnt, stream=st))
    # new inputs in the same buffers: the replay must answer for them
    perm = torch.randperm(n, device="cuda")
    o.copy_(o[perm]); d.copy_(d[perm])
    dist.zero_(); vis.zero_(); mask.fill_(0xFF); cnt.zero_()
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(dist, want[0][perm]) and torch.equal(vis, want[1][perm]) and torch.equal(mask, want[2][perm])
    assert int(cnt.item()) == want[3]
    ddf.ddf_destroy(m)


@pytest.mark.parametrize("kind", ["hash", "dense"])
def test_ao_wavefront_call_replays_from_a_graph(ddf, kind):
    """ddf_query_ao_wavefront with the fused reduce never reads the hit count on the host: capturable"""
    if kind == "hash":
        hl = layout_hash_paper(); mlp = make_hash_mlp(hl).copy(); mlp[-1] = 1.0
        m = ddf.ddf_create_hashgrid(make_hash_table(hl, ddf.ddf_hashgrid_table_entries(hl)), mlp, hl)
        W, H = 250, 200
    else:
        lay = layout_c1(); blob = make_weights(lay).copy(); blob[-1] = 0x3F80
        m = ddf.ddf_create(blob, lay)
        W, H = 100, 50
    n = W * H
    o_np, d_np = random_rays(n)
    o = torch.from_numpy(o_np).cuda(); d = torch.from_numpy(d_np).cuda()
    dist = torch.empty(n, device="cuda"); vis = torch.empty(n, device="cuda"); nrm = torch.empty((n, 3), device="cuda")
    ao = torch.empty(n, device="cuda"); cnt = torch.zeros(1, dtype=torch.int64, device="cuda")
    call = lambda st=None: ddf.ddf_query_ao_wavefront(m, o, d, W, H, 16, 11, 3, 1e-3, 2.0, dist, vis, nrm, ao, cnt, stream=st)
    call()                                                                                # eager: creates the workspaces
    torch.cuda.synchronize()
    g = _capture(lambda st: call(st))
    o.copy_(o.flip(0).contiguous()); d.copy_(d.flip(0).contiguous())                      # new inputs in the same buffers
    call(); torch.cuda.synchronize()
    want = (dist.clone(), vis.clone(), nrm.clone(), ao.clone(), int(cnt.item()))
    assert 0 < want[4] < 16 * n
    dist.zero_(); vis.zero_(); nrm.zero_(); ao.zero_(); cnt.zero_()
    g.replay(); torch.cuda.synchronize()
    assert torch.equal(dist, want[0]) and torch.equal(vis, want[1]) and torch.equal(nrm, want[2]) and torch.equal(ao, want[3])
    assert int(cnt.item()) == want[4]
    # the whole shaded frame (shadow loop for two lights + AO loop on one primary query) replays too
    mask = torch.empty(n, dtype=torch.uint8, device="cuda"); cs = torch.zeros(2, dtype=torch.int64, device="cuda")
    lights = [(3.0, 3.0, 3.0), (-3.0, 2.0, 1.0)]
    shaded = lambda st=None: ddf.ddf_query_shaded(m, o, d, W, H, lights, 16, 11, 3, 1e-3, 2.0, dist, vis, mask, nrm, ao, cs, stream=st)
    shaded(); torch.cuda.synchronize()
    g2 = _capture(lambda st: shaded(st))
    o.copy_(o.flip(0).contiguous()); d.copy_(d.flip(0).contiguous())
    shaded(); torch.cuda.synchronize()
    want2 = (dist.clone(), vis.clone(), mask.clone(), nrm.clone(), ao.clone(), cs.clone())
    for x in (dist, vis, mask, nrm, ao, cs): x.zero_()
    g2.replay(); torch.cuda.synchronize()
    for got, ref in zip((dist, vis, mask, nrm, ao, cs), want2): assert torch.equal(got, ref)
    assert int(cs[0].item()) > 0 and int(cs[1].item()) > 0
    ddf.ddf_destroy(m)


def test_training_pass_replays_from_a_graph(ddf, orc):
    """loss + gradients of one batch (gather -> tcgen05 MLP -> scatter, chained by programmatic dependent
    launch, then the fold and the copies out) captured and replayed on a new batch, against the oracle."""
    lay = HashLayout(n_levels=6, log2_table=12, n_freq_dir=4, n_hidden=2)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(dist_clamp=2.0))
    n = 700
    rng = np.random.default_rng(11)

    def batch(seed):
        o, d = random_rays(n + seed)
        return ((o[seed:] * 1.5).astype(np.float32), np.ascontiguousarray(d[seed:]),
                rng.uniform(0.2, 3.0, n).astype(np.float32), (rng.uniform(size=n) < 0.6).astype(np.uint8))
    o0, d0, t0, h0 = batch(0)
    o = torch.from_numpy(o0).cuda(); d = torch.from_numpy(d0).cuda(); t = torch.from_numpy(t0).cuda(); hit = torch.from_numpy(h0).cuda()
    loss = torch.zeros(1, device="cuda"); gt = torch.empty(2 * n_ent, device="cuda"); gm = torch.empty(len(mlp), device="cuda")
    ddf.ddf_trainer_loss_grads(tr, o, d, t, hit, n, loss, gt, gm)                          # eager: workspace for n rays
    torch.cuda.synchronize()
    g = _capture(lambda st: ddf.ddf_trainer_loss_grads(tr, o, d, t, hit, n, loss, gt, gm, stream=st))
    o1, d1, t1, h1 = batch(5)
    o.copy_(torch.from_numpy(o1)); d.copy_(torch.from_numpy(d1)); t.copy_(torch.from_numpy(t1)); hit.copy_(torch.from_numpy(h1))
    for _ in range(2):                                       # twice: the accumulators are left clean by the captured work
        loss.zero_(); gt.fill_(7.0); gm.fill_(7.0)
        g.replay(); torch.cuda.synchronize()
        rl, rgt, rgm = orc.hash_loss_grads(lay, table, mlp, o1, d1, t1, h1, orc.train_params(dist_clamp=2.0))
        assert abs(float(loss) - rl) < 2e-5 * max(1.0, abs(rl))
        assert np.abs(gm.cpu().numpy() - rgm).max() <= 2e-4 * np.abs(rgm).max()
        assert np.abs(gt.cpu().numpy() - rgt).max() <= 2e-4 * np.abs(rgt).max()
    ddf.ddf_trainer_destroy(tr)
