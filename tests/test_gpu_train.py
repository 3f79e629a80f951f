"""Training the hash-grid field on the GPU against oracle/ddf_hash_oracle.c:
loss and gradients of one batch, Adam steps, the batch generator, and a short run whose loss falls.
Both arithmetics of include/ddf.h run every test against the fp64 oracle.  DDF_TRAIN_FP32 (CUDA
cores, atomic accumulation): gradients agree to 2e-4 of their scale.  DDF_TRAIN_BF16X3 (tensor cores,
every operand split into two bf16 terms, lo x lo dropped): a product carries ~2^-16 relative error, far
inside the same bound, so both are held to it.  Parameters after k Adam steps
agree to a few lr * 1e-2 either way."""
import numpy as np
import pytest
import torch

from ddf_inputs import MASTER_SEED, STREAMS, HashLayout, layout_hash_paper, make_hash_table, make_hash_mlp, random_rays

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def ddf():
    import paper_2606_00817_b200 as pkg
    pkg.build()
    assert torch.cuda.is_available()
    return pkg


def _cuda(a):
    return torch.from_numpy(np.ascontiguousarray(a)).cuda()


def _batch(n, seed=3):
    o, d = random_rays(n)
    rng = np.random.default_rng(seed)
    return (o * 1.5).astype(np.float32), d, rng.uniform(0.2, 3.0, n).astype(np.float32), (rng.uniform(size=n) < 0.6).astype(np.uint8)


ARITH = [pytest.param(1, id="fp32"), pytest.param(0, id="bf16x3")]
LOSS_TOL = {1: 2e-5, 0: 2e-5}
GRAD_TOL = {1: 2e-4, 0: 2e-4}


@pytest.mark.parametrize("arith", ARITH)
@pytest.mark.parametrize("kw", [dict(n_levels=4, log2_table=10, base_res=4, growth=2.0, n_freq_dir=2, n_hidden=2),
                                dict(n_levels=6, log2_table=12, n_freq_dir=4, n_hidden=1),
                                dict()])
def test_loss_and_gradients_match_oracle(ddf, orc, kw, arith):
    lay = HashLayout(**kw)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    n = 1000 if kw else 300                                  # the paper-size table: fewer rays, the oracle's gradient is dense
    o, d, t, hit = _batch(n)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(dist_clamp=2.0, arithmetic=arith))
    loss = torch.zeros(1, device="cuda"); gt = torch.empty(2 * n_ent, device="cuda"); gm = torch.empty(len(mlp), device="cuda")
    ddf.ddf_trainer_loss_grads(tr, _cuda(o), _cuda(d), _cuda(t), _cuda(hit), n, loss, gt, gm)
    torch.cuda.synchronize()
    rl, rgt, rgm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, orc.train_params(dist_clamp=2.0))
    print("arith", arith, "loss err", abs(float(loss) - rl) / max(1.0, abs(rl)))
    assert abs(float(loss) - rl) < LOSS_TOL[arith] * max(1.0, abs(rl))
    for g, r, what in ((gm.cpu().numpy(), rgm, "mlp"), (gt.cpu().numpy(), rgt, "table")):
        scale = np.abs(r).max()
        print("arith", arith, what, "max err / scale", np.abs(g - r).max() / scale, "rms err / rms", np.sqrt(((g - r) ** 2).mean() / (r ** 2).mean()))
        assert scale > 0 and np.abs(g - r).max() <= GRAD_TOL[arith] * scale + 1e-9, (what, np.abs(g - r).max(), scale)
        assert np.array_equal(g == 0, r == 0) or what == "mlp"       # untouched table entries stay exactly zero
    # a second call gives the same answer: the accumulator was left clean
    ddf.ddf_trainer_loss_grads(tr, _cuda(o), _cuda(d), _cuda(t), _cuda(hit), n, loss, gt, gm)
    assert np.abs(gm.cpu().numpy() - rgm).max() <= GRAD_TOL[arith] * np.abs(rgm).max()
    ddf.ddf_trainer_destroy(tr)


@pytest.mark.parametrize("arith", ARITH)
@pytest.mark.parametrize("kw,n", [(dict(n_levels=1, log2_table=14, n_freq_dir=0, n_hidden=1), 1),
                                  (dict(n_levels=1, log2_table=14, n_freq_dir=0, n_hidden=2), 129),
                                  (dict(n_levels=16, log2_table=9, base_res=2, growth=1.3, n_freq_dir=4, n_hidden=2), 127),
                                  (dict(n_levels=3, log2_table=19, base_res=16, growth=1.5, n_freq_dir=1, n_hidden=1), 128)])
def test_degenerate_layouts_and_batches(ddf, orc, arith, kw, n):
    """one ray; one level with an odd entry count (no replicated accumulator) and no direction bands (a 5-wide
    input); 16 tiny levels that are all replicated; batches of T - 1, T, T + 1 rays"""
    lay = HashLayout(**kw)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    o, d, t, hit = _batch(n, seed=n)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(dist_clamp=2.0, arithmetic=arith))
    loss = torch.zeros(1, device="cuda"); gt = torch.empty(2 * n_ent, device="cuda"); gm = torch.empty(len(mlp), device="cuda")
    ddf.ddf_trainer_loss_grads(tr, _cuda(o), _cuda(d), _cuda(t), _cuda(hit), n, loss, gt, gm)
    torch.cuda.synchronize()
    rl, rgt, rgm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, orc.train_params(dist_clamp=2.0))
    assert abs(float(loss) - rl) < LOSS_TOL[arith] * max(1.0, abs(rl))
    for g, r in ((gm.cpu().numpy(), rgm), (gt.cpu().numpy(), rgt)):
        assert np.isfinite(g).all() and np.abs(g - r).max() <= GRAD_TOL[arith] * np.abs(r).max() + 1e-9
    assert np.array_equal(gt.cpu().numpy() == 0, rgt == 0)
    ddf.ddf_trainer_destroy(tr)


@pytest.mark.parametrize("arith", ARITH)
def test_more_tiles_than_sms_ragged_tail_and_a_growing_batch(ddf, orc, arith):
    """40,001 rays = 313 tiles of 128 on 148 SMs: every CTA walks several tiles (the tensor-core path keeps its
    weight-gradient accumulator in tensor memory across them) and the last tile has one ray; the same trainer
    first sees a small batch, so its feature workspace has to grow."""
    lay = HashLayout(n_levels=5, log2_table=11, base_res=4, growth=1.7, n_freq_dir=3, n_hidden=2)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(dist_clamp=2.0, arithmetic=arith))
    P = orc.train_params(dist_clamp=2.0)
    for n in (130, 40001):
        o, d, t, hit = _batch(n + 600, seed=n)
        # The loss has no gradient where a hidden pre-activation is 0, and a forward pass rounded at 2^-17
        # (bf16x3) or 2^-24 (fp32) instead of fp64 puts a ray that close to a kink on the other side of it
        # (reading T7).  Among 40,000 rays x 128 units a few always are: keep the rays whose every
        # pre-activation clears 1e-4 (about 1 % go) and compare the gradients of that batch.
        keep = np.nonzero(orc.hash_relu_margin(lay, table, mlp, o, d) > 1e-4)[0][:n]
        assert len(keep) == n
        o, d, t, hit = (np.ascontiguousarray(a[keep]) for a in (o, d, t, hit))
        loss = torch.zeros(1, device="cuda"); gt = torch.empty(2 * n_ent, device="cuda"); gm = torch.empty(len(mlp), device="cuda")
        ddf.ddf_trainer_loss_grads(tr, _cuda(o), _cuda(d), _cuda(t), _cuda(hit), n, loss, gt, gm)
        torch.cuda.synchronize()
        rl, rgt, rgm = orc.hash_loss_grads(lay, table, mlp, o, d, t, hit, P)
        assert abs(float(loss) - rl) < 5e-5 * max(1.0, abs(rl))                 # 313 atomic partial sums in fp32
        for g, r in ((gm.cpu().numpy(), rgm), (gt.cpu().numpy(), rgt)):
            assert np.abs(g - r).max() <= GRAD_TOL[arith] * np.abs(r).max() + 1e-9, (n, np.abs(g - r).max() / np.abs(r).max())
    ddf.ddf_trainer_destroy(tr)


@pytest.mark.parametrize("arith", ARITH)
def test_adam_steps_match_oracle(ddf, orc, arith):
    lay = HashLayout(n_levels=4, log2_table=10, base_res=4, growth=2.0, n_freq_dir=2, n_hidden=2)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    kwargs = dict(lr0=1e-2, total_steps=10, dist_clamp=2.0, adam_eps=1e-8)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(arithmetic=arith, **kwargs))
    P = orc.train_params(**kwargs)
    rt, rm = table.copy(), mlp.copy()
    mt, vt, mm, vm = np.zeros(len(rt)), np.zeros(len(rt)), np.zeros(len(rm)), np.zeros(len(rm))
    losses = []
    for s in range(4):
        o, d, t, hit = _batch(512, seed=10 + s)
        loss = torch.zeros(1, device="cuda")
        ddf.ddf_trainer_step(tr, _cuda(o), _cuda(d), _cuda(t), _cuda(hit), 512, loss)
        rl, gt, gm = orc.hash_loss_grads(lay, rt, rm, o, d, t, hit, P)
        lr = orc.lr_at(P, s)
        orc.adam_step(rt, gt, mt, vt, s + 1, lr, P); orc.adam_step(rm, gm, mm, vm, s + 1, lr, P)
        losses.append((float(loss), rl))
    assert ddf.ddf_trainer_steps(tr) == 4
    gt_, gm_ = ddf.ddf_trainer_export(tr, len(table), len(mlp))
    for (a, b) in losses:
        assert abs(a - b) < 1e-3 * max(1.0, abs(b)), losses
    # Adam divides by sqrt(v): where a gradient is ~1e-7 of the scale its sign is rounding noise, so compare in
    # units of the step size lr (each step moves a parameter by at most ~lr)
    touched = (rt != table)
    assert np.abs(gm_ - rm).max() < 0.05 * 1e-2 * 4 and np.abs(gt_ - rt)[touched].max() < 0.05 * 1e-2 * 4
    assert np.abs(gm_ - rm).mean() < 2e-3 * 1e-2 and np.array_equal(gt_[~touched], table[~touched])
    ddf.ddf_trainer_destroy(tr)


@pytest.mark.parametrize("arith", ARITH)
def test_steps_on_a_side_stream_follow_the_work_already_in_it(ddf, orc, arith):
    """The kernels of a step are chained by programmatic dependent launch: each may be scheduled before its
    predecessor has finished and waits where it first needs it.  Batches are generated and consumed back to
    back on a side stream, with no synchronisation, into ONE set of buffers that the next generator call
    overwrites; the result must be the run that synchronises after every call."""
    lay = HashLayout(n_levels=6, log2_table=12, n_freq_dir=4, n_hidden=2)
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=0.5); mlp = make_hash_mlp(lay, bias_scale=0.2)
    sc = orc.TRAIN_SCENE
    scene = ddf.DdfScene(sc["sphere_c"], sc["sphere_r"], sc["bmin"], sc["bmax"])
    B, steps = 5000, 12
    out = []
    for mode in ("async", "sync"):
        tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(total_steps=steps, lr0=1e-3, arithmetic=arith))
        st = torch.cuda.Stream()
        o = torch.empty((B, 3), device="cuda"); d = torch.empty((B, 3), device="cuda")
        t = torch.empty(B, device="cuda"); hit = torch.empty(B, dtype=torch.uint8, device="cuda")
        losses = torch.zeros(steps, device="cuda")
        torch.cuda.synchronize()
        for s in range(steps):
            ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], s, B, 2.0, o, d, t, hit, stream=st.cuda_stream)
            if mode == "sync": torch.cuda.synchronize()
            ddf.ddf_trainer_step(tr, o, d, t, hit, B, losses[s:s + 1], stream=st.cuda_stream)
            if mode == "sync": torch.cuda.synchronize()
        torch.cuda.synchronize()
        tt, mm = ddf.ddf_trainer_export(tr, 2 * n_ent, len(mlp))
        out.append((losses.cpu().numpy(), tt, mm))
        ddf.ddf_trainer_destroy(tr)
    (la, ta, ma), (ls, ts, ms) = out
    assert np.isfinite(la).all() and np.allclose(la, ls, rtol=2e-4, atol=1e-6), (la, ls)
    # atomics reorder the sums, Adam divides by sqrt(v): compare in units of the total step budget (12 x lr)
    assert np.abs(ma - ms).max() < 0.05 * steps * 1e-3 and np.abs(ta - ts).max() < 0.05 * steps * 1e-3
    assert np.abs(ma - ms).mean() < 1e-5 and np.abs(ta - ts).mean() < 1e-5


def test_supervision_and_batch_generator(ddf, orc):
    sc = orc.TRAIN_SCENE
    scene = ddf.DdfScene(sc["sphere_c"], sc["sphere_r"], sc["bmin"], sc["bmax"])
    n = 20000
    o, d = random_rays(n); o = (o * 2.0).astype(np.float32)
    t = torch.empty(n, device="cuda"); hit = torch.empty(n, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, _cuda(o), _cuda(d), n, t, hit)
    ref = np.array([orc.solid_scene_raycast(o[i], d[i], sc["sphere_c"], sc["sphere_r"], sc["bmin"], sc["bmax"]) for i in range(n)])
    assert np.array_equal(hit.cpu().numpy().astype(bool), ref > 0) and 0.05 < (ref > 0).mean() < 0.95
    assert np.allclose(t.cpu().numpy()[ref > 0], ref[ref > 0], rtol=1e-6, atol=1e-6)
    # batch generator against its twin
    og = torch.empty((n, 3), device="cuda"); dg = torch.empty((n, 3), device="cuda")
    ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], 7, n, 2.0, og, dg, t, hit)
    ro, rd, rt, rh = orc.gen_train_batch(MASTER_SEED, STREAMS["train_rays"], 7, n, 2.0)
    same = hit.cpu().numpy() == rh
    close = same & (np.abs(og.cpu().numpy() - ro).max(axis=1) < 1e-4) & (np.abs(dg.cpu().numpy() - rd).max(axis=1) < 1e-4)
    assert same.mean() > 0.999 and close.mean() > 0.998          # fp32 vs fp64 flips a grazing ray now and then
    assert np.allclose(t.cpu().numpy()[close], rt[close], atol=2e-4)
    assert np.allclose(np.linalg.norm(dg.cpu().numpy(), axis=1), 1.0, atol=1e-5)
    # the targets are the analytic first-surface distances of the rays that were emitted
    t2 = torch.empty(n, device="cuda"); h2 = torch.empty(n, dtype=torch.uint8, device="cuda")
    ddf.ddf_scene_raycast(scene, og, dg, n, t2, h2)
    hh = hit.cpu().numpy().astype(bool)
    ok = (h2.cpu().numpy().astype(bool) == hh)
    assert ok.mean() > 0.995                                     # surface-anchored origins sit 1e-3 off the surface
    both = ok & hh
    assert np.abs(t2.cpu().numpy() - t.cpu().numpy())[both].max() < 1e-3
    assert 0.3 < hh.mean() < 0.95


@pytest.mark.parametrize("arith", ARITH)
def test_short_training_run_reduces_the_loss_and_exports_a_usable_field(ddf, orc, arith):
    lay = layout_hash_paper()
    n_ent = ddf.ddf_hashgrid_table_entries(lay)
    table = make_hash_table(lay, n_ent, scale=1e-4); mlp = make_hash_mlp(lay)
    tr = ddf.ddf_trainer_create(table, mlp, lay, ddf.make_train_params(total_steps=1500, arithmetic=arith))
    sc = orc.TRAIN_SCENE
    scene = ddf.DdfScene(sc["sphere_c"], sc["sphere_r"], sc["bmin"], sc["bmax"])
    B = 16384
    o = torch.empty((B, 3), device="cuda"); d = torch.empty((B, 3), device="cuda")
    t = torch.empty(B, device="cuda"); hit = torch.empty(B, dtype=torch.uint8, device="cuda")
    losses = torch.zeros(1500, device="cuda")
    for s in range(1500):
        ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], s, B, 2.0, o, d, t, hit)
        ddf.ddf_trainer_step(tr, o, d, t, hit, B, losses[s:s + 1])
    torch.cuda.synchronize()
    l = losses.cpu().numpy()
    assert np.isfinite(l).all() and l[-20:].mean() < 0.35 * l[:5].mean(), (l[:5], l[-5:])
    tt, mm = ddf.ddf_trainer_export(tr, 2 * n_ent, len(mlp))
    ddf.ddf_trainer_destroy(tr)
    # the exported field, served by the inference kernel, agrees with the analytic scene on fresh rays
    m = ddf.ddf_create_hashgrid(tt, mm, lay)
    ddf.ddf_gen_train_batch(scene, MASTER_SEED, STREAMS["train_rays"], 100000, B, 2.0, o, d, t, hit)
    dist = torch.empty(B, device="cuda"); vis = torch.empty(B, device="cuda")
    ddf.ddf_query(m, o, d, B, dist, vis)
    agree = ((vis > 0.5) == (hit > 0)).float().mean().item()
    hh = hit > 0
    err = (dist - t).abs()[hh].median().item()
    print("arith", arith, "agree", agree, "median err", err, "loss", l[:3], l[-3:])
    assert agree > 0.88 and err < 0.06, (agree, err)
    ddf.ddf_destroy(m)
