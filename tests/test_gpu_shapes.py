"""Layouts at the edges of what each kernel serves (one layer, 16 layers, 8 column chunks, skip into
the last layer, no frequency bands, 16 bands, point input, widths that are padded, networks that only
the CUDA-core path takes): logits against both oracle modes through the C ABI."""
import numpy as np
import pytest
import torch

from ddf_inputs import Layout, make_weights, random_rays

pytestmark = pytest.mark.gpu

LAYOUTS = [
    (Layout(0, 10, 4, 1, 256, -1, 2, 1), 1),      # a single hidden layer on the wide kernel
    (Layout(0, 10, 4, 2, 768, 1, 2, 1), 1),       # 3 column chunks, skip into the last layer
    (Layout(0, 4, 4, 3, 2048, 2, 2, 1), 1),       # 8 column chunks: the widest the kernel tiles
    (Layout(0, 10, 4, 16, 256, 15, 2, 1), 1),     # 16 layers: the deepest the wide kernel takes
    (Layout(1, 10, 0, 2, 512, 1, 1, 0), 1),       # point input, one linear output (SDF family)
    (Layout(0, 0, 0, 2, 256, -1, 2, 0), 1),       # no frequency bands: E = 6
    (Layout(0, 16, 16, 2, 256, 1, 2, 1), 1),      # 16 bands each: E = 198 (4 K blocks of gamma)
    (Layout(0, 10, 4, 1, 64, -1, 2, 0), 1),       # narrow kernel, one layer, two gamma blocks
    (Layout(0, 0, 0, 3, 128, 2, 2, 0), 1),        # narrow kernel, skip into the last layer
    (Layout(0, 10, 4, 3, 1000, 1, 2, 0), 1),      # width padded 1000 -> 1024
    (Layout(0, 10, 4, 20, 64, 7, 1, 1), 0),       # 20 x 64: too deep for either tensor-core kernel
]


@pytest.mark.parametrize("lay,fused", LAYOUTS)
def test_edge_layouts_match_oracle(orc, lay, fused):
    import paper_2606_00817_b200 as ddf
    ddf.build()
    o, d = random_rays(700, seed=9)
    if lay.input_kind == 1:
        d = None
    blob = make_weights(lay, seed=3, bias_scale=0.1)
    m = ddf.ddf_create(blob, lay)
    assert ddf.ddf_get_info(m, 0) == fused
    od, dd = torch.from_numpy(o).cuda(), torch.from_numpy(d).cuda() if d is not None else None
    zq, _, _ = orc.forward(lay, blob, o, d, mode=1)
    ze, _, _ = orc.forward(lay, blob, o, d, mode=0)
    assert 0.1 < np.abs(zq).mean() < 5.0                       # the comparison is not vacuous
    # the wide kernel answers a batch this small either as one persistent launch (path 3) or split by
    # output columns, one launch per layer (path 4, the automatic choice here): both against the oracle
    wide = bool(fused) and ddf.ddf_get_info(m, 3) == 256
    zs = []
    for path in ((3, 4, 0) if wide else (0,)):
        ddf.ddf_set_path(m, path)
        z = torch.full((700, lay.n_out), float("nan"), device="cuda")
        ddf.ddf_query_logits(m, od, dd, 700, z)
        torch.cuda.synchronize()
        launches = ddf.ddf_get_info(m, 1)
        if wide:
            assert launches == (1 if path == 3 else lay.n_hidden + 2)
        else:
            assert (launches == 1) == bool(fused)
        e = np.abs(z.cpu().numpy() - zq)
        assert e.max() <= 4e-2 and e.mean() <= 3e-3, (path, e.max(), e.mean())
        assert np.abs(z.cpu().numpy() - ze).max() <= 6e-2
        zs.append(z)
    for z in zs[1:]:
        assert torch.equal(z, zs[0])                           # the same bits whichever way the batch is cut
    ddf.ddf_destroy(m)
