"""Pins of the hash-grid DDF oracle (oracle/ddf_hash_oracle.c) - CPU only.

What is fixed from outside the oracle: the paper's own counts ("about 13M" table
parameters, "about 8k" MLP parameters, "52 MB"), the interpolation invariants of a trilinear
grid (partition of unity, exact reproduction of linear fields, vertex values, continuity), the
index formulas of the encoding the paper follows, recomputed here with Python integers, and an
independent numpy evaluator with a different loop structure.
"""
import numpy as np
import pytest

from ddf_inputs import (HashLayout, layout_hash_paper, make_hash_table, make_hash_mlp, hash_mlp_shapes,
                        random_rays, f32_to_bf16_bits, bf16_bits_to_f32)

P2, P3 = 2654435761, 805459861


def test_paper_counts(orc):
    """16 levels x 2 features x 2^19 entries, base 16, growth 1.5 -> "about 13M"
    parameters and, with the "about 8k" MLP, "a stored field of 52 MB"."""
    lay = layout_hash_paper()
    res = [orc.hash_level(lay, l)[0] for l in range(16)]
    assert res == [16, 24, 36, 54, 81, 121, 182, 273, 410, 615, 922, 1383, 2075, 3113, 4670, 7006]   # floor(16 * 1.5^l)
    ent = [orc.hash_level(lay, l)[1] for l in range(16)]
    assert ent[:4] == [17 ** 3, 25 ** 3, 37 ** 3, 55 ** 3]         # whole grids that fit 2^19
    assert ent[4:] == [2 ** 19] * 12 and 82 ** 3 > 2 ** 19         # the rest is hashed
    assert [orc.hash_level(lay, l)[3] for l in range(16)] == [False] * 4 + [True] * 12
    n = orc.hash_table_entries(lay)
    assert n == 6_529_022 and 12.5e6 < 2 * n < 13.5e6             # "about 13M parameters"
    assert orc.hash_mlp_in(lay) == 32 + 27
    assert orc.hash_mlp_params(lay) == 59 * 64 + 64 + 64 * 64 + 64 + 64 * 2 + 2 == 8130   # "about 8k"
    assert abs((2 * n + 8130) * 4 / 1e6 - 52.0) < 0.5             # "52 MB"
    offs = [orc.hash_level(lay, l)[2] for l in range(16)]
    assert offs == list(np.cumsum([0] + ent[:-1]))
    # the same facts as a cited fixture (tests/golden/hashgrid_paper_counts.txt)
    import os
    gold = {}
    for line in open(os.path.join(os.path.dirname(__file__), "golden", "hashgrid_paper_counts.txt")):
        if line.strip() and not line.startswith("#"):
            k, *v = line.split(); gold[k] = v
    assert [int(x) for x in gold["resolutions"]] == res and int(gold["table_entries"][0]) == n
    assert int(gold["table_parameters"][0]) == 2 * n and round(2 * n / 1e6) == int(gold["paper_table_parameters_millions"][0])
    assert int(gold["mlp_parameters"][0]) == orc.hash_mlp_params(lay) and round(8130 / 1e3) == int(gold["paper_mlp_parameters_thousands"][0])
    assert round((2 * n + 8130) * 4 / 1e6) == int(gold["paper_field_megabytes"][0])


def test_index_formulas_by_hand(orc):
    lay = layout_hash_paper()
    # dense level 1 (N = 24, 25 vertices per axis): x fastest
    assert orc.hash_index(lay, 1, 3, 4, 5) == 3 + 25 * (4 + 25 * 5)
    assert orc.hash_index(lay, 0, 16, 16, 16) == 17 ** 3 - 1
    # hashed level: (ix ^ iy * pi2 ^ iz * pi3) mod 2^19 with 32-bit products
    for (ix, iy, iz) in [(1, 2, 3), (81, 0, 0), (0, 81, 0), (7005, 7006, 6999), (123456, 7, 99999)]:
        want = (ix ^ ((iy * P2) & 0xFFFFFFFF) ^ ((iz * P3) & 0xFFFFFFFF)) % (1 << 19)
        assert orc.hash_index(lay, 15, ix, iy, iz) == want
    assert orc.hash_index(lay, 4, 1, 0, 0) == 1 and orc.hash_index(lay, 4, 0, 1, 0) == P2 % (1 << 19)


def _small(**kw):
    base = dict(n_levels=3, n_features=2, log2_table=12, base_res=4, growth=2.0,
                box_min=(-1.0, -1.0, -1.0), box_max=(1.0, 1.0, 1.0), n_freq_dir=2, n_hidden=2, width=8)
    base.update(kw)
    return HashLayout(**base)


def test_partition_of_unity_and_constant_table(orc):
    lay = layout_hash_paper()
    n = orc.hash_table_entries(lay)
    table = np.full(2 * n, 0.375, np.float32)
    x = random_rays(500)[0] * 3.0
    f = orc.hash_encode(lay, table, x)
    assert np.allclose(f, 0.375, atol=1e-14)


def test_linear_field_is_reproduced_on_dense_levels(orc):
    """table[vertex] = a.v / N  =>  feature(x) = a.x01 exactly (trilinear interpolation reproduces
    linear functions): fails for a wrong corner weight, a swapped axis or a wrong stride."""
    lay = _small()                                      # N = 4, 8, 16: 5^3, 9^3 dense; 17^3 > 4096 hashed
    assert [orc.hash_level(lay, l)[3] for l in range(3)] == [False, False, True]
    n = orc.hash_table_entries(lay)
    table = np.zeros((n, 2), np.float32)
    a0, a1 = np.array([1.0, 2.0, 4.0]), np.array([-3.0, 0.5, 0.25])
    for l in range(2):
        N, ent, off, _ = orc.hash_level(lay, l)
        V = N + 1
        idx = np.arange(ent)
        v = np.stack([idx % V, (idx // V) % V, idx // (V * V)], axis=1) / N
        table[off:off + ent, 0] = v @ a0
        table[off:off + ent, 1] = v @ a1
    x = random_rays(400)[0]                              # inside the box [-1, 1]^3
    x01 = ((x - np.float32(-1.0)) / np.float32(2.0)).astype(np.float64)
    f = orc.hash_encode(lay, table.reshape(-1), x)
    for l in range(2):
        assert np.allclose(f[:, 2 * l], x01 @ a0, atol=1e-6)
        assert np.allclose(f[:, 2 * l + 1], x01 @ a1, atol=1e-6)


def test_vertex_values_clamping_and_continuity(orc):
    lay = _small()
    n = orc.hash_table_entries(lay)
    rng = np.random.default_rng(5)
    table = rng.uniform(-1, 1, (n, 2)).astype(np.float32)
    # a point on a vertex of level 0 (N = 4): x01 = (1, 2, 3)/4 -> x = 2 x01 - 1, exactly representable
    x = np.array([[-0.5, 0.0, 0.5]], np.float32)
    f = orc.hash_encode(lay, table.reshape(-1), x)
    N0, _, off0, _ = orc.hash_level(lay, 0)
    assert np.allclose(f[0, :2], table[off0 + 1 + 5 * (2 + 5 * 3)], atol=1e-15)
    # the far corner of the box is the last vertex; outside points clamp to the box (reading H2)
    far = np.array([[1.0, 1.0, 1.0], [7.0, 1.5, 2.0]], np.float32)
    g = orc.hash_encode(lay, table.reshape(-1), far)
    assert np.allclose(g[0, :2], table[off0 + 5 ** 3 - 1], atol=1e-15) and np.array_equal(g[0], g[1])
    # hashed level 2 at a vertex: x01 = (3, 5, 9)/16
    xv = (2.0 * np.array([[3, 5, 9]]) / 16 - 1.0).astype(np.float32)
    N2, _, off2, hashed = orc.hash_level(lay, 2)
    assert hashed and N2 == 16
    want = (3 ^ ((5 * P2) & 0xFFFFFFFF) ^ ((9 * P3) & 0xFFFFFFFF)) % (1 << 12)
    assert np.allclose(orc.hash_encode(lay, table.reshape(-1), xv)[0, 4:6], table[off2 + want], atol=1e-15)
    # continuity across a cell face of every level (x01 = 0.5 is a face of all three)
    eps = np.float32(2.0 ** -20)
    a = np.array([[0.0 - eps, 0.3, -0.7]], np.float32); b = np.array([[0.0 + eps, 0.3, -0.7]], np.float32)
    fa, fb = orc.hash_encode(lay, table.reshape(-1), a), orc.hash_encode(lay, table.reshape(-1), b)
    assert np.abs(fa - fb).max() < 1e-4


def _numpy_hash_forward(lay, table, mlp, o, d, orc):
    """Independent evaluator: vectorised over rays and corners, einsum for the MLP."""
    T = 1 << lay.log2_table
    tab = np.asarray(table, np.float64).reshape(-1, lay.n_features)
    bmin, bmax = np.array(lay.box_min, np.float32), np.array(lay.box_max, np.float32)
    x01 = np.clip((o.astype(np.float32) - bmin) / (bmax - bmin), np.float32(0), np.float32(1)).astype(np.float32)
    feats, off = [], 0
    for l in range(lay.n_levels):
        N = int(np.floor(lay.base_res * lay.growth ** l)); V = N + 1
        dense = V ** 3 <= T
        pos = (x01 * np.float32(N)).astype(np.float32)
        c0 = np.minimum(np.floor(pos), N - 1)
        w = (pos - c0.astype(np.float32)).astype(np.float64); c0 = c0.astype(np.int64)
        acc = np.zeros((o.shape[0], lay.n_features))
        for bz in (0, 1):
            for by in (0, 1):
                for bx in (0, 1):
                    ix, iy, iz = c0[:, 0] + bx, c0[:, 1] + by, c0[:, 2] + bz
                    idx = ix + V * (iy + V * iz) if dense else ((ix ^ ((iy * P2) & 0xFFFFFFFF) ^ ((iz * P3) & 0xFFFFFFFF)) % T)
                    wt = np.where(bx, w[:, 0], 1 - w[:, 0]) * np.where(by, w[:, 1], 1 - w[:, 1]) * np.where(bz, w[:, 2], 1 - w[:, 2])
                    acc += wt[:, None] * tab[off + idx]
        feats.append(acc); off += V ** 3 if dense else T
    dd = d.astype(np.float64)
    g = [dd] + [fn(np.pi * dd * 2.0 ** k) for k in range(lay.n_freq_dir) for fn in (np.sin, np.cos)]
    h = np.concatenate(feats + g, axis=1)
    m = np.asarray(mlp, np.float64); p = 0
    shapes = hash_mlp_shapes(lay)
    for li, (no, ni) in enumerate(shapes):
        W = m[p:p + no * ni].reshape(no, ni); p += no * ni
        b = m[p:p + no]; p += no
        h = np.einsum("nk,jk->nj", h, W) + b
        if li < len(shapes) - 1:
            h = np.maximum(h, 0.0)
    return h


@pytest.mark.parametrize("kw", [dict(), dict(n_levels=5, growth=1.5, base_res=3, log2_table=8, n_freq_dir=0, n_hidden=1),
                                dict(n_features=4, n_hidden=3, width=5, box_min=(-2.0, -1.0, 0.0), box_max=(1.0, 3.0, 0.5))])
def test_brute_force_small_fields(orc, kw):
    lay = _small(**kw)
    n = orc.hash_table_entries(lay)
    table = make_hash_table(lay, n)
    mlp = make_hash_mlp(lay, bias_scale=0.3)
    o, d = random_rays(300)
    o = o * 1.5                                          # some origins outside the box: clamped
    z, t, xi = orc.hash_forward(lay, table, mlp, o, d)
    zr = _numpy_hash_forward(lay, table, mlp, o, d, orc)
    assert np.abs(z - zr).max() < 1e-10
    assert np.allclose(t, np.maximum(zr[:, 0], 0) + np.log1p(np.exp(-np.abs(zr[:, 0]))), atol=1e-12)
    assert np.allclose(xi, 1 / (1 + np.exp(-zr[:, 1])), atol=1e-12)


def test_brute_force_paper_field_and_fp16_table(orc):
    for td in (0, 2):
        lay = HashLayout(table_dtype=td)
        n = orc.hash_table_entries(lay)
        table = make_hash_table(lay, n)
        mlp = make_hash_mlp(lay)
        o, d = random_rays(200)
        o = o * 2.9
        z, _, _ = orc.hash_forward(lay, table, mlp, o, d)
        tab = table if td == 0 else table.view(np.float16).astype(np.float32)
        zr = _numpy_hash_forward(lay, tab, mlp, o, d, orc)
        assert np.abs(z - zr).max() < 1e-10
        assert 0.05 < np.abs(z).mean() < 10.0            # logits are O(1): the classification test is not vacuous


def test_zero_mlp_gives_head_of_bias_and_quantised_mode(orc):
    lay = _small()
    n = orc.hash_table_entries(lay)
    table = make_hash_table(lay, n)
    mlp = np.zeros(orc.hash_mlp_params(lay), np.float32)
    mlp[-2:] = [2.0, -1.0]
    o, d = random_rays(50)
    z, t, xi = orc.hash_forward(lay, table, mlp, o, d)
    assert np.allclose(t, 2.1269280110429727, atol=1e-15) and np.allclose(xi, 0.2689414213699951, atol=1e-15)
    # quantised mode = exact mode on inputs/weights that are already bf16 and a 1-layer net whose
    # only rounding point is the (bf16-exact) input: identity-like check of where rounding happens
    lay1 = _small(n_hidden=1, width=4, n_freq_dir=0)
    mlp1 = bf16_bits_to_f32(f32_to_bf16_bits(make_hash_mlp(lay1, bias_scale=0.2)))
    tab1 = np.full(2 * orc.hash_table_entries(lay1), 0.5, np.float32)          # features = 0.5: bf16-exact
    d1 = np.tile(np.array([[0.0, 0.0, 1.0]], np.float32), (50, 1))             # gamma(d) bf16-exact
    z0, _, _ = orc.hash_forward(lay1, tab1, mlp1, o, d1, mode=0)
    z1, _, _ = orc.hash_forward(lay1, tab1, mlp1, o, d1, mode=1)
    assert np.array_equal(z0, z1)
    # and it does round otherwise
    zq, _, _ = orc.hash_forward(lay, table, make_hash_mlp(lay), o, d, mode=1)
    ze, _, _ = orc.hash_forward(lay, table, make_hash_mlp(lay), o, d, mode=0)
    assert 0 < np.abs(zq - ze).max() < 5e-2
