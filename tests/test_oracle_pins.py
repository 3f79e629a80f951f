"""Pins for the CPU oracle: closed forms, worked examples, brute force.

None of these re-types the oracle's formula in the same shape: values come from
tests/golden/ (cited there), from closed forms, or from an independent numpy evaluator with a
different loop structure (matrix products on whole batches, float64).
"""
import math
import os

import numpy as np
import pytest

from ddf_inputs import Layout, layout_c0, blob_layer_shapes, blob_num_elements, make_weights, random_rays
from ddf_inputs import bf16_bits_to_f32, f32_to_bf16_bits

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _blob_from_layers(lay, layers):
    """layers: list of (W[out][in], b[out]) -> fp32 blob."""
    parts = []
    for (W, b), (o, i) in zip(layers, blob_layer_shapes(lay)):
        W = np.asarray(W, dtype=np.float64)
        assert W.shape == (o, i), (W.shape, (o, i))
        parts += [W.reshape(-1), np.asarray(b, dtype=np.float64).reshape(o)]
    return np.concatenate(parts).astype(np.float32)


def _numpy_gamma(lay, o, d):
    """Independent encoder: vectorised over rays, np.sin/np.cos of (2^k * pi * x)."""
    def enc(v, L):
        cols = [v]
        for k in range(L):
            cols += [np.sin((2.0 ** k) * np.pi * v), np.cos((2.0 ** k) * np.pi * v)]
        return np.concatenate(cols, axis=1)
    g = enc(o.astype(np.float64), lay.n_freq_origin)
    if lay.input_kind == 0:
        g = np.concatenate([g, enc(d.astype(np.float64), lay.n_freq_dir)], axis=1)
    return g


def _numpy_forward(lay, blob, o, d):
    """Brute-force fp64 evaluator (P6): batch matrix products, no per-ray loop."""
    blob = np.asarray(blob)
    w = bf16_bits_to_f32(blob).astype(np.float64) if lay.weight_dtype == 1 else blob.astype(np.float64)
    g = _numpy_gamma(lay, o, d)
    h = g
    off = 0
    shapes = blob_layer_shapes(lay)
    for l, (no, ni) in enumerate(shapes[:-1]):
        W = w[off:off + no * ni].reshape(no, ni); off += no * ni
        b = w[off:off + no]; off += no
        x = np.concatenate([h, g], axis=1) if l == lay.skip_layer else h
        h = np.maximum(x @ W.T + b, 0.0)
    no, ni = shapes[-1]
    W = w[off:off + no * ni].reshape(no, ni); off += no * ni
    b = w[off:off + no]
    return h @ W.T + b


# ------------------------------------------------------------------ P1 / P2: heads

def test_head_golden_values(orc):
    for line in open(os.path.join(GOLD, "head_values.txt")):
        if line.startswith("#") or not line.strip():
            continue
        name, arg, val = line.split()
        got = getattr(orc, name)(float(arg))
        assert got == pytest.approx(float(val), rel=1e-13, abs=1e-300), (name, arg)


def test_head_identities(orc):
    for z in [-40.0, -3.5, -1e-3, 0.0, 0.7, 12.0, 55.0]:
        assert orc.softplus(z) - orc.softplus(-z) == pytest.approx(z, abs=1e-13)
        assert orc.sigmoid(z) + orc.sigmoid(-z) == pytest.approx(1.0, abs=1e-15)
    assert orc.softplus(800.0) == 800.0 and orc.softplus(-800.0) == 0.0     # no overflow
    assert orc.sigmoid(-800.0) == 0.0 and orc.sigmoid(800.0) == 1.0


def test_zero_weights_give_head_of_bias(orc):
    """P1: all W = 0 => t = softplus(b_out[0]), xi = sigmoid(b_out[1]) for every ray."""
    lay = layout_c0()
    o, d = random_rays(64)
    blob = np.zeros(blob_num_elements(lay), np.float32)
    z, t, xi = orc.forward(lay, blob, o, d)
    assert np.all(t == math.log(2.0)) and np.all(xi == 0.5)
    blob[-2:] = [1.25, -0.5]
    z, t, xi = orc.forward(lay, blob, o, d)
    assert np.allclose(t, 1.25 + math.log1p(math.exp(-1.25)), rtol=1e-15)
    assert np.allclose(xi, 1.0 / (1.0 + math.exp(0.5)), rtol=1e-15)


# ------------------------------------------------------------------ P3: encoding

def test_encoding_worked_example(orc):
    want = np.loadtxt(os.path.join(GOLD, "encoding_example.txt")).reshape(-1)
    lay = Layout(0, 2, 2, 1, 2, -1, 2, 0)
    g = orc.encode(lay, [[0.25, 0.0, -0.5]], [[0.0, 0.0, 1.0]])[0]
    assert g.shape == (30,)
    assert np.allclose(g, want, atol=1e-15)
    assert g.sum() == pytest.approx(7.164213562373095, abs=1e-14)


def test_encoding_norm_invariant_and_definition(orc):
    """|gamma(v)|^2 = |v|^2 + 3L; and gamma matches sin/cos(2^k pi x) from an independent encoder."""
    lay = Layout(0, 10, 4, 1, 2, -1, 2, 0)
    o, d = random_rays(257)
    o = (o * 2.5).astype(np.float32)
    g = orc.encode(lay, o, d)
    assert g.shape == (257, 90)
    n2 = (g[:, :63] ** 2).sum(1)
    assert np.allclose(n2, (o.astype(np.float64) ** 2).sum(1) + 30.0, atol=1e-9)
    assert np.allclose((g[:, 63:] ** 2).sum(1), 1.0 + 12.0, atol=1e-6)   # |d| = 1 up to fp32
    # high bands lose ~2^k ulp in the naive product 2^k*pi*x; the oracle scales exactly first
    assert np.allclose(g, _numpy_gamma(lay, o, d), atol=2e-12)


def test_encoding_point_kind(orc):
    lay = Layout(1, 10, 0, 1, 2, -1, 1, 0)
    assert orc.enc_dim(lay) == 63
    assert orc.enc_dim(layout_c0()) == 54


# ------------------------------------------------------------------ P4 / P5 / P7: wiring

def test_all_ones_network(orc):
    """P4: the P3 ray through one all-ones hidden layer of width 2."""
    lay = Layout(0, 2, 2, 1, 2, -1, 2, 0)
    blob = _blob_from_layers(lay, [(np.ones((2, 30)), [0, 0]), ([[0.5, 0.5], [-0.25, -0.25]], [0, 1])])
    z, t, xi = orc.forward(lay, blob, [[0.25, 0.0, -0.5]], [[0.0, 0.0, 1.0]])
    assert z[0, 0] == pytest.approx(7.164213562373095, abs=1e-14)
    assert z[0, 1] == pytest.approx(-2.5821067811865475, abs=1e-14)
    assert t[0] == pytest.approx(7.164987050427735, rel=1e-14)
    assert xi[0] == pytest.approx(0.07029891333177019, rel=1e-13)


def test_hand_example_no_trig(orc):
    """P7: L = 0, o=(1,2,3), d=(0,0,1) => h=(1,0), z=(2,-1)."""
    lay = Layout(0, 0, 0, 1, 2, -1, 2, 0)
    blob = _blob_from_layers(lay, [([[1, 0, 0, 0, 0, 0], [0, -1, 0, 0, 0, 1]], [0, 0]),
                                   ([[2, 5], [-1, 3]], [0, 0])])
    z, t, xi = orc.forward(lay, blob, [[1.0, 2.0, 3.0]], [[0.0, 0.0, 1.0]])
    assert z[0].tolist() == [2.0, -1.0]
    assert t[0] == pytest.approx(2.1269280110429727, rel=1e-15)
    assert xi[0] == pytest.approx(0.2689414213699951, rel=1e-15)


def _selector_layers(E, n_hidden, skip_layer, c0, c1, through_skip):
    """P5: width 2E; one layer computes (ReLU(g), ReLU(-g)), the others are identities; the
    head takes c*(h+ - h-) so z = c . gamma exactly."""
    W = 2 * E
    sel = np.concatenate([np.eye(E), -np.eye(E)], axis=0)            # [2E][E]
    layers = []
    for l in range(n_hidden):
        nin = E if l == 0 else W
        if l == skip_layer:
            nin = W + E
        Wl = np.zeros((W, nin))
        if through_skip:
            if l == skip_layer:
                Wl[:, W:] = sel              # h-part zero: output depends on the ray only via the skip
            elif l > skip_layer:
                Wl[:, :W] = np.eye(W)
            # layers before the skip: zero weights (their output is discarded)
        else:
            if l == 0:
                Wl[:, :E] = sel
            else:
                Wl[:, :W] = np.eye(W)        # gamma-part of the skip layer stays zero
        layers.append((Wl, np.zeros(W)))
    head = np.stack([np.concatenate([c0, -c0]), np.concatenate([c1, -c1])])
    layers.append((head, np.zeros(2)))
    return layers


@pytest.mark.parametrize("through_skip", [False, True])
def test_identity_layers_pass_encoding_through(orc, through_skip):
    lay = Layout(0, 2, 1, 4, 2 * 24, 2, 2, 0)
    E = 24
    rng = np.random.default_rng(5)
    c0, c1 = rng.standard_normal(E), rng.standard_normal(E)
    # keep the coefficients fp32-exact so that the fp32 blob stores them exactly
    c0, c1 = c0.astype(np.float32).astype(np.float64), c1.astype(np.float32).astype(np.float64)
    blob = _blob_from_layers(lay, _selector_layers(E, 4, 2, c0, c1, through_skip))
    o, d = random_rays(33)
    z, t, xi = orc.forward(lay, blob, o, d)
    g = _numpy_gamma(lay, o, d)
    assert np.allclose(z[:, 0], g @ c0, atol=1e-12)
    assert np.allclose(z[:, 1], g @ c1, atol=1e-12)
    assert np.allclose(t, np.logaddexp(0.0, g @ c0), atol=1e-12)


def test_skip_order_is_h_then_gamma(orc):
    """A transposed concat ([gamma ; h]) would read the wrong columns: weight only column `width`
    (= gamma[0] = o_x) of the skip layer."""
    lay = Layout(0, 1, 0, 2, 4, 1, 2, 0)
    E = 12
    W0 = np.zeros((4, E)); W1 = np.zeros((4, 4 + E)); W1[0, 4] = 1.0
    blob = _blob_from_layers(lay, [(W0, np.ones(4)), (W1, np.zeros(4)), ([[1, 0, 0, 0], [0, 0, 0, 0]], [0, 0])])
    z, _, _ = orc.forward(lay, blob, [[0.75, -0.5, 0.25]], [[0.0, 0.0, 1.0]])
    assert z[0, 0] == 0.75


# ------------------------------------------------------------------ P6: brute force

@pytest.mark.parametrize("cfg", [
    Layout(0, 2, 1, 1, 4, -1, 2, 0), Layout(0, 3, 2, 3, 8, -1, 2, 0), Layout(0, 3, 2, 3, 8, 1, 2, 0),
    Layout(0, 4, 4, 4, 6, 3, 2, 1), Layout(1, 5, 0, 3, 7, 2, 1, 0), Layout(1, 10, 0, 2, 5, -1, 1, 1),
])
def test_brute_force_tiny_networks(orc, cfg):
    blob = make_weights(cfg, seed=99, bias_scale=0.3)
    o, d = random_rays(41, seed=7)
    z, t, xi = orc.forward(cfg, blob, o, d if cfg.input_kind == 0 else None)
    zr = _numpy_forward(cfg, blob, o, d)
    assert np.allclose(z, zr, atol=1e-11, rtol=1e-11)
    assert np.allclose(t, np.logaddexp(0.0, zr[:, 0]), rtol=1e-12)
    if cfg.n_out == 2:
        assert np.allclose(xi, 1.0 / (1.0 + np.exp(-zr[:, 1])), rtol=1e-12)


def test_brute_force_config0(orc):
    lay = layout_c0()
    blob = make_weights(lay)
    assert blob.dtype == np.float32 and blob.size == 11776 + 64 * 3 + 2
    o, d = random_rays(4096)
    z, t, xi = orc.forward(lay, blob, o, d)
    assert np.allclose(z, _numpy_forward(lay, blob, o, d), atol=1e-11)
    # sanity of reading A7: logits are O(1), not collapsed to 0
    assert 0.3 < z.std() < 3.0


# ------------------------------------------------------------------ P8: invariances, quantised mode

def test_permutation_and_scaling_invariance(orc):
    lay = Layout(0, 3, 2, 3, 16, 1, 2, 1)
    blob = make_weights(lay, seed=3)
    o, d = random_rays(50, seed=11)
    z, _, _ = orc.forward(lay, blob, o, d)
    perm = np.random.default_rng(0).permutation(50)
    zp, _, _ = orc.forward(lay, blob, o[perm], d[perm])
    assert np.array_equal(zp, z[perm])
    for mode in (0, 1):
        # (iv) zero biases: scaling the head weights by 2^3 scales the logits exactly
        w = bf16_bits_to_f32(blob).copy()
        no, ni = blob_layer_shapes(lay)[-1]
        w[-(no * ni + no):] *= 8.0
        z1, _, _ = orc.forward(lay, blob, o, d, mode=mode)
        z8, _, _ = orc.forward(lay, f32_to_bf16_bits(w), o, d, mode=mode)
        assert np.array_equal(z8, 8.0 * z1)


def test_quantised_mode_rounds_where_stated(orc):
    """Reading A11: gamma and hidden activations to bf16, the last hidden layer not."""
    assert orc.round_bf16(1.0 + 2.0 ** -8) == 1.0                  # tie -> even
    assert orc.round_bf16(1.0 + 3 * 2.0 ** -8) == 1.0 + 2.0 ** -6  # tie -> even (up)
    assert orc.round_bf16(0.1) == float(bf16_bits_to_f32(f32_to_bf16_bits(np.array([0.1], np.float32)))[0])
    lay = Layout(0, 0, 0, 2, 2, -1, 2, 0)
    x = 1.0 + 2.0 ** -10                                            # not a bf16 value
    blob = _blob_from_layers(lay, [(np.eye(2, 6), [0, 0]), (np.eye(2), [2.0 ** -12, 0]), (np.eye(2), [0, 0])])
    z0, _, _ = orc.forward(lay, blob, [[x, 0.5, 0]], [[0, 0, 1]], mode=0)
    z1, _, _ = orc.forward(lay, blob, [[x, 0.5, 0]], [[0, 0, 1]], mode=1)
    assert z0[0, 0] == float(np.float32(x)) + 2.0 ** -12
    assert z1[0, 0] == 1.0 + 2.0 ** -12        # gamma rounded, layer-0 output rounded, layer 1 kept
    # quantised and exact agree to bf16 accuracy on a real network
    lay = layout_c0()
    blob = make_weights(lay)
    o, d = random_rays(512)
    za, _, _ = orc.forward(lay, blob, o, d, mode=0)
    zb, _, _ = orc.forward(lay, blob, o, d, mode=1)
    err = np.abs(za - zb).max()
    assert 1e-5 < err < 5e-2
