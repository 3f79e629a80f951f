"""Seeded Kaiming-uniform weights (reading A7: U(+-sqrt(6/fan_in)) for every layer).

Element `i` of the blob (running index over the whole blob, weights and biases alike) draws
u = uniform01(seed, stream, i); weights are (2u-1)*bound rounded to fp32; biases are zero, or
(2u-1)*bias_scale when `bias_scale` > 0 (tests of the bias path).  For weight_dtype = 1 the
fp32 values are rounded to bf16 (round-to-nearest-even) and returned as raw uint16.
"""
import numpy as np

from .rng import uniform01, MASTER_SEED, STREAMS
from .layouts import blob_layer_shapes, hash_mlp_shapes


def f32_to_bf16_bits(x):
    """RNE rounding of finite fp32 values to bf16, returned as uint16 bit patterns."""
    b = np.ascontiguousarray(x, dtype=np.float32).view(np.uint32).astype(np.uint64)
    r = (b + np.uint64(0x7FFF) + ((b >> np.uint64(16)) & np.uint64(1))) >> np.uint64(16)
    return r.astype(np.uint16)


def bf16_bits_to_f32(bits):
    return (np.ascontiguousarray(bits, dtype=np.uint16).astype(np.uint32) << np.uint32(16)).view(np.float32)


def make_weights(lay, seed=MASTER_SEED, stream=None, bias_scale=0.0):
    """Returns the blob as a 1-D array: float32 (weight_dtype 0) or uint16 bf16 bits (1)."""
    if stream is None:
        stream = STREAMS["weights_sdf"] if lay.input_kind == 1 else STREAMS["weights_ddf"]
    parts = []
    off = 0
    for (o, i) in blob_layer_shapes(lay):
        bound = np.sqrt(6.0 / i)
        idx = np.arange(off, off + o * i, dtype=np.uint64)
        w = ((2.0 * uniform01(seed, stream, idx) - 1.0) * bound).astype(np.float32)
        off += o * i
        if bias_scale > 0.0:
            idx = np.arange(off, off + o, dtype=np.uint64)
            b = ((2.0 * uniform01(seed, stream, idx) - 1.0) * bias_scale).astype(np.float32)
        else:
            b = np.zeros(o, dtype=np.float32)
        off += o
        parts += [w, b]
    blob = np.concatenate(parts)
    if lay.weight_dtype == 1:
        return f32_to_bf16_bits(blob)
    return blob


def f32_to_f16_bits(x):
    return np.ascontiguousarray(x, dtype=np.float32).astype(np.float16).view(np.uint16)


def make_hash_table(lay, n_entries, seed=MASTER_SEED, stream=None, scale=1.0):
    """Seeded feature table: `n_entries` x n_features values U(-scale, scale) (stand-ins for trained
    features), fp32 or fp16 bits per lay.table_dtype.  The entry count is passed in by the caller
    (from the oracle in tests, from the library in bench.py): this module holds no grid arithmetic."""
    if stream is None:
        stream = STREAMS["hash_table"]
    idx = np.arange(int(n_entries) * lay.n_features, dtype=np.uint64)
    t = ((2.0 * uniform01(seed, stream, idx) - 1.0) * scale).astype(np.float32)
    return f32_to_f16_bits(t) if lay.table_dtype == 2 else t


def make_hash_mlp(lay, seed=MASTER_SEED, stream=None, bias_scale=0.0):
    """MLP blob of the hash-grid field: layers then head, W[out][in] row-major then b[out];
    U(+-sqrt(6/fan_in)) weights (reading A7), zero or seeded biases."""
    if stream is None:
        stream = STREAMS["hash_mlp"]
    parts, off = [], 0
    for (o, i) in hash_mlp_shapes(lay):
        bound = np.sqrt(6.0 / i)
        w = ((2.0 * uniform01(seed, stream, np.arange(off, off + o * i, dtype=np.uint64)) - 1.0) * bound).astype(np.float32)
        off += o * i
        if bias_scale > 0.0:
            b = ((2.0 * uniform01(seed, stream, np.arange(off, off + o, dtype=np.uint64)) - 1.0) * bias_scale).astype(np.float32)
        else:
            b = np.zeros(o, dtype=np.float32)
        off += o
        parts += [w, b]
    blob = np.concatenate(parts)
    return f32_to_bf16_bits(blob) if lay.mlp_dtype == 1 else blob
