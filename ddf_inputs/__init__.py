"""Seeded synthetic inputs shared by the oracle tests and the CUDA path.

This module holds NO arithmetic of the method (no encoding, no MLP, no heads, no ray
generators of SURVEY.md rows a9-a11): it only draws the random numbers that both sides
receive as plain arrays - network weights and the `configs[0]` style random ray batch -
and describes the benchmark layouts of BASELINE.json.  Neither `oracle/` nor
`paper_2606_00817_b200/` imports the other; both may be fed from here.

Random numbers (reading A8): a counter-based SplitMix64-style mixer keyed by
(seed, stream, index); u = (top 24 bits) * 2^-24 in [0, 1).
"""
from .rng import mix64, u64_at, uniform01, MASTER_SEED, STREAMS
from .layouts import (Layout, layout_c0, layout_c1, layout_sdf, blob_layer_shapes, blob_num_elements,
                      HashLayout, layout_hash_paper, hash_mlp_shapes)
from .weights import make_weights, f32_to_bf16_bits, bf16_bits_to_f32, make_hash_table, make_hash_mlp, f32_to_f16_bits
from .rays import random_rays

__all__ = [
    "mix64", "u64_at", "uniform01", "MASTER_SEED", "STREAMS",
    "Layout", "layout_c0", "layout_c1", "layout_sdf", "blob_layer_shapes", "blob_num_elements",
    "make_weights", "f32_to_bf16_bits", "bf16_bits_to_f32", "random_rays",
    "HashLayout", "layout_hash_paper", "hash_mlp_shapes", "make_hash_table", "make_hash_mlp", "f32_to_f16_bits",
]
