"""Network layouts of BASELINE.json's configs (field names follow include/ddf.h `ddf_layout`).

Weight blob (SURVEY.md 8(b) conventions): layers 0..n_hidden-1 then the head; each layer is
W[out][in] row-major followed by b[out]; `in` of layer 0 is E = (3+6*L_o) + (3+6*L_d)
(input_kind 0: ray) or E = 3+6*L_o (input_kind 1: point); `in` of the skip layer is
width+E ordered [h ; gamma].
"""
from dataclasses import dataclass


@dataclass(frozen=True)
class Layout:
    input_kind: int = 0        # 0 = ray (origin+direction), 1 = point (SDF)
    n_freq_origin: int = 10
    n_freq_dir: int = 4
    n_hidden: int = 8
    width: int = 1280
    skip_layer: int = 4        # 0-based; -1 = none
    n_out: int = 2
    weight_dtype: int = 1      # 0 = fp32, 1 = bf16 (raw uint16)

    @property
    def enc_dim(self):
        e = 3 + 6 * self.n_freq_origin
        if self.input_kind == 0:
            e += 3 + 6 * self.n_freq_dir
        return e


def layout_c0():
    """configs[0]: 54-dim input, 3 hidden layers of width 64, fp32 weights."""
    return Layout(0, 4, 4, 3, 64, -1, 2, 0)


def layout_c1():
    """configs[1] (reading A4-A): 90-dim input, 8 x 1280, skip into layer 4, bf16 weights."""
    return Layout(0, 10, 4, 8, 1280, 4, 2, 1)


def layout_sdf():
    """configs[4] sphere-tracing network (A18): point input, L=10, 8 x 1280, one linear output."""
    return Layout(1, 10, 0, 8, 1280, 4, 1, 1)


def blob_layer_shapes(lay):
    """[(out, in)] for every layer including the head, in blob order."""
    shapes = []
    e = lay.enc_dim
    fan_in = e
    for l in range(lay.n_hidden):
        if l == lay.skip_layer and l > 0:
            fan_in = lay.width + e
        shapes.append((lay.width, fan_in))
        fan_in = lay.width
    shapes.append((lay.n_out, fan_in))
    return shapes


def blob_num_elements(lay):
    return sum(o * i + o for o, i in blob_layer_shapes(lay))


@dataclass(frozen=True)
class HashLayout:
    """The paper's own field: multiresolution hash grid on the origin, L_d
    sinusoidal direction bands, a small ReLU MLP.  Field names follow `ddf_hashgrid_layout`."""
    n_levels: int = 16
    n_features: int = 2
    log2_table: int = 19
    base_res: int = 16
    growth: float = 1.5
    box_min: tuple = (-3.0, -3.0, -3.0)
    box_max: tuple = (3.0, 3.0, 3.0)
    n_freq_dir: int = 4
    n_hidden: int = 2
    width: int = 64
    n_out: int = 2
    table_dtype: int = 0       # 0 = fp32, 2 = fp16 (raw uint16)
    mlp_dtype: int = 0         # 0 = fp32, 1 = bf16 (raw uint16)

    @property
    def mlp_in(self):
        return self.n_levels * self.n_features + 3 + 6 * self.n_freq_dir


def layout_hash_paper():
    """16 levels x 2 features, T = 2^19, base 16, growth 1.5, 4 direction bands,
    2 x 64 MLP; fp32 table (the paper's 52 MB).  Box: DESIGN.md reading H7."""
    return HashLayout()


def hash_mlp_shapes(lay):
    shapes, fan_in = [], lay.mlp_in
    for _ in range(lay.n_hidden):
        shapes.append((lay.width, fan_in))
        fan_in = lay.width
    shapes.append((lay.n_out, fan_in))
    return shapes
