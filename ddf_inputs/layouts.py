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
