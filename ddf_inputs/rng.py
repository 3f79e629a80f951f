"""Counter-based random numbers (reading A8).

    mix64(z):  z += 0x9E3779B97F4A7C15
               z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9
               z = (z ^ (z >> 27)) * 0x94D049BB133111EB
               return z ^ (z >> 31)                      (all mod 2^64)
    u64_at(seed, stream, i) = mix64( mix64( mix64(seed) ^ stream ) ^ i )
    uniform01 = (u64 >> 40) * 2^-24                      (24 bits, exact in fp32)

The oracle (C) and the CUDA generators each re-implement these three lines themselves.
"""
import numpy as np

MASTER_SEED = 20260600817
STREAMS = {
    "weights_ddf": 1, "weights_sdf": 2, "rays_c0": 3, "camera_pos": 4,
    "shadow_points": 5, "ao_samples": 6, "biases": 7, "hash_table": 8, "hash_mlp": 9, "train_rays": 10,
}

_M1 = np.uint64(0x9E3779B97F4A7C15)
_M2 = np.uint64(0xBF58476D1CE4E5B9)
_M3 = np.uint64(0x94D049BB133111EB)


def mix64(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = z + _M1
        z = (z ^ (z >> np.uint64(30))) * _M2
        z = (z ^ (z >> np.uint64(27))) * _M3
        return z ^ (z >> np.uint64(31))


def u64_at(seed, stream, idx):
    key = mix64(mix64(np.uint64(seed)) ^ np.uint64(stream))
    return mix64(key ^ np.asarray(idx, dtype=np.uint64))


def uniform01(seed, stream, idx):
    """float64 array of exact 24-bit uniforms in [0,1)."""
    return (u64_at(seed, stream, idx) >> np.uint64(40)).astype(np.float64) * (2.0 ** -24)
