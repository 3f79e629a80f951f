"""configs[0]-style random ray batch: origins uniform in [-1,1)^3, directions uniform on S^2.

Ray i uses counters 5i..5i+4 of its stream: three for the origin, two (u1, u2) for the
direction with z = 2*u1-1, phi = 2*pi*u2, d = (sqrt(1-z^2) cos phi, sqrt(1-z^2) sin phi, z),
renormalised after the cast to fp32 (reading A9).  Generated once on the host;
the same arrays go to the oracle and to the GPU.
"""
import numpy as np

from .rng import uniform01, MASTER_SEED, STREAMS


def random_rays(n, seed=MASTER_SEED, stream=None, start=0):
    if stream is None:
        stream = STREAMS["rays_c0"]
    i = np.arange(start, start + n, dtype=np.uint64) * np.uint64(5)
    u = [uniform01(seed, stream, i + np.uint64(k)) for k in range(5)]
    o = np.stack([2.0 * u[0] - 1.0, 2.0 * u[1] - 1.0, 2.0 * u[2] - 1.0], axis=1).astype(np.float32)
    z = 2.0 * u[3] - 1.0
    phi = 2.0 * np.pi * u[4]
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    d = np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1).astype(np.float32)
    d /= np.linalg.norm(d.astype(np.float64), axis=1, keepdims=True).astype(np.float32)
    return np.ascontiguousarray(o), np.ascontiguousarray(d.astype(np.float32))
