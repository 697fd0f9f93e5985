"""Stateless counter-based generator: u = hash64(seed, stream, index)."""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)


def _mix(z):
    # splitmix64 finaliser on uint64 arrays (wrap-around arithmetic is intended)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        z = z ^ (z >> np.uint64(31))
    return z


def hash64(seed, stream, index):
    """64-bit hash of (seed, stream, index); `index` may be an integer array."""
    idx = np.asarray(index, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = _mix(np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + np.uint64(0x9E3779B97F4A7C15))
        z = _mix(z ^ (np.uint64(stream) * np.uint64(0xD1B54A32D192ED03)))
        z = _mix(z + idx * np.uint64(0x9E3779B97F4A7C15))
    return z


def uniform01(seed, stream, index):
    """Uniform doubles in [0, 1) with 53 random bits."""
    return (hash64(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def random_unit_vectors(seed, n, stream=0):
    """n vectors uniform on the unit sphere: z = 2u1-1, phi = 2 pi u2; fp64 -> fp32 once.

    Returns a float32 array of shape (3, n) (SoA, component first).
    """
    i = np.arange(n, dtype=np.uint64)
    z = 2.0 * uniform01(seed, 2 * stream, i) - 1.0
    phi = 2.0 * np.pi * uniform01(seed, 2 * stream + 1, i)
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    return np.stack([s * np.cos(phi), s * np.sin(phi), z]).astype(np.float32)
