"""Counter-based RNG: value = f(seed, stream, index) only.

splitmix64 finaliser applied to a mix of (seed, stream, index); uniform in
[0,1) from the top 53 bits; normals by Box-Muller on two decorrelated streams.
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)

# stream ids name the quantity they feed
STREAM = dict(affine=1, noise=2, field_dir=3, field_phase=4, field_k=5, alpha=6,
              ep_dir=7, void=8, mat=9, shuffle=10, sample=11, aux=12)


def _splitmix(z):
    z = (z + np.uint64(0x9E3779B97F4A7C15)) & _M64
    z = ((z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)) & _M64
    z = ((z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)) & _M64
    return z ^ (z >> np.uint64(31))


def bits(seed, stream, index):
    with np.errstate(over="ignore"):
        idx = np.asarray(index, dtype=np.uint64)
        s = _splitmix(np.uint64(seed) * np.uint64(0x100000001B3) + np.uint64(stream))
        return _splitmix(_splitmix(idx ^ s) + s)


def uniform(seed, stream, index):
    """U[0,1) for every entry of `index` (any integer array)."""
    return (bits(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed, stream, index):
    idx = np.asarray(index, dtype=np.uint64)
    u1 = uniform(seed, stream, idx * np.uint64(2))
    u2 = uniform(seed, stream, idx * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def permutation(seed, stream, n):
    """Seeded permutation of range(n): argsort of counter-based keys (ties by index)."""
    keys = bits(seed, stream, np.arange(n, dtype=np.uint64))
    return np.argsort(keys, kind="stable").astype(np.int64)
