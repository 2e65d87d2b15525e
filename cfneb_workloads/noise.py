"""Counter-based seeded Gaussian noise: SplitMix64 -> 53-bit uniforms -> Box-Muller.

Generated once by the harness and handed as arrays to both the oracle and the
CUDA path, so neither side draws random numbers.
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _splitmix64(seed, n):
    """First n outputs of SplitMix64 started at `seed` (vectorised over the counter)."""
    with np.errstate(over="ignore"):
        k = np.arange(1, n + 1, dtype=np.uint64)
        z = np.uint64(seed) + k * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def splitmix64_uniforms(seed, n):
    """n uniforms in (0,1): ((z >> 11) + 0.5) * 2^-53."""
    z = _splitmix64(seed, n)
    return ((z >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def splitmix64_normals(seed, n):
    """n standard normals: Box-Muller cosine branch on consecutive uniform pairs."""
    u = splitmix64_uniforms(seed, 2 * n)
    u1 = u[0::2]
    u2 = u[1::2]
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
