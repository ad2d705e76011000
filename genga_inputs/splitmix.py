"""SplitMix64 as a counter-based generator (no dependence on numpy's RNG versions).

Output k (k = 0, 1, ...) of the stream with seed ``s`` is ``mix(s + (k + 1) * GAMMA)`` with
Steele/Lea/Flood's constants, so any slice of the stream can be produced independently and
vectorised.  Uniforms are the top 53 bits scaled to [0, 1).
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(seed: int, start: int, count: int) -> np.ndarray:
    """uint64 outputs ``start .. start+count-1`` of the SplitMix64 stream seeded with ``seed``."""
    with np.errstate(over="ignore"):
        k = np.arange(start + 1, start + 1 + count, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniforms(seed: int, start: int, count: int) -> np.ndarray:
    """float64 uniforms in [0, 1) from the top 53 bits of each SplitMix64 output."""
    z = splitmix64(seed, start, count)
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
