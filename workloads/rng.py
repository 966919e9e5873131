"""Counter-based SplitMix64 stream: seeds mean the same thing on every box.

Input generation only (SURVEY.md §8(d) "Synthetic inputs"): this module holds none of the
method's arithmetic.  Element i of the stream with seed s is mix(s + (i+1)*GAMMA) — the
published SplitMix64 output function applied to a Weyl sequence — so any slice can be drawn
independently.
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def u64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n raw 64-bit outputs, stream positions offset .. offset+n-1."""
    with np.errstate(over="ignore"):
        i = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + i * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n doubles in [0,1): top 53 bits of each output times 2^-53."""
    return (u64(seed, n, offset) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform(seed: int, n: int, lo: float, hi: float, offset: int = 0) -> np.ndarray:
    return lo + (hi - lo) * uniform01(seed, n, offset)


def normal(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """n standard normals by Box-Muller; normal k uses stream positions offset+2k, offset+2k+1."""
    u = uniform01(seed, 2 * n, offset)
    u1 = 1.0 - u[0::2]            # (0,1]
    u2 = u[1::2]
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
