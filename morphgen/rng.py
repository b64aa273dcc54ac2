"""Counter-based random numbers for the synthetic inputs.

``value = mix(seed, stream, index)``: a SplitMix64-style finaliser applied to a
64-bit counter, so that any element can be generated in any order (CPU oracle,
Python harness, tests) and always gets the same value.  This module holds no
arithmetic of the Hines method; it only draws numbers.

Recipe (recorded in DESIGN.md, "Synthetic inputs"):

    z  = seed + stream * 0xD1B54A32D192ED03 + index * 0x9E3779B97F4A7C15   (mod 2^64)
    z  = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9
    z  = (z ^ (z >> 27)) * 0x94D049BB133111EB
    z  =  z ^ (z >> 31)
    u  = (z >> 11) * 2^-53           in [0, 1)
"""
from __future__ import annotations

import numpy as np

BASE_SEED = 181012742  # arXiv 1810.12742

# streams
STREAM_TOPOLOGY = 1
STREAM_LENGTH = 2
STREAM_A = 3
STREAM_SIGMA = 4
STREAM_B = 5
STREAM_CLASS = 6

_MASK = (1 << 64) - 1
_G = 0x9E3779B97F4A7C15
_S = 0xD1B54A32D192ED03
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def hash64(seed: int, stream: int, index) -> np.ndarray:
    """64-bit hash of (seed, stream, index[]); index is any integer array."""
    z = np.array(index, dtype=np.uint64, copy=True)
    base = np.uint64((int(seed) + int(stream) * _S) & _MASK)
    with np.errstate(over="ignore"):
        z *= np.uint64(_G)
        z += base
        z ^= z >> np.uint64(30)
        z *= _M1
        z ^= z >> np.uint64(27)
        z *= _M2
        z ^= z >> np.uint64(31)
    return z


def uniform01(seed: int, stream: int, index) -> np.ndarray:
    """float64 uniform in [0, 1) from the top 53 bits of hash64."""
    z = hash64(seed, stream, index)
    z >>= np.uint64(11)
    return z.astype(np.float64) * (1.0 / 9007199254740992.0)


def uniform(seed: int, stream: int, index, lo: float, hi: float) -> np.ndarray:
    r = uniform01(seed, stream, index)
    r *= (hi - lo)
    r += lo
    return r


def hash64_scalar(seed: int, stream: int, index: int) -> int:
    """Pure-Python twin of hash64 for one index (used by tests of this module)."""
    z = (int(seed) + int(stream) * _S + int(index) * _G) & _MASK
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _MASK
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _MASK
    return z ^ (z >> 31)
