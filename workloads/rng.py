"""Counter-based random numbers for the synthetic inputs.

Every number is a pure function of (seed, stream, counter): the splitmix64
finaliser applied to ``seed_mix + (counter + 1) * GOLDEN``.  Nothing here is
part of the NNP method; the oracle and the CUDA path both *receive* the arrays
this module produces (they never draw numbers themselves).

No dependence on numpy's Generator algorithms, so the streams do not drift
between numpy versions.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_MASK64 = (1 << 64) - 1


def _mix_array(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> np.uint64(30)
    z *= _M1
    z ^= z >> np.uint64(27)
    z *= _M2
    z ^= z >> np.uint64(31)
    return z


def _mix_int(z: int) -> int:
    z &= _MASK64
    z ^= z >> 30
    z = (z * 0xBF58476D1CE4E5B9) & _MASK64
    z ^= z >> 27
    z = (z * 0x94D049BB133111EB) & _MASK64
    z ^= z >> 31
    return z


def stream_key(seed: int, *stream: int) -> int:
    """Derive a 64-bit key from a seed and any number of integer stream ids."""
    k = _mix_int(seed + 0x9E3779B97F4A7C15)
    for s in stream:
        k = _mix_int(k ^ _mix_int((int(s) + 1) * 0x9E3779B97F4A7C15))
    return k


def bits(key: int, counters: np.ndarray) -> np.ndarray:
    """64 random bits per counter value (uint64 in, uint64 out)."""
    c = np.asarray(counters, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (c + np.uint64(1)) * _GOLDEN + np.uint64(key)
        return _mix_array(z)


def uniform(key: int, counters: np.ndarray) -> np.ndarray:
    """Uniform doubles in [0, 1): top 53 bits * 2**-53."""
    return (bits(key, counters) >> np.uint64(11)).astype(np.float64) * (2.0 ** -53)


def normal(key: int, counters: np.ndarray) -> np.ndarray:
    """Standard normals by Box-Muller; counter c uses raw counters 2c and 2c+1."""
    c = np.asarray(counters, dtype=np.uint64)
    with np.errstate(over="ignore"):
        u1 = ((bits(key, c * np.uint64(2)) >> np.uint64(11)).astype(np.float64) + 1.0) * (2.0 ** -53)
        u2 = uniform(key, c * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
