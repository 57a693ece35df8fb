"""Counter-based random numbers for the synthetic inputs (SURVEY.md §8(c) "G. Event generator").

Every draw is a pure function of (seed, named sub-stream, counter), so any
consumer can regenerate any input without replaying a sequence.  This module
holds no arithmetic of the tracking method itself: it only makes inputs.

mix64 is the SplitMix64 output function applied to key + counter * golden.
"""
from __future__ import annotations

import hashlib

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_TWO_M53 = 2.0 ** -53


def mix64(z: np.ndarray) -> np.ndarray:
    """SplitMix64 finaliser on a uint64 array (wrapping arithmetic)."""
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def stream_key(seed: int, name: str) -> np.uint64:
    """64-bit key of the sub-stream `name` of `seed` (first 8 bytes of SHA-256)."""
    h = hashlib.sha256(f"{int(seed)}:{name}".encode()).digest()
    return np.uint64(int.from_bytes(h[:8], "little"))


class Stream:
    """A named sub-stream: u64(ctr), uniform(ctr) in [0,1), normal(ctr) ~ N(0,1)."""

    def __init__(self, seed: int, name: str):
        self.key = stream_key(seed, name)

    def u64(self, ctr) -> np.ndarray:
        ctr = np.asarray(ctr, dtype=np.uint64)
        with np.errstate(over="ignore"):
            return mix64(self.key + (ctr + np.uint64(1)) * _GOLDEN)

    def uniform(self, ctr) -> np.ndarray:
        """Top 53 bits times 2^-53: uniform on [0, 1) in fp64."""
        return (self.u64(ctr) >> np.uint64(11)).astype(np.float64) * _TWO_M53

    def normal(self, ctr) -> np.ndarray:
        """Box-Muller from counters 2*ctr and 2*ctr+1."""
        ctr = np.asarray(ctr, dtype=np.uint64)
        u1 = 1.0 - self.uniform(ctr * np.uint64(2))          # (0, 1]
        u2 = self.uniform(ctr * np.uint64(2) + np.uint64(1))
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)
