"""Counter-based random numbers for the synthetic inputs.

`u64(seed, counter)` is the splitmix64 finaliser applied to `seed * GOLDEN + counter`;
everything else (uniform doubles, normals, Poisson) is derived from it, so a stream
is a pure function of (seed, counter) and is the same scalar or vectorised, on any
numpy version.  This is input generation only; it is not part of the method.
"""
from __future__ import annotations

import math

import numpy as np

_M64 = (1 << 64) - 1
_GOLDEN = 0x9E3779B97F4A7C15


def u64(seed: int, counter: int) -> int:
    z = (seed * _GOLDEN + (counter + 1) * 0xD1342543DE82EF95) & _M64
    z = ((z ^ (z >> 30)) * 0xBF58476D1CE4E5B9) & _M64
    z = ((z ^ (z >> 27)) * 0x94D049BB133111EB) & _M64
    return z ^ (z >> 31)


def u64_array(seed, counter) -> np.ndarray:
    """Vectorised `u64`; `seed` and `counter` broadcast (uint64 wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        s = np.asarray(seed, dtype=np.uint64)
        c = np.asarray(counter, dtype=np.uint64)
        z = s * np.uint64(_GOLDEN) + (c + np.uint64(1)) * np.uint64(0xD1342543DE82EF95)
        z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
        z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
        return z ^ (z >> np.uint64(31))


def uniform_array(seed, counter) -> np.ndarray:
    """Doubles in [0,1) with 53 random bits."""
    return (u64_array(seed, counter) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))


class Stream:
    """Sequential view of the counter-based generator (one per seed)."""

    def __init__(self, seed: int):
        self.seed = int(seed)
        self.counter = 0

    def next_u64(self) -> int:
        v = u64(self.seed, self.counter)
        self.counter += 1
        return v

    def uniform(self) -> float:
        return (self.next_u64() >> 11) * (1.0 / (1 << 53))

    def uniforms(self, n: int) -> np.ndarray:
        c = np.arange(self.counter, self.counter + n, dtype=np.uint64)
        self.counter += n
        return uniform_array(np.uint64(self.seed), c)

    def integer(self, n: int) -> int:
        """Uniform integer in [0, n)."""
        return min(int(self.uniform() * n), n - 1)

    def normal(self) -> float:
        u1 = 1.0 - self.uniform()
        u2 = self.uniform()
        return math.sqrt(-2.0 * math.log(u1)) * math.cos(2.0 * math.pi * u2)

    def poisson(self, mean: float) -> int:
        """Poisson variate by inversion (sequential search from 0); fine for mean <= a few hundred."""
        u = self.uniform()
        p = math.exp(-mean)
        k = 0
        cdf = p
        while u > cdf and k < 10000:
            k += 1
            p *= mean / k
            cdf += p
        return k
