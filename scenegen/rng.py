"""Counter-based SplitMix64, vectorised with NumPy.

Output i of a stream depends only on (seed, stream, i), so draws can be made in
bulk (tens of millions of weights) and still be reproduced one at a time.
Uniform floats use the top 24 bits: u = (z >> 40) * 2^-24, exact in float32.
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


class SplitMix64:
    """One independent stream per (seed, stream) pair; `counter` advances per draw."""

    def __init__(self, seed: int, stream: int = 0):
        with np.errstate(over="ignore"):
            s = _mix(np.uint64(seed) * np.uint64(1000003) + np.uint64(stream) + _GAMMA)
        self.base = np.uint64(s)
        self.counter = 0

    def bits(self, m: int) -> np.ndarray:
        """Next m 64-bit outputs."""
        idx = np.arange(self.counter + 1, self.counter + 1 + m, dtype=np.uint64)
        self.counter += m
        with np.errstate(over="ignore"):
            return _mix(self.base + idx * _GAMMA)

    def uniform(self, m: int) -> np.ndarray:
        """m float64 values in [0,1) carrying 24 random bits each."""
        return (self.bits(m) >> np.uint64(40)).astype(np.float64) * (1.0 / 16777216.0)

    def uniform1(self) -> float:
        return float(self.uniform(1)[0])

    def randint(self, lo: int, hi: int) -> int:
        """Integer in [lo, hi) (hi > lo), by scaling a 24-bit uniform."""
        return lo + int(self.uniform1() * (hi - lo))
