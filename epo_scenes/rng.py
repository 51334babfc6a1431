"""Counter-based SplitMix64 streams for the synthetic-scene generator.

Vectorised with numpy uint64 wrap-around arithmetic so that drawing 10^8 normals (depth noise for
500 views) stays fast, and so that every draw is a pure function of (seed, counter): the arrays fed to
the CPU oracle and to the CUDA library are bit-identical on every machine.

This module holds no arithmetic of the EPO method (SURVEY.md §8(d) "Generator").
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


class SplitMix64:
    """SplitMix64 with an explicit counter; `fork(tag)` derives an independent stream."""

    def __init__(self, seed: int):
        self.seed = np.uint64(seed & 0xFFFFFFFFFFFFFFFF)
        self.counter = 0

    def fork(self, tag: int) -> "SplitMix64":
        with np.errstate(over="ignore"):
            s = _mix(np.array([self.seed + _GOLDEN * np.uint64(2 * tag + 1)], dtype=np.uint64))[0]
        return SplitMix64(int(s))

    def raw(self, n: int) -> np.ndarray:
        with np.errstate(over="ignore"):
            idx = np.arange(self.counter + 1, self.counter + n + 1, dtype=np.uint64)
            out = _mix(self.seed + idx * _GOLDEN)
        self.counter += n
        return out

    def uniform(self, n: int, lo: float = 0.0, hi: float = 1.0) -> np.ndarray:
        """Uniforms in [lo, hi) from the top 53 bits."""
        u = (self.raw(n) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
        return lo + (hi - lo) * u

    def normal(self, n: int) -> np.ndarray:
        """Standard normals by Box-Muller (both branches used)."""
        m = (n + 1) // 2
        u1 = 1.0 - self.uniform(m)          # (0, 1]
        u2 = self.uniform(m)
        r = np.sqrt(-2.0 * np.log(u1))
        z = np.concatenate([r * np.cos(2 * np.pi * u2), r * np.sin(2 * np.pi * u2)])
        return z[:n]

    def integers(self, n: int, hi: int) -> np.ndarray:
        """Integers in [0, hi) (multiplicative range reduction of a 53-bit uniform)."""
        return np.minimum((self.uniform(n) * hi).astype(np.int64), hi - 1)

    def unit_vectors(self, n: int) -> np.ndarray:
        v = self.normal(3 * n).reshape(n, 3)
        return v / np.linalg.norm(v, axis=1, keepdims=True)
