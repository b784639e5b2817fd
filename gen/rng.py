"""Counter-based random numbers for the synthetic event generator.

Own splitmix64 mixer so that events are reproducible bit for bit on any machine and numpy version
(SURVEY.md Appendix D asks for exactly this).  A stream is addressed by (seed, key); element i of a
stream is mix64(base + (i+1)*GOLDEN).  No state is carried, so draws do not depend on call order.

This module holds no tracking arithmetic; it only serves gen/events.py.
"""
from __future__ import annotations

import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix64(x: np.ndarray) -> np.ndarray:
    x = np.asarray(x, dtype=np.uint64).copy()
    with np.errstate(over="ignore"):
        x ^= x >> np.uint64(30)
        x *= _M1
        x ^= x >> np.uint64(27)
        x *= _M2
        x ^= x >> np.uint64(31)
    return x


class Rng:
    """Stateless stream family: Rng(seed).uniform(key, n) is a pure function of (seed, key, n)."""

    def __init__(self, seed: int):
        self.seed = int(seed) & 0xFFFFFFFFFFFFFFFF

    def _base(self, key: int) -> np.uint64:
        with np.errstate(over="ignore"):
            a = _mix64(np.array([self.seed], dtype=np.uint64))[0]
            b = _mix64(np.array([(int(key) * 0xD1342543DE82EF95 + 0x632BE59BD9B4E019) & 0xFFFFFFFFFFFFFFFF],
                                dtype=np.uint64))[0]
            return _mix64(np.array([a ^ b], dtype=np.uint64))[0]

    def bits(self, key: int, n: int) -> np.ndarray:
        base = self._base(key)
        with np.errstate(over="ignore"):
            ctr = (np.arange(1, n + 1, dtype=np.uint64) * _GOLDEN) + base
        return _mix64(ctr)

    def uniform(self, key: int, n: int) -> np.ndarray:
        """n doubles in the open interval (0, 1)."""
        return ((self.bits(key, n) >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)

    def normal(self, key: int, n: int) -> np.ndarray:
        """n standard normals (Box-Muller on two sub-streams)."""
        u1 = self.uniform(2 * key + 1_000_003, n)
        u2 = self.uniform(2 * key + 1_000_004, n)
        return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)

    def exponential(self, key: int, n: int, mean: float) -> np.ndarray:
        return -mean * np.log(self.uniform(key, n))

    def poisson(self, key: int, lam: np.ndarray) -> np.ndarray:
        """One Poisson draw per entry of lam, by inverse CDF on one uniform per entry (lam < 700)."""
        lam = np.asarray(lam, dtype=np.float64)
        u = self.uniform(key, lam.size).reshape(lam.shape)
        k = np.zeros(lam.shape, dtype=np.int64)
        p = np.exp(-lam)
        cdf = p.copy()
        todo = (u > cdf) & (lam > 0)
        it = 0
        while todo.any() and it < 5000:
            k[todo] += 1
            p[todo] *= lam[todo] / k[todo]
            cdf[todo] += p[todo]
            todo &= u > cdf
            it += 1
        return k

    def permutation_keys(self, key: int, n: int) -> np.ndarray:
        """n sort keys; argsort of them is a uniform random permutation."""
        return self.bits(key, n)
