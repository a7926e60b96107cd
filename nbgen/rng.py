"""Counter-based random streams for the synthetic particle sets.

One independent splitmix64 stream per particle, so a set is the same no matter in which order or
on how many workers it is generated.  This module holds no N-body arithmetic: it only makes
uniform numbers, permutations and integer levels.  It is shared by the tests, the oracle harness
and bench.py; neither `oracle/` nor the CUDA path contains any of it.
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_KMUL = np.uint64(0xD1B54A32D192ED03)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_TWO_M53 = 2.0 ** -53


def _mix(z):
    z = (z ^ (z >> np.uint64(30))) * _C1
    z = (z ^ (z >> np.uint64(27))) * _C2
    return z ^ (z >> np.uint64(31))


class Streams:
    """`count` independent streams; stream k of seed s starts at s*GAMMA + k*KMUL (mod 2^64) and
    throws its first output away."""

    def __init__(self, seed, count, first=0):
        with np.errstate(over="ignore"):
            k = np.arange(first, first + count, dtype=np.uint64)
            self.state = np.uint64(seed) * _GAMMA + k * _KMUL
            self.state += _GAMMA  # discard the first output

    def bits(self, sel=None):
        """Next 64 random bits of the selected streams (all when sel is None)."""
        with np.errstate(over="ignore"):
            if sel is None:
                self.state += _GAMMA
                return _mix(self.state.copy())
            self.state[sel] += _GAMMA
            return _mix(self.state[sel])

    def uniform(self, sel=None):
        """Next uniform in [0, 1) with 53 random bits."""
        return (self.bits(sel) >> np.uint64(11)).astype(np.float64) * _TWO_M53


def permutation(seed, n):
    """Seeded permutation of 0..n-1: indices sorted by one 64-bit key per index (stable, so equal
    keys keep index order).  The first m entries are the 'active subset of size m'; subsets of
    different sizes are nested."""
    keys = Streams(seed, n).bits()
    return np.argsort(keys, kind="stable").astype(np.int32)


def integers(seed, n, lo, hi):
    """One integer per index, uniform in [lo, hi] inclusive."""
    u = Streams(seed, n).uniform()
    return lo + np.minimum((u * (hi - lo + 1)).astype(np.int64), hi - lo)
