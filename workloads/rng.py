"""Counter-based uniform generator (SplitMix64 finaliser), random access by counter.

u(seed, k) = mix64(seed + (k + 1) * GOLDEN) >> 11) * 2^-53   in [0, 1)

Any draw can be produced without producing the ones before it, so a test can build point
x = 3071 of config c2 without building points 0..3070.
"""
import numpy as np

_GOLDEN = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64_uniform(seed: int, counters) -> np.ndarray:
    """Uniform doubles in [0,1) for the given 64-bit counters (array-like of ints)."""
    k = np.asarray(counters, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(seed) + (k + np.uint64(1)) * _GOLDEN
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
