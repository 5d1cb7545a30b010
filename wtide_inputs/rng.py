"""Counter-based integer hash: uniform(seed, config, track, carrier, draw) in [0, 1).

splitmix64-style finaliser applied to a combined 64-bit key; uniform = top 24 bits * 2^-24,
so every value is exactly representable in float32 and identical wherever it is evaluated.
"""
import numpy as np

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_G = np.uint64(0x9E3779B97F4A7C15)


def _mix(z):
    with np.errstate(over="ignore"):
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def hash64(seed, config, track, carrier, draw):
    with np.errstate(over="ignore"):
        z = _mix(np.asarray(seed, dtype=np.uint64) + _G)
        for v in (config, track, carrier, draw):
            z = _mix(z + (np.asarray(v, dtype=np.uint64) + np.uint64(1)) * _G)
    return z


def uniform(seed, config, track, carrier, draw):
    """float64 array (values are multiples of 2^-24) broadcast over the integer arguments."""
    return (hash64(seed, config, track, carrier, draw) >> np.uint64(40)).astype(np.float64) * (2.0 ** -24)
