"""Counter-based seeded random numbers for the synthetic workloads (input generation only;
no arithmetic of the method lives here).

value(seed, tag, index) depends only on its three arguments, so any element of any input
array can be regenerated anywhere, in any order (reading G11).

    h   = splitmix64-finaliser applied to (seed, tag, index)
    u   = (h >> 11 + 0.5) * 2^-53                      uniform in (0,1)
    z   = sqrt(-2 ln u1) cos(2 pi u2)                  Box-Muller, u1/u2 from two hashes
"""
import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def _mix(x):
    x = np.asarray(x, dtype=np.uint64)
    with np.errstate(over="ignore"):
        x = (x ^ (x >> np.uint64(30))) * _C1
        x = (x ^ (x >> np.uint64(27))) * _C2
        x = x ^ (x >> np.uint64(31))
    return x


def hash64(seed, tag, index):
    """64-bit hash of (seed, tag, index[, stream]); index may be an array."""
    with np.errstate(over="ignore"):
        s = _mix(np.uint64(seed) * _GOLD + np.uint64(tag))
        return _mix(s + (np.asarray(index, dtype=np.uint64) + np.uint64(1)) * _GOLD)


def uniform(seed, tag, index):
    h = hash64(seed, tag, index)
    return ((h >> np.uint64(11)).astype(np.float64) + 0.5) * (1.0 / 9007199254740992.0)


def normal(seed, tag, index):
    """Standard normal for every element of `index` (Box-Muller on two decorrelated hashes)."""
    idx = np.asarray(index, dtype=np.uint64)
    u1 = uniform(seed, 2 * tag, idx)
    u2 = uniform(seed, 2 * tag + 1, idx)
    return np.sqrt(-2.0 * np.log(u1)) * np.cos(2.0 * np.pi * u2)


def normal_array(seed, tag, shape):
    n = int(np.prod(shape))
    return normal(seed, tag, np.arange(n, dtype=np.uint64)).reshape(shape)
