"""Counter-based uniform random numbers (splitmix64 finaliser over a mixed counter).

draw(seed, config, b, stream, i) depends on nothing else, so generation is vectorised over
any subset of scenarios and is reproducible per scenario.
"""
import numpy as np

MASTER_SEED = 20231008  # arXiv id of the paper; per-config seed = MASTER_SEED + config #

_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)
_G = np.uint64(0x9E3779B97F4A7C15)


def _mix(z):
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def _bits(seed, b, stream, i):
    """uint64 hash of (seed, b, stream, i); b and i broadcast against each other."""
    with np.errstate(over="ignore"):
        b = np.asarray(b, dtype=np.uint64)
        i = np.asarray(i, dtype=np.uint64)
        z = _mix(np.uint64(seed) * _G + np.uint64(stream))
        z = _mix(z + (b + np.uint64(1)) * _G)
        z = _mix(z + (i + np.uint64(1)) * _M2)
        return z


def uniform(seed, b, stream, shape_tail, lo=0.0, hi=1.0):
    """float64 uniforms in [lo, hi), shape = b.shape + shape_tail.

    b: int array of scenario ids; stream: small int naming the quantity drawn."""
    b = np.asarray(b, dtype=np.uint64)
    n = int(np.prod(shape_tail)) if len(shape_tail) else 1
    i = np.arange(n, dtype=np.uint64)
    z = _bits(seed, b.reshape(b.shape + (1,)), stream, i)
    u = (z >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)
    u = u.reshape(b.shape + tuple(shape_tail))
    return lo + (hi - lo) * u


def randint(seed, b, stream, shape_tail, n):
    """ints in [0, n), shape = b.shape + shape_tail."""
    u = uniform(seed, b, stream, shape_tail)
    return np.minimum((u * n).astype(np.int64), n - 1)
