"""Counter-based random numbers shared by the oracle-side and CUDA-side tests.

No generator state: element ``index`` of stream ``stream`` under ``seed`` is
``splitmix64(seed ^ (stream * GOLD) + index)``, so any element can be regenerated
anywhere (SURVEY.md §8(d) "Common generator rules").  This module holds none of
the rendering method's arithmetic.
"""
import numpy as np

GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64(x):
    """SplitMix64 finaliser applied to ``x + GOLD`` (uint64 wrap-around arithmetic)."""
    with np.errstate(over="ignore"):
        z = np.asarray(x, dtype=np.uint64) + GOLD
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        return z ^ (z >> np.uint64(31))


def hash_u64(seed, stream, index):
    with np.errstate(over="ignore"):
        base = np.uint64(seed) ^ (np.uint64(stream) * GOLD)
        return splitmix64(base + np.asarray(index, dtype=np.uint64))


def uniform(seed, stream, index):
    """U[0,1) doubles from the top 53 bits."""
    return (hash_u64(seed, stream, index) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed, stream, index):
    """Standard normals by Box-Muller from streams ``stream`` and ``stream + 0x5151``."""
    u1 = uniform(seed, stream, index)
    u2 = uniform(seed, stream + 0x5151, index)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def uniform_chunked(seed, stream, n, lo, hi, dtype=np.float32, chunk=1 << 24):
    """``n`` uniforms in [lo,hi) as ``dtype`` without a huge uint64 temporary."""
    out = np.empty(n, dtype=dtype)
    for s in range(0, n, chunk):
        e = min(n, s + chunk)
        out[s:e] = lo + (hi - lo) * uniform(seed, stream, np.arange(s, e, dtype=np.uint64))
    return out
