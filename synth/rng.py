"""Counter-based RNG: SplitMix64 streams keyed by (seed, stream id).

Every array is drawn from its own stream so that changing N or drawing an
extra array never shifts another array's values.  Pure numpy, vectorised.
"""
import numpy as np

_GOLD = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def _mix(z):
    z = (z ^ (z >> np.uint64(30))) * _M1
    z = (z ^ (z >> np.uint64(27))) * _M2
    return z ^ (z >> np.uint64(31))


def splitmix64(seed, stream, start, count):
    """`count` 64-bit outputs, counters start..start+count-1, of stream (seed, stream)."""
    with np.errstate(over="ignore"):
        base = _mix(np.uint64(seed) * _GOLD + np.uint64(stream) + np.uint64(1))
        ctr = np.arange(start, start + count, dtype=np.uint64) + np.uint64(1)
        return _mix(base + ctr * _GOLD)


def uniform01(seed, stream, count, start=0):
    """float64 uniforms in [0,1) from the top 24 bits (exactly representable in fp32)."""
    z = splitmix64(seed, stream, start, count)
    return (z >> np.uint64(40)).astype(np.float64) * (1.0 / 16777216.0)


def normal01(seed, stream, count):
    """Standard normals by Box-Muller in fp64 (two uniforms per pair of normals)."""
    half = (count + 1) // 2
    z = splitmix64(seed, stream, 0, 2 * half)
    u1 = ((z[0::2] >> np.uint64(40)).astype(np.float64) + 1.0) * (1.0 / 16777216.0)  # (0,1]
    u2 = (z[1::2] >> np.uint64(40)).astype(np.float64) * (1.0 / 16777216.0)
    r = np.sqrt(-2.0 * np.log(u1))
    out = np.empty(2 * half, dtype=np.float64)
    out[0::2] = r * np.cos(2.0 * np.pi * u2)
    out[1::2] = r * np.sin(2.0 * np.pi * u2)
    return out[:count]
