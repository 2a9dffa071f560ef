"""Counter-based, random-access generator keyed by (seed, stream, index).

    u64(seed, stream, i) = sm64( sm64( sm64(seed) ^ stream ) ^ i )

where sm64 is the SplitMix64 output function applied to (z + 0x9E3779B97F4A7C15):
    z += 0x9E3779B97F4A7C15; z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EB; return z ^ (z >> 31)          (all mod 2^64)

uniform01 = (u64 >> 11) * 2^-53  in [0, 1).
normal(i) = sqrt(-2 ln(1 - U(2i))) * cos(2 pi U(2i+1))   (Box-Muller, cosine branch), drawn in fp64.
Any index range can be produced independently, so month-long streams are generated chunk by chunk.
"""
import numpy as np

_M = np.uint64(0xFFFFFFFFFFFFFFFF)
_G = np.uint64(0x9E3779B97F4A7C15)
_A = np.uint64(0xBF58476D1CE4E5B9)
_B = np.uint64(0x94D049BB133111EB)


def _sm64(z):
    z = np.asarray(z, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = z + _G
        z = (z ^ (z >> np.uint64(30))) * _A
        z = (z ^ (z >> np.uint64(27))) * _B
        return z ^ (z >> np.uint64(31))


def u64(seed, stream, idx):
    """64-bit words for integer array `idx` (any shape)."""
    key = _sm64(_sm64(np.uint64(seed & 0xFFFFFFFFFFFFFFFF)) ^ np.uint64(stream & 0xFFFFFFFFFFFFFFFF))
    return _sm64(key ^ np.asarray(idx, dtype=np.uint64))


def uniform01(seed, stream, idx):
    return (u64(seed, stream, idx) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed, stream, start, count):
    """`count` standard normals for sample indices start .. start+count-1 (fp64)."""
    i = np.arange(start, start + count, dtype=np.uint64)
    u1 = uniform01(seed, stream, i * np.uint64(2))
    u2 = uniform01(seed, stream, i * np.uint64(2) + np.uint64(1))
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)
