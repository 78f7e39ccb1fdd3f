"""Counter-based splitmix64 (SURVEY.md §8(d) "Common rules").

u(key, idx) is a pure function of (key, idx): no state, so the oracle harness
and the GPU harness can draw the same numbers in any order.
"""
import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_M1 = np.uint64(0xBF58476D1CE4E5B9)
_M2 = np.uint64(0x94D049BB133111EB)


def splitmix64_u64(key, idx):
    """idx-th output (0-based) of the splitmix64 stream seeded with `key`."""
    idx = np.asarray(idx, dtype=np.uint64)
    with np.errstate(over="ignore"):
        z = np.uint64(key) + (idx + np.uint64(1)) * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _M1
        z = (z ^ (z >> np.uint64(27))) * _M2
        z = z ^ (z >> np.uint64(31))
    return z


def uniform01(key, idx):
    """double in [0,1): top 53 bits of the splitmix64 output."""
    return (splitmix64_u64(key, idx) >> np.uint64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal01(key, n):
    """n standard normals by Box-Muller on the pairs (u[2i], u[2i+1])."""
    m = (n + 1) // 2
    i = np.arange(m, dtype=np.uint64)
    u1 = 1.0 - uniform01(key, 2 * i)          # (0,1]
    u2 = uniform01(key, 2 * i + np.uint64(1))
    r = np.sqrt(-2.0 * np.log(u1))
    out = np.empty(2 * m, dtype=np.float64)
    out[0::2] = r * np.cos(2.0 * np.pi * u2)
    out[1::2] = r * np.sin(2.0 * np.pi * u2)
    return out[:n]
