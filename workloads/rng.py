"""Counter-based random numbers for the seeded synthetic workloads.

Every random number is a pure function of (seed, stream, index), so any slice of any
array can be regenerated independently and chunked/threaded generation gives the same
bytes as a single pass.  This module holds no rendering arithmetic: it is shared by the
oracle-side and the CUDA-side tests and by bench.py only as a source of inputs.

The mixer is the splitmix64 finaliser (public-domain constant set by S. Vigna) applied to
a counter built from seed, stream and index.  It is restated here, not imported, so that
the byte stream cannot change with a library version ("Concrete
inputs").
"""
from __future__ import annotations

import numpy as np

_U64 = np.uint64
_GOLDEN = _U64(0x9E3779B97F4A7C15)
_M1 = _U64(0xBF58476D1CE4E5B9)
_M2 = _U64(0x94D049BB133111EB)
_STREAM_MUL = _U64(0xD1342543DE82EF95)


def _mix(z: np.ndarray) -> np.ndarray:
    z = z.copy()
    z ^= z >> _U64(30)
    z *= _M1
    z ^= z >> _U64(27)
    z *= _M2
    z ^= z >> _U64(31)
    return z


def bits64(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """64 random bits for each entry of `index` (uint64 array)."""
    with np.errstate(over="ignore"):
        base = _U64(seed & 0xFFFFFFFFFFFFFFFF) + _U64(stream & 0xFFFFFFFF) * _STREAM_MUL
        z = (index.astype(np.uint64) + _U64(1)) * _GOLDEN + base
        return _mix(_mix(z))


def uniform(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """float64 uniform on [0, 1) with 53 random bits."""
    return (bits64(seed, stream, index) >> _U64(11)).astype(np.float64) * (1.0 / 9007199254740992.0)


def normal(seed: int, stream: int, index: np.ndarray) -> np.ndarray:
    """float64 standard normal by Box-Muller; uses streams `stream` and `stream + 1`."""
    u1 = uniform(seed, stream, index)
    u2 = uniform(seed, stream + 1, index)
    # 1 - u1 is in (0, 1], so the log is finite
    return np.sqrt(-2.0 * np.log1p(-u1)) * np.cos(2.0 * np.pi * u2)


def index_range(start: int, stop: int) -> np.ndarray:
    return np.arange(start, stop, dtype=np.uint64)
