"""Counter-based seeded generator (SplitMix64 finaliser) for the synthetic workloads.

Every draw is a pure function of (seed, stream, index), so inputs do not depend on
numpy's generator implementation.  Holds none of the method's arithmetic.
"""
from __future__ import annotations

import numpy as np

SEED = 20190110
_M64 = (1 << 64) - 1


def _mix(z: np.ndarray) -> np.ndarray:
    z = (z + np.uint64(0x9E3779B97F4A7C15)).astype(np.uint64)
    z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
    z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
    return z ^ (z >> np.uint64(31))


def _key(seed: int, stream) -> np.uint64:
    h = np.uint64(seed & _M64)
    if isinstance(stream, (tuple, list)):
        parts = stream
    else:
        parts = (stream,)
    with np.errstate(over="ignore"):
        for p in parts:
            if isinstance(p, str):
                v = 1469598103934665603
                for ch in p.encode():
                    v = ((v ^ ch) * 1099511628211) & _M64
                p = v
            h = _mix(np.array([h ^ np.uint64(int(p) & _M64)], dtype=np.uint64))[0]
    return h


def bits(stream, n: int, seed: int = SEED, offset: int = 0) -> np.ndarray:
    """n uint64 words of stream `stream` (an int, str or tuple of them)."""
    k = _key(seed, stream)
    with np.errstate(over="ignore"):
        idx = np.arange(offset, offset + n, dtype=np.uint64)
        return _mix(_mix(idx * np.uint64(0xD1342543DE82EF95) + k) ^ k)


def uniform(stream, n: int, lo: float = 0.0, hi: float = 1.0, seed: int = SEED) -> np.ndarray:
    u = (bits(stream, n, seed) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))
    return lo + (hi - lo) * u


def randint(stream, n: int, lo: int, hi: int, seed: int = SEED) -> np.ndarray:
    """integers in [lo, hi) (modulo draw; bias < 2^-40 for the ranges used here)."""
    return (lo + (bits(stream, n, seed) % np.uint64(hi - lo)).astype(np.int64)).astype(np.int64)


def normal(stream, n: int, seed: int = SEED) -> np.ndarray:
    u1 = uniform((stream, "bm1") if not isinstance(stream, tuple) else stream + ("bm1",), n,
                 seed=seed)
    u2 = uniform((stream, "bm2") if not isinstance(stream, tuple) else stream + ("bm2",), n,
                 seed=seed)
    return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)


def permutation(stream, n: int, seed: int = SEED) -> np.ndarray:
    return np.argsort(bits(stream, n, seed), kind="stable")
