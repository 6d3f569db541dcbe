"""Pool content generator g (numpy side).

g64(seed, plane, q) = SplitMix64 finaliser of (seed ^ (plane << 40)) + q, and
the four 16-bit words 4q .. 4q+3 of a plane are its little-endian 16-bit lanes.
Uniform 16-bit patterns on purpose: they include bf16 NaN / Inf / subnormal
encodings, so any float conversion in a kernel corrupts them (BASELINE.json
configs[0] "seeded uniform 16-bit patterns").

The CUDA twin is workloads/csrc/kvfill.cu; tests/test_gpu_fill.py compares the
two on sampled pages.  This is test data generation, not the path under test.
"""
from __future__ import annotations

import numpy as np

_M64 = np.uint64(0xFFFFFFFFFFFFFFFF)
_GOLD = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)


def _mix64(x: np.ndarray) -> np.ndarray:
    with np.errstate(over="ignore"):
        z = (x + _GOLD) & _M64
        z = ((z ^ (z >> np.uint64(30))) * _C1) & _M64
        z = ((z ^ (z >> np.uint64(27))) * _C2) & _M64
        return z ^ (z >> np.uint64(31))


def g_words(seed: int, plane: int, first_word: int, n_words: int) -> np.ndarray:
    """uint16 words [first_word, first_word + n_words) of plane `plane`."""
    first_word, n_words = int(first_word), int(n_words)
    q0 = first_word // 4
    q1 = (first_word + n_words + 3) // 4
    base = np.uint64((int(seed) ^ (int(plane) << 40)) & 0xFFFFFFFFFFFFFFFF)
    with np.errstate(over="ignore"):
        q = (np.arange(q0, q1, dtype=np.uint64) + base) & _M64
    w = _mix64(q).view("<u2")  # 4 little-endian lanes per 64-bit hash
    lo = first_word - 4 * q0
    return w[lo: lo + n_words].copy()


def fill_plane_np(seed: int, plane: int, n_words: int) -> np.ndarray:
    return g_words(seed, plane, 0, n_words)
