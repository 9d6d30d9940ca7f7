"""Python-int <-> uint32 limb packing for the tests (test infrastructure).

Radix representation X = sum_i x_i 2^(32 i), 32-bit limbs (Eq. 22-23; 310).
Array layout [..., L, N]: limb index before coefficient index, limb 0 least significant.
"""
from __future__ import annotations

import numpy as np


def to_limbs(coeffs, L: int) -> np.ndarray:
    """N non-negative Python ints (< 2^(32 L)) -> uint32 array [L, N]."""
    N = len(coeffs)
    out = np.empty((L, N), dtype=np.uint32)
    cur = [int(c) for c in coeffs]
    assert all(c >= 0 for c in cur)
    for i in range(L):
        out[i] = np.array([c & 0xFFFFFFFF for c in cur], dtype=np.uint64).astype(np.uint32)
        cur = [c >> 32 for c in cur]
    assert not any(cur), "value does not fit in L limbs"
    return out


def from_limbs(arr: np.ndarray) -> list:
    """uint32 array [L, N] -> N Python ints."""
    L, N = arr.shape
    out = [0] * N
    for i in range(L - 1, -1, -1):
        col = arr[i].tolist()
        out = [(o << 32) | int(c) for o, c in zip(out, col)]
    return out
