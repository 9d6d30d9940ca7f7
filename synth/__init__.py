"""Seeded synthetic input generators shared by the tests, the oracle harness and bench.py.

This module holds NONE of the method's arithmetic: no ring product, no NTT, no CRT, no
rounding rule.  It only draws random numbers in a fixed order and shapes them the way the
paper's workloads are shaped (random ciphertexts, cnum per tensor, logN,
logQ; SURVEY.md 8c-A13 for the samplers the paper leaves open).

Everything is driven by ``numpy.random.Generator(PCG64(seed))``.
Layout of limb arrays: ``[..., L, N]`` uint32, limb 0 least significant (Eq. 22).
"""
from __future__ import annotations

import numpy as np


def rng(seed: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(seed))


def limbs_for_bits(bits: int) -> int:
    """Number of 32-bit limbs that hold a `bits`-bit value."""
    return (bits + 31) // 32


def uniform_limbs(g: np.random.Generator, lead_shape, N: int, bits: int) -> np.ndarray:
    """Coefficients uniform in [0, 2^bits) as uint32 limbs, shape lead_shape + (L, N)."""
    L = limbs_for_bits(bits)
    shape = tuple(lead_shape) + (L, N)
    a = g.integers(0, 1 << 32, size=shape, dtype=np.uint64).astype(np.uint32)
    top = bits - 32 * (L - 1)
    if top < 32:
        a[..., L - 1, :] &= np.uint32((1 << top) - 1)
    return a


def ternary_hwt(g: np.random.Generator, N: int, h: int) -> np.ndarray:
    """Ternary vector with exactly h non-zero entries (distinct positions, signs +-1 uniform)."""
    s = np.zeros(N, dtype=np.int64)
    pos = g.choice(N, size=min(h, N), replace=False)
    sign = g.integers(0, 2, size=pos.shape[0]) * 2 - 1
    s[pos] = sign
    return s


def ternary_uniform(g: np.random.Generator, N: int) -> np.ndarray:
    """Entries uniform over {-1, 0, 1}."""
    return g.integers(-1, 2, size=N).astype(np.int64)


def gaussian_error(g: np.random.Generator, N: int, sigma: float = 3.2) -> np.ndarray:
    """Rounded normal, sigma = 3.2 (the configs' 'discrete Gaussian')."""
    return np.rint(g.normal(0.0, sigma, size=N)).astype(np.int64)


def unit_disk(g: np.random.Generator, n: int) -> np.ndarray:
    """n complex values uniform in the unit disk, by rejection, fixed draw order."""
    out = np.empty(n, dtype=np.complex128)
    k = 0
    while k < n:
        xy = g.uniform(-1.0, 1.0, size=(2 * (n - k) + 8, 2))
        z = xy[:, 0] + 1j * xy[:, 1]
        z = z[np.abs(z) <= 1.0][: n - k]
        out[k : k + z.shape[0]] = z
        k += z.shape[0]
    return out


def uniform_mod(g: np.random.Generator, n: int, t: int) -> np.ndarray:
    """n integers uniform in [0, t), t < 2^63."""
    return g.integers(0, t, size=n, dtype=np.int64)


def uniform_big(g: np.random.Generator, N: int, bits: int) -> list:
    """N Python ints uniform in [0, 2^bits) (drawn as limbs, same stream as uniform_limbs)."""
    a = uniform_limbs(g, (), N, bits)
    L = a.shape[0]
    out = [0] * N
    for i in range(L - 1, -1, -1):
        col = a[i].tolist()
        out = [(o << 32) | c for o, c in zip(out, col)]
    return out
