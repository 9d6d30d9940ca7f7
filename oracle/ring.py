"""Negacyclic product in Z_M[X]/(X^N + 1) on arbitrary-precision integers (test infrastructure).

pm(a, b, M) is the plain definition:
    ctilde(x) = sum_i sum_j a_i b_j x^(i+j)                         (Eq. 5)
    c_i       = ctilde_i - ctilde_(N+i)   (mod M)                    (Eq. 6)
with the result as the canonical representative in [0, M).

Two routes, both exact:
  pm_schoolbook  Eq. 5-6 written out, O(N^2) big-int products (small N).
  pm_ntt         the oracle's own route for large N (Eq. 7; 326-328):
                 residues mod the oracle's primes -> Eq. 8 NTT -> pointwise -> Eq. 9 -> integer
                 by the direct CRT formula Eq. 1 (NOT Garner, and not the CUDA
                 path's primes) -> centred lift -> mod M.
Inputs are sequences of Python ints (any sign); outputs lists of Python ints in [0, M).
"""
from __future__ import annotations

import numpy as np

from . import ntt as _ntt

SCHOOLBOOK_MAX_N = 1 << 10


def pm_schoolbook(a, b, M: int) -> list:
    """Eq. 5 then Eq. 6, literally."""
    N = len(a)
    assert len(b) == N
    bo = np.array([int(v) for v in b], dtype=object)
    ct = np.zeros(2 * N, dtype=object)            # ctilde, degree <= 2N-2
    for i in range(N):
        ai = int(a[i])
        if ai:
            ct[i : i + N] += ai * bo             # Eq. 5
    return [int(ct[i] - ct[N + i]) % M for i in range(N)]   # Eq. 6


def crt_direct(residues, primes):
    """Eq. 1: X = | sum_i x_i * qhat_i * [qhat_i^-1]_{q_i} |_Mp,  qhat_i = Mp / q_i.

    residues: list (one per prime) of uint64 arrays of length N.  Returns (N Python ints in [0, Mp), Mp).
    """
    Mp = 1
    for q in primes:
        Mp *= q
    N = residues[0].shape[0]
    acc = np.zeros(N, dtype=object)
    for x, q in zip(residues, primes):
        qhat = Mp // q
        c = qhat * pow(qhat % q, -1, q)
        acc += x.astype(object) * c
    return [int(v) % Mp for v in acc], Mp


def pm_ntt(a, b, M: int) -> list:
    """Negacyclic product through the oracle's own NTT; exact for any integer inputs."""
    N = len(a)
    assert len(b) == N and N & (N - 1) == 0
    ao = np.array([int(v) for v in a], dtype=object)
    bo = np.array([int(v) for v in b], dtype=object)
    amax = max(1, int(max(abs(int(v)) for v in a)))
    bmax = max(1, int(max(abs(int(v)) for v in b)))
    # |c_k| <= N * amax * bmax; the centred lift needs the prime product > 2 * that.
    primes = _ntt.oracle_primes(N, 2 * N * amax * bmax)
    res = []
    for q in primes:
        psi = _ntt.primitive_2n_root(q, N)
        ra = (ao % q).astype(np.uint64)
        rb = (bo % q).astype(np.uint64)
        fa = _ntt.ntt_forward(ra, q, psi)
        fb = _ntt.ntt_forward(rb, q, psi)
        fc = (fa * fb) % np.uint64(q)                      # Eq. 7 Hadamard product
        res.append(_ntt.ntt_inverse(fc, q, psi))
    X, Mp = crt_direct(res, primes)
    half = Mp // 2
    return [((x - Mp) if x > half else x) % M for x in X]  # centred lift, then mod M


def pm(a, b, M: int) -> list:
    """The negacyclic product mod M; schoolbook where it finishes in seconds, own NTT above."""
    if len(a) <= SCHOOLBOOK_MAX_N:
        return pm_schoolbook(a, b, M)
    return pm_ntt(a, b, M)


def pm_coeff(a, b, k: int, M: int) -> int:
    """One output coefficient c_k of Eq. 5-6, O(N): used to spot-check full-size results."""
    N = len(a)
    s = 0
    for i in range(N):
        j = k - i
        if j >= 0:
            s += int(a[i]) * int(b[j])
        else:
            s -= int(a[i]) * int(b[j + N])
    return s % M


def add(a, b, M: int) -> list:
    return [(int(x) + int(y)) % M for x, y in zip(a, b)]


def centre(x: int, M: int) -> int:
    """Representative of x mod M in (-M/2, M/2] for even M, [-(M-1)/2, (M-1)/2] for odd M."""
    x %= M
    return x - M if x > M // 2 else x
