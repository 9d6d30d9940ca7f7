"""Oracle's own negacyclic NTT (test infrastructure; shares nothing with the CUDA path).

Follows the paper's order and notation:
  * primes q = 1 (mod 2N) so a primitive 2N-th root psi exists
  * forward:  twist a_j <- a_j * psi^j, then a standard cyclic NTT with omega = psi^2
              (PAPER.md:346-350, 376-385), which is Eq. 8:
              abar_i = sum_j a_j psi^((2i+1) j)  mod q
  * inverse:  Eq. 9:  a_i = N^-1 psi^-i sum_j abar_j omega^(-ij) mod q
Outputs are in natural index order i = 0..N-1, exactly as Eq. 8 / Eq. 9 are written.

The oracle picks its OWN primes (the smallest primes above 2^30 that are 1 mod 2N), which are
not the ones the CUDA library uses; any exact choice yields the same ring product.
"""
from __future__ import annotations

import numpy as np

_MR_BASES = (2, 3, 5, 7, 11, 13, 17, 19, 23, 29, 31, 37)


def is_prime(n: int) -> bool:
    """Deterministic Miller-Rabin for n < 3.3e24 (bases 2..37)."""
    if n < 2:
        return False
    for b in _MR_BASES:
        if n % b == 0:
            return n == b
    d, r = n - 1, 0
    while d % 2 == 0:
        d //= 2
        r += 1
    for b in _MR_BASES:
        x = pow(b, d, n)
        if x == 1 or x == n - 1:
            continue
        for _ in range(r - 1):
            x = x * x % n
            if x == n - 1:
                break
        else:
            return False
    return True


def oracle_primes(N: int, min_product: int) -> list:
    """Smallest primes > 2^30 with q = 1 (mod 2N), ascending, until their product > min_product."""
    step = 2 * N
    q = (1 << 30) // step * step + step + 1
    out, prod = [], 1
    while prod <= min_product:
        if q >= (1 << 31):
            raise ValueError("oracle prime range exhausted")
        if is_prime(q):
            out.append(q)
            prod *= q
        q += step
    return out


def primitive_2n_root(q: int, N: int) -> int:
    """A primitive 2N-th root of unity psi mod q: psi^N = -1."""
    assert (q - 1) % (2 * N) == 0
    e = (q - 1) // (2 * N)
    for g in range(2, 1000):
        psi = pow(g, e, q)
        if pow(psi, N, q) == q - 1:
            return psi
    raise ValueError("no root found")


def _bitrev_perm(N: int) -> np.ndarray:
    n = N.bit_length() - 1
    idx = np.arange(N, dtype=np.int64)
    rev = np.zeros(N, dtype=np.int64)
    for b in range(n):
        rev |= ((idx >> b) & 1) << (n - 1 - b)
    return rev


def _powers(base: int, count: int, q: int) -> np.ndarray:
    out = np.empty(count, dtype=np.uint64)
    x = 1
    for i in range(count):
        out[i] = x
        x = x * base % q
    return out


def cyclic_ntt(a: np.ndarray, omega: int, q: int) -> np.ndarray:
    """Standard length-N cyclic transform A_i = sum_j a_j omega^(ij) mod q, natural order in and out.

    Iterative Cooley-Tukey: bit-reverse the input, then log2 N butterfly stages.
    a: uint64 array of values < q < 2^31 (products stay below 2^62).
    """
    N = a.shape[0]
    Q = np.uint64(q)
    x = a[_bitrev_perm(N)].astype(np.uint64)
    m = 2
    while m <= N:
        half = m // 2
        w = _powers(pow(omega, N // m, q), half, q)
        x = x.reshape(N // m, m)
        u = x[:, :half].copy()
        v = (x[:, half:] * w) % Q
        x[:, :half] = (u + v) % Q
        x[:, half:] = (u + Q - v) % Q
        x = x.reshape(N)
        m *= 2
    return x


def ntt_forward(a: np.ndarray, q: int, psi: int) -> np.ndarray:
    """Eq. 8: twist by psi^j, then cyclic NTT with omega = psi^2."""
    N = a.shape[0]
    Q = np.uint64(q)
    tw = _powers(psi, N, q)
    return cyclic_ntt((a.astype(np.uint64) * tw) % Q, psi * psi % q, q)


def ntt_inverse(abar: np.ndarray, q: int, psi: int) -> np.ndarray:
    """Eq. 9: cyclic transform with omega^-1, then N^-1 * psi^-i."""
    N = abar.shape[0]
    Q = np.uint64(q)
    omega_inv = pow(psi * psi % q, -1, q)
    x = cyclic_ntt(abar.astype(np.uint64), omega_inv, q)
    n_inv = pow(N, -1, q)
    untw = (_powers(pow(psi, -1, q), N, q) * np.uint64(n_inv)) % Q
    return (x * untw) % Q


def ntt_forward_direct(a, q: int, psi: int) -> list:
    """Eq. 8 evaluated literally, O(N^2), on Python ints.  Used only to pin ntt_forward."""
    N = len(a)
    return [sum(int(a[j]) * pow(psi, (2 * i + 1) * j, q) for j in range(N)) % q for i in range(N)]
