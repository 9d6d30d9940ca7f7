"""Key generation, symmetric encryption, decryption and CKKS encode/decode (test infrastructure).

Host-side only: the paper does all of this on the CPU before offloading and
gives no formulas; the readings are DESIGN.md section 3 (SURVEY.md 8c steps 4 and 8, A1, A2, A10,
A13, A14).  Floating point appears only in encode/decode and is checked only through the
numeric CKKS bound (north_star): max |decode(Dec(mult)) - z z'| <= 2^-20 at Delta = 2^40.

Random numbers come from `synth` (seeded, fixed draw order: s, e', a', then per ciphertext
a, e, message); no randomness is drawn here.
"""
from __future__ import annotations

import numpy as np

import synth
from .ring import pm, add, centre
from .scheme import Params


def pm_sparse(a, s, M: int) -> list:
    """a * s for a sparse small s, straight from Eq. 5-6 skipping zero terms:
    each non-zero s_j contributes s_j * a_i to position i+j, negated past X^N."""
    N = len(a)
    ao = np.array([int(v) for v in a], dtype=object)
    acc = np.zeros(N, dtype=object)
    for j in np.nonzero(np.asarray(s))[0]:
        j = int(j)
        sj = int(s[j])
        acc[j:] += sj * ao[: N - j]
        if j:
            acc[:j] -= sj * ao[N - j :]
    return [int(v) % M for v in acc]


def pm_secret(a, s, M: int) -> list:
    """a * s with s a small (ternary) polynomial: sparse route if s is sparse, general pm otherwise."""
    nz = int(np.count_nonzero(np.asarray(s)))
    if nz <= 256:
        return pm_sparse(a, s, M)
    return pm(a, [int(v) % M for v in s], M)


def keygen(prm: Params, g: np.random.Generator, hwt: int | None = 64, sigma: float = 3.2):
    """Secret s (ternary; Hamming weight `hwt`, or uniform ternary if hwt is None) and the
    relinearisation key evk = (b', a') mod PQ (DESIGN 3, A2, A10):
        CKKS: b' = -a' s + e' + P s^2,   BGV: b' = -a' s + t e' + P s^2."""
    N, PQ = prm.N, prm.PQ
    s = synth.ternary_hwt(g, N, hwt) if hwt is not None else synth.ternary_uniform(g, N)
    e = synth.gaussian_error(g, N, sigma)
    a = synth.uniform_big(g, N, (PQ - 1).bit_length() - (0 if prm.is_ckks else 1))
    s_list = [int(v) for v in s]
    s2 = pm([v % PQ for v in s_list], [v % PQ for v in s_list], PQ)
    a_s = pm_secret(a, s_list, PQ)
    mult = 1 if prm.is_ckks else prm.t
    b = [(-x + mult * int(ee) + prm.P * y) % PQ for x, ee, y in zip(a_s, e, s2)]
    return s_list, (b, a)


def encrypt(prm: Params, g: np.random.Generator, s, m, sigma: float = 3.2):
    """Symmetric encryption of the integer polynomial m:  c1 = a uniform, c0 = -a s + e + m (CKKS)
    or -a s + t e + m (BGV), mod Q."""
    N, Q = prm.N, prm.Q
    a = synth.uniform_big(g, N, (Q - 1).bit_length() - (0 if prm.is_ckks else 1))
    e = synth.gaussian_error(g, N, sigma)
    mult = 1 if prm.is_ckks else prm.t
    a_s = pm_secret(a, s, Q)
    c0 = [(-x + mult * int(ee) + int(mm)) % Q for x, ee, mm in zip(a_s, e, m)]
    return c0, a


def decrypt(ct, s, Q: int) -> list:
    """mu = c0 + c1 s mod Q, recentred (DESIGN 3, A1)."""
    c0, c1 = ct
    return [centre(v, Q) for v in add(c0, pm_secret(c1, s, Q), Q)]


def decrypt3(d, s, Q: int) -> list:
    """d0 + d1 s + d2 s^2 mod Q, recentred: what a tensor triple decrypts to."""
    d0, d1, d2 = d
    d2s = pm_secret(d2, s, Q)
    inner = add(d1, d2s, Q)
    return [centre(v, Q) for v in add(d0, pm_secret(inner, s, Q), Q)]


def decrypt_bgv(ct, s, prm: Params) -> list:
    return [v % prm.t for v in decrypt(ct, s, prm.Q)]


# --- CKKS canonical-embedding encode / decode, full packing N/2 slots (DESIGN 3, A14) ---------
# slot j sits at the root zeta_j = exp(i pi (2j+1) / N), the kernel of Eq. 10-11

def encode(z: np.ndarray, N: int, scale: float) -> list:
    """m_k = round( (2/N) Re sum_j scale z_j conj(zeta_j)^k ),  k = 0..N-1.
    sum_j z_j exp(-i pi (2j+1) k / N) = exp(-i pi k / N) * FFT_N(z padded)[k]."""
    assert z.shape[0] == N // 2
    zp = np.zeros(N, dtype=np.complex128)
    zp[: N // 2] = z
    k = np.arange(N)
    v = np.exp(-1j * np.pi * k / N) * np.fft.fft(zp)
    m = np.rint((2.0 / N) * scale * v.real)
    return [int(x) for x in m]


def decode(m, N: int, scale: float) -> np.ndarray:
    """z_j = m(zeta_j) / scale = sum_k m_k exp(i pi (2j+1) k / N) / scale,  j < N/2."""
    k = np.arange(N)
    mf = np.array([float(int(x)) for x in m], dtype=np.float64)
    v = np.fft.ifft(mf * np.exp(1j * np.pi * k / N)) * N
    return v[: N // 2] / scale


def rotkeygen(prm: Params, g: np.random.Generator, s, k: int, sigma: float = 3.2):
    """Rotation / conjugation key for the Galois element k (DESIGN 3, NEXT-2 reading): rk = (b', a') mod PQ,
    b' = -a' s + e' + P sigma_k(s)  (BGV: t e')."""
    from .scheme import automorphism
    N, PQ = prm.N, prm.PQ
    e = synth.gaussian_error(g, N, sigma)
    a = synth.uniform_big(g, N, (PQ - 1).bit_length() - (0 if prm.is_ckks else 1))
    sk = automorphism([v % PQ for v in s], k, PQ)
    a_s = pm_secret(a, s, PQ)
    mult = 1 if prm.is_ckks else prm.t
    b = [(-x + mult * int(ee) + prm.P * y) % PQ for x, ee, y in zip(a_s, e, sk)]
    return b, a


def slot_image(N: int, k: int):
    """Where the automorphism X -> X^k sends the slots of `encode` (roots zeta_j = exp(i pi (2j+1)/N), j < N/2):
    (sigma_k m)(zeta_j) = m(zeta_j^k) = m(zeta_j') with 2j'+1 = k (2j+1) mod 2N.  Returns (src, conj): new slot j holds
    z[src[j]], conjugated where conj[j] (j' >= N/2 is the conjugate of slot N-1-j')."""
    src, conj = [], []
    for j in range(N // 2):
        jp = ((k * (2 * j + 1)) % (2 * N) - 1) // 2
        if jp < N // 2:
            src.append(jp); conj.append(False)
        else:
            src.append(N - 1 - jp); conj.append(True)
    return src, conj
