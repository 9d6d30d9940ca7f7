"""Parameters and the homomorphic hot path on arbitrary-precision integers (test infrastructure).

The paper names the operations (`mult_pairwise_into` = ciphertext product followed by
relinearisation; `rescaleBy_pairwise_into`) and the ring
(Z_Q[X]/(X^N+1), Q = 2^logQ for CKKS) but prints no formula for key switching
or rounding; the readings used here are the ones listed in DESIGN.md section 3.

Ciphertext ct = (c0, c1), decryption c0 + c1*s mod Q.  Tensor triple (d0, d1, d2) decrypts as
d0 + d1*s + d2*s^2.  Every polynomial is a list of N Python ints in [0, modulus).
"""
from __future__ import annotations

from dataclasses import dataclass

from .ring import pm, add


def make_modulus(log: int, t: int) -> int:
    """t == 0: 2^log (CKKS).  t > 0: the least odd integer > 2^log that is 1 (mod t) (BGV)."""
    if t == 0:
        return 1 << log
    q = (1 << log) + 1
    while not (q % 2 == 1 and q % t == 1):
        q += 1
    return q


@dataclass(frozen=True)
class Params:
    N: int
    logQ: int
    logP: int
    t: int = 0          # 0 = CKKS, odd t > 0 = BGV plaintext modulus

    @property
    def Q(self) -> int:
        return make_modulus(self.logQ, self.t)

    @property
    def P(self) -> int:
        return make_modulus(self.logP, self.t)

    @property
    def PQ(self) -> int:
        return self.P * self.Q

    @property
    def L(self) -> int:
        return ((self.Q - 1).bit_length() + 31) // 32

    @property
    def L_PQ(self) -> int:
        return ((self.PQ - 1).bit_length() + 31) // 32

    @property
    def is_ckks(self) -> bool:
        return self.t == 0


def polymul(prm: Params, a, b) -> list:
    """c = a * b in Z_Q[X]/(X^N+1)."""
    return pm(a, b, prm.Q)


def he_mult(prm: Params, ct1, ct2):
    """Tensor product (north_star item 4):
    d0 = c0*c0', d1 = c0*c1' + c1*c0', d2 = c1*c1'   (all mod Q)."""
    Q = prm.Q
    c0, c1 = ct1
    e0, e1 = ct2
    d0 = pm(c0, e0, Q)
    d1 = add(pm(c0, e1, Q), pm(c1, e0, Q), Q)
    d2 = pm(c1, e1, Q)
    return d0, d1, d2


def round_shift(x: int, k: int) -> int:
    """floor((x + 2^(k-1)) / 2^k): round half up on the canonical representative (DESIGN 3, A3)."""
    return (x + (1 << (k - 1))) >> k


def relinearize_ckks(prm: Params, d, evk):
    """CKKS key switch with one big auxiliary modulus P = 2^logP (DESIGN 3, A2-A4):
    x_b = d2*b' mod PQ, x_a = d2*a' mod PQ as canonical values in [0, PQ);
    k = ((x + P/2) >> logP) mod Q;  out = (d0 + k_b, d1 + k_a) mod Q."""
    assert prm.is_ckks
    Q, PQ = prm.Q, prm.PQ
    d0, d1, d2 = d
    evk_b, evk_a = evk
    xb = pm(d2, evk_b, PQ)
    xa = pm(d2, evk_a, PQ)
    kb = [round_shift(x, prm.logP) % Q for x in xb]
    ka = [round_shift(x, prm.logP) % Q for x in xa]
    return add(d0, kb, Q), add(d1, ka, Q)


def _div_p_bgv(x: int, P: int, Q: int, t: int, Pinv_t: int) -> int:
    """One coefficient of the BGV divide-by-P (DESIGN 3, A10 / SURVEY 8c step 6)."""
    r = x % P
    if r > P // 2:                 # recentre to (-P/2, P/2); P odd, no tie
        r -= P
    k = (-r * Pinv_t) % t
    if k > t // 2:                 # recentre to (-t/2, t/2); t odd, no tie
        k -= t
    assert (x - r) % P == 0
    return ((x - r) // P - k) % Q


def relinearize_bgv(prm: Params, d, evk):
    """BGV key switch, P and Q odd, P = 1 (mod t): nearest multiple of P removed, then the
    mod-t correction k so that the removed quantity r + P*k is 0 (mod t)."""
    assert not prm.is_ckks
    Q, P, PQ, t = prm.Q, prm.P, prm.PQ, prm.t
    Pinv_t = pow(P % t, -1, t)
    d0, d1, d2 = d
    evk_b, evk_a = evk
    xb = pm(d2, evk_b, PQ)
    xa = pm(d2, evk_a, PQ)
    kb = [_div_p_bgv(x, P, Q, t, Pinv_t) for x in xb]
    ka = [_div_p_bgv(x, P, Q, t, Pinv_t) for x in xa]
    return add(d0, kb, Q), add(d1, ka, Q)


def relinearize(prm: Params, d, evk):
    return relinearize_ckks(prm, d, evk) if prm.is_ckks else relinearize_bgv(prm, d, evk)


def rescale(prm: Params, ct, p: int):
    """CKKS rescale by 2^p (DESIGN 3, A3):
    c' = ((c + 2^(p-1)) >> p) mod 2^(logQ - p) on canonical c in [0, Q), both components."""
    assert prm.is_ckks and 1 <= p < prm.logQ
    Q2 = 1 << (prm.logQ - p)
    return tuple([round_shift(int(c), p) % Q2 for c in comp] for comp in ct)


# ---- NEXT-1: the coefficient-wise ciphertext operations and the level drop -----------------------------
# The paper lists them by name only (add_pairwise_into, sub_pairwise_into, negate_pairwise_into, PAPER.md:654-662;
# moddownBy_pairwise_into, "modulus switching operation to reduce ciphertext level").  In the ring
# Z_Q[X]/(X^N+1) they are the component-wise definitions below on canonical representatives in [0, Q); with
# Q = 2^logq dropping to a smaller power of two is reduction mod 2^logq' (A3 / A12 conventions).
def ct_add(prm: Params, ct1, ct2):
    Q = prm.Q
    return tuple([(x + y) % Q for x, y in zip(a, b)] for a, b in zip(ct1, ct2))


def ct_sub(prm: Params, ct1, ct2):
    Q = prm.Q
    return tuple([(x - y) % Q for x, y in zip(a, b)] for a, b in zip(ct1, ct2))


def ct_negate(prm: Params, ct):
    Q = prm.Q
    return tuple([(-x) % Q for x in a] for a in ct)


def moddown(prm: Params, ct, new_logq: int):
    """CKKS only: the same ciphertext one or more levels down, every coefficient mod 2^new_logq."""
    assert prm.is_ckks and 1 <= new_logq <= prm.logQ
    m = 1 << new_logq
    return tuple([x % m for x in a] for a in ct)


# ---- NEXT-4: BGV modulus switching ----------------------------------------------------------------------
# The paper names a "CKKS-BGV scheme" and lists one level-reducing operation (moddownBy_pairwise_into,
# "modulus switching operation to reduce ciphertext level") without a BGV formula: PARITY UNPINNED by the
# paper.  Reading (A20): the switch goes from Q to Q' = make_modulus(new_logQ, t), a modulus of the same
# construction (odd, 1 mod t), and each coefficient c in [0, Q) becomes the integer nearest to c Q'/Q, corrected by the
# same centred multiple of t as in the divide-by-P of the key switch (step 6 of SURVEY.md 8c): with x = c Q' in [0, Q Q'),
#     r = x mod Q centred,  k = (-r Q^-1) mod t centred,  c' = ((x - r)/Q - k) mod Q'.
# The removed quantity delta = r + Q k is 0 (mod Q-multiples aside) mod t and |delta| <= Q (1 + t)/2, so with
# Q = Q' = 1 (mod t) the plaintext m + t e decrypts to the same m under Q' while the noise shrinks by Q'/Q.
def modswitch_bgv(prm: Params, ct, new_logQ: int):
    """BGV ciphertext mod Q -> the same plaintext mod Q' = make_modulus(new_logQ, t), every component."""
    assert not prm.is_ckks and 1 <= new_logQ < prm.logQ
    Q, t = prm.Q, prm.t
    Q2 = make_modulus(new_logQ, t)
    Qinv_t = pow(Q % t, -1, t)
    return tuple([_div_p_bgv(int(c) * Q2, Q, Q2, t, Qinv_t) for c in comp] for comp in ct)


# ---- NEXT-2: slot rotation / conjugation --------------------------------------------------------------------
# The paper names the operations (conjugate_pairwise_into, leftrotate_broadcast_into with "precomputed Galois / rotation
# keys") and gives no formula.  Reading: the Galois automorphism sigma_k: a(X) -> a(X^k) on both
# components, then the key switch of A2 / A3 / A10 with the key rk = (b', a'), b' = -a' s + e' + P sigma_k(s): the triple
# (sigma(c0), 0, sigma(c1)) decrypts under (1, s, sigma_k(s)) exactly like a tensor triple under (1, s, s^2), so the
# relinearisation procedure applies unchanged.
def automorphism(a, k: int, M: int) -> list:
    """a(X^k) mod (X^N + 1, M), k odd: coefficient i moves to i k mod 2N, negated when that is >= N."""
    N = len(a)
    assert k % 2 == 1
    out = [0] * N
    for i, x in enumerate(a):
        j = (i * k) % (2 * N)
        if j < N:
            out[j] = x % M
        else:
            out[j - N] = (-x) % M
    return out


def rotate(prm: Params, ct, k: int, rk):
    Q = prm.Q
    d = (automorphism(ct[0], k, Q), [0] * prm.N, automorphism(ct[1], k, Q))
    return relinearize(prm, d, rk)


# ---- NEXT-3: ciphertext x plaintext ----------------------------------------------------------------------
# multconstvec_pairwise_into / multconst_broadcast_into: "element-wise multiplication with
# per-ciphertext constants" / "of a single constant across a ciphertext tensor".  On an encoded plaintext polynomial m
# this is the ring product on both components (decryption is linear: (c0 + c1 s) m = c0 m + (c1 m) s).
def mult_plain(prm: Params, ct, m):
    Q = prm.Q
    return pm(ct[0], m, Q), pm(ct[1], m, Q)


def add_plain(prm: Params, ct, m):
    """ct + plaintext polynomial m (addconst_pairwise / _broadcast: names only): the plaintext is added
    to component 0, since Dec = c0 + c1 s is linear and Dec of (m, 0) is m."""
    Q = prm.Q
    return [(x + y) % Q for x, y in zip(ct[0], m)], list(ct[1])


def mult_scalar(prm: Params, ct, k: int):
    """ct times the integer constant k (multconst with a scalar: names only): every coefficient of both
    components times k mod Q; k may be negative."""
    Q = prm.Q
    return tuple([(x * k) % Q for x in a] for a in ct)


def mul_monomial(prm: Params, ct, k: int):
    """X^k * ct, 0 <= k < 2N: the ring product with a monomial on every component (a signed rotation of the coefficients,
    pin P3).  k = N/2 multiplies every CKKS slot by the imaginary unit (imult_pairwise_into):
    zeta_j^(N/2) = exp(i pi (2j+1)/2) = +-i ... the sign alternates with j, see tests."""
    N, Q = prm.N, prm.Q
    mono = [0] * N
    if k < N:
        mono[k] = 1
    else:
        mono[k - N] = Q - 1
    return tuple(pm(a, mono, Q) for a in ct)
