"""Pins for the CPU oracle: each check ties an oracle function to something other than itself
(hand brute force, closed forms, a library big-int multiply, algebraic laws, decryption
invariants).  CPU only.  Citations: PAPER.md line numbers; DESIGN.md section 3 for readings."""
import os
import random

import numpy as np
import pytest

import synth
from oracle import harness, ntt, ring, scheme
from oracle.limbs import from_limbs, to_limbs

GOLD = os.path.join(os.path.dirname(__file__), "golden")


def _read_golden(name):
    out = {}
    with open(os.path.join(GOLD, name)) as f:
        for line in f:
            line = line.strip()
            if not line or line.startswith("#"):
                continue
            k, *v = line.split()
            out[k] = [int(x) for x in v]
    return out


def _naive_negacyclic(a, b):
    """Eq. 5-6 expanded term by term into a dict of exponents (test-local)."""
    N = len(a)
    tilde = {}
    for i, x in enumerate(a):
        for j, y in enumerate(b):
            tilde[i + j] = tilde.get(i + j, 0) + x * y
    return [tilde.get(i, 0) - tilde.get(N + i, 0) for i in range(N)]


# ---- P2: hand brute force, tiny case -------------------------------------------------------
def test_p2_golden_n4():
    g = _read_golden("negacyclic_n4.txt")
    a, b = g["a"], g["b"]
    big = 1 << 64
    got = ring.pm_schoolbook(a, b, big)
    assert [ring.centre(v, big) for v in got] == g["integers"]
    assert ring.pm_schoolbook(a, b, 256) == g["mod256"]
    assert ring.pm_schoolbook(a, b, 97) == g["mod97"]
    assert ring.pm_ntt(a, b, 256) == g["mod256"]
    assert ring.pm_ntt(a, b, 97) == g["mod97"]


# ---- P1: definition on random small inputs ---------------------------------------------------
@pytest.mark.parametrize("N,bits", [(8, 5), (8, 70), (16, 128), (32, 33)])
def test_p1_definition_small(N, bits):
    rnd = random.Random(N * 1000 + bits)
    M = (1 << bits) - rnd.randrange(0, 3)
    a = [rnd.randrange(M) for _ in range(N)]
    b = [rnd.randrange(M) for _ in range(N)]
    want = [v % M for v in _naive_negacyclic(a, b)]
    assert ring.pm_schoolbook(a, b, M) == want
    assert ring.pm_ntt(a, b, M) == want
    for k in (0, 1, N - 1):
        assert ring.pm_coeff(a, b, k, M) == want[k]


# ---- P3: monomials ---------------------------------------------------------------------------
@pytest.mark.parametrize("route", [ring.pm_schoolbook, ring.pm_ntt])
def test_p3_monomials(route):
    N, Q = 64, 1 << 100
    rnd = random.Random(3)
    a = [rnd.randrange(Q) for _ in range(N)]
    one = [1] + [0] * (N - 1)
    assert route(a, one, Q) == a                                  # a * 1 = a
    x = [0, 1] + [0] * (N - 2)
    xn1 = [0] * (N - 1) + [1]
    assert route(x, xn1, Q) == [Q - 1] + [0] * (N - 1)           # X * X^(N-1) = -1
    for k in (1, 5, N - 1):
        xk = [0] * N
        xk[k] = 1
        want = [(-a[i - k + N]) % Q if i < k else a[i - k] for i in range(N)]   # signed rotation
        assert route(a, xk, Q) == want


# ---- P4: ring laws ---------------------------------------------------------------------------
def test_p4_ring_laws():
    N, Q = 32, (1 << 90) + 7
    rnd = random.Random(4)
    a, b, c = ([rnd.randrange(Q) for _ in range(N)] for _ in range(3))
    pm = ring.pm_ntt
    assert pm(a, b, Q) == pm(b, a, Q)
    assert pm(a, ring.add(b, c, Q), Q) == ring.add(pm(a, b, Q), pm(a, c, Q), Q)
    assert pm(pm(a, b, Q), c, Q) == pm(a, pm(b, c, Q), Q)


# ---- P5: closed form at the extreme of the bound -------------------------------------------------
@pytest.mark.parametrize("N,logQ", [(16, 64), (256, 128), (2048, 218)])
def test_p5_all_qm1_closed_form(N, logQ):
    """a = b = (Q-1, ..., Q-1): c_k = (Q-1)^2 ((k+1) - (N-1-k)) = 2k + 2 - N (mod Q).
    The raw values reach +N(Q-1)^2 and -(N-2)(Q-1)^2, i.e. both ends of the CRT range."""
    Q = 1 << logQ
    a = [Q - 1] * N
    want = [(2 * k + 2 - N) % Q for k in range(N)]
    assert ring.pm(a, a, Q) == want
    if N <= 256:
        assert ring.pm_schoolbook(a, a, Q) == want
    assert ring.pm_ntt(a, a, Q) == want


# ---- P6: reduction to one library big-int multiply (Kronecker substitution) ----------------------
def _kronecker(a, b, M):
    N = len(a)
    w = 2 * max(max(a), max(b), 1).bit_length() + N.bit_length() + 1
    A = sum(int(v) << (w * i) for i, v in enumerate(a))
    B = sum(int(v) << (w * i) for i, v in enumerate(b))
    C = A * B
    mask = (1 << w) - 1
    ct = [(C >> (w * i)) & mask for i in range(2 * N)]
    return [(ct[i] - ct[N + i]) % M for i in range(N)]


@pytest.mark.parametrize("N,logQ", [(64, 128), (1024, 128), (4096, 218)])
def test_p6_kronecker(N, logQ):
    g = synth.rng(60 + N)
    Q = 1 << logQ
    a = synth.uniform_big(g, N, logQ)
    b = synth.uniform_big(g, N, logQ)
    want = _kronecker(a, b, Q)
    assert ring.pm_ntt(a, b, Q) == want
    if N <= 1024:
        assert ring.pm_schoolbook(a, b, Q) == want       # schoolbook vs its NTT at N <= 2^10
    for k in (0, N // 2, N - 1):
        assert ring.pm_coeff(a, b, k, Q) == want[k]


# ---- P7: transforms and CRT ------------------------------------------------------------------
@pytest.mark.parametrize("N", [8, 64])
def test_p7_ntt_matches_eq8_and_inverts(N):
    q = ntt.oracle_primes(N, 1 << 40)[1]
    assert q % (2 * N) == 1 and ntt.is_prime(q)
    psi = ntt.primitive_2n_root(q, N)
    assert pow(psi, N, q) == q - 1 and pow(psi, 2 * N, q) == 1
    rnd = random.Random(N)
    a = np.array([rnd.randrange(q) for _ in range(N)], dtype=np.uint64)
    fa = ntt.ntt_forward(a, q, psi)
    assert [int(v) for v in fa] == ntt.ntt_forward_direct(a, q, psi)          # Eq. 8 literally
    assert np.array_equal(ntt.ntt_inverse(fa, q, psi), a)                      # Eq. 9 inverts Eq. 8


def test_p7_ntt_roundtrip_large_and_convolution():
    N = 4096
    q = ntt.oracle_primes(N, 1)[0]
    psi = ntt.primitive_2n_root(q, N)
    g = synth.rng(7)
    a = g.integers(0, q, size=N, dtype=np.uint64)
    b = g.integers(0, q, size=N, dtype=np.uint64)
    assert np.array_equal(ntt.ntt_inverse(ntt.ntt_forward(a, q, psi), q, psi), a)
    c = ntt.ntt_inverse(ntt.ntt_forward(a, q, psi) * ntt.ntt_forward(b, q, psi) % np.uint64(q), q, psi)
    for k in (0, 17, N - 1):                                                   # Eq. 7 against Eq. 5-6
        assert int(c[k]) == ring.pm_coeff(a.tolist(), b.tolist(), k, q)


def test_p7_crt_roundtrip():
    primes = ntt.oracle_primes(64, 1 << 200)
    Mp = 1
    for q in primes:
        Mp *= q
    rnd = random.Random(9)
    xs = [rnd.randrange(Mp) for _ in range(5)] + [0, 1, Mp - 1]
    res = [np.array([x % q for x in xs], dtype=np.uint64) for q in primes]
    got, Mp2 = ring.crt_direct(res, primes)
    assert Mp2 == Mp and got == xs


def test_miller_rabin_small():
    sieve = [n for n in range(2, 2000) if all(n % d for d in range(2, int(n ** 0.5) + 1))]
    assert [n for n in range(2, 2000) if ntt.is_prime(n)] == sieve
    assert not ntt.is_prime(3215031751) and ntt.is_prime(2147483647)          # strong pseudoprime to 2,3,5,7


# ---- limbs -----------------------------------------------------------------------------------
def test_limb_packing():
    rnd = random.Random(1)
    xs = [rnd.randrange(1 << 218) for _ in range(16)] + [0, (1 << 218) - 1]
    arr = to_limbs(xs, 7)
    assert arr.shape == (7, 18) and arr.dtype == np.uint32
    assert from_limbs(arr) == xs
    assert int(arr[0, -1]) == 0xFFFFFFFF and int(arr[6, -1]) == (1 << (218 - 192)) - 1
    g = synth.rng(5)
    u = synth.uniform_limbs(g, (2,), 8, 218)
    assert u.shape == (2, 7, 8) and int(u[:, 6].max()) < (1 << 26)


# ---- moduli ----------------------------------------------------------------------------------
def test_bgv_modulus_c4():
    g = _read_golden("moduli.txt")
    t, lg, off = g["t"][0], g["log"][0], g["offset"][0]
    Q = scheme.make_modulus(lg, t)
    assert Q == (1 << lg) + off and Q % 2 == 1 and Q % t == 1
    assert all(not (c % 2 == 1 and c % t == 1) for c in range((1 << lg) + 1, Q))
    prm = scheme.Params(1 << 14, 437, 437, t)
    assert prm.P == prm.Q and prm.L == 14 and prm.L_PQ == 28
    assert scheme.Params(1 << 16, 1240, 1240).L == 39 and scheme.Params(1 << 16, 1240, 1240).L_PQ == 78


# ---- R1: rescale rounding interval -----------------------------------------------------------------
def test_r1_rescale_interval():
    prm = scheme.Params(16, 128, 128)
    g = synth.rng(11)
    ct = (synth.uniform_big(g, 16, 128), synth.uniform_big(g, 16, 128))
    ct[0][0] = 0
    ct[0][1] = (1 << 128) - 1
    ct[0][2] = 1 << 39
    ct[0][3] = (1 << 39) - 1
    for p in (1, 40, 127):
        out = scheme.rescale(prm, ct, p)
        Q2 = 1 << (128 - p)
        for comp_in, comp_out in zip(ct, out):
            for c, cp in zip(comp_in, comp_out):
                assert 0 <= cp < Q2
                # cp = round(c / 2^p) mod Q2 with ties up: 2^p cp - c in (-2^(p-1), 2^(p-1)] mod 2^logQ
                diff = ring.centre((cp << p) - c, 1 << 128)
                assert -(1 << (p - 1)) < diff <= (1 << (p - 1))
    assert scheme.rescale(prm, ([1 << 39] + [0] * 15, [0] * 16), 40)[0][0] == 1      # tie rounds up
    assert scheme.rescale(prm, ([(1 << 39) - 1] + [0] * 15, [0] * 16), 40)[0][0] == 0


# ---- harness: encode / decode ------------------------------------------------------------------
def test_encode_decode_roundtrip_and_homomorphism():
    N, D = 256, float(1 << 40)
    g = synth.rng(21)
    z1, z2 = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
    assert np.abs(z1).max() <= 1.0
    m1, m2 = harness.encode(z1, N, D), harness.encode(z2, N, D)
    assert np.abs(harness.decode(m1, N, D) - z1).max() < 1e-9
    # direct evaluation of m(zeta_j) for one slot (kernel of Eq. 10)
    j = 5
    zeta = np.exp(1j * np.pi * (2 * j + 1) / N)
    direct = sum(int(m1[k]) * zeta ** k for k in range(N)) / D
    assert abs(direct - z1[j]) < 1e-9
    big = 1 << 200
    prod = [ring.centre(v, big) for v in ring.pm_schoolbook(m1, m2, big)]
    assert np.abs(harness.decode(prod, N, D * D) - z1 * z2).max() < 1e-8


def test_pm_sparse_matches_definition():
    N, Q = 64, 1 << 77
    g = synth.rng(31)
    a = synth.uniform_big(g, N, 77)
    s = [int(v) for v in synth.ternary_hwt(g, N, 9)]
    assert harness.pm_sparse(a, s, Q) == ring.pm_schoolbook(a, [v % Q for v in s], Q)
    assert sum(1 for v in s if v) == 9 and set(s) <= {-1, 0, 1}


# ---- R2/R3/R5: CKKS ----------------------------------------------------------------------------
def _ckks_setup(N, logQ, logP, seed, hwt):
    prm = scheme.Params(N, logQ, logP)
    g = synth.rng(seed)
    s, evk = harness.keygen(prm, g, hwt=hwt)
    D = float(1 << 40)
    z1, z2 = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
    ct1 = harness.encrypt(prm, g, s, harness.encode(z1, N, D))
    ct2 = harness.encrypt(prm, g, s, harness.encode(z2, N, D))
    return prm, s, evk, z1, z2, ct1, ct2, D


def test_r3_ckks_end_to_end_config1():
    """BASELINE.json configs[0]: N=2^10, Q=P=2^128, Delta=2^40, HWT 64, sigma 3.2, seed 0."""
    N = 1 << 10
    prm, s, evk, z1, z2, ct1, ct2, D = _ckks_setup(N, 128, 128, 0, 64)
    assert np.abs(harness.decode(harness.decrypt(ct1, s, prm.Q), N, D) - z1).max() < 1e-6
    d = scheme.he_mult(prm, ct1, ct2)
    # tensor triple decrypts to the product of the two decryptions (exact ring identity)
    mu1 = harness.decrypt(ct1, s, prm.Q)
    mu2 = harness.decrypt(ct2, s, prm.Q)
    assert harness.decrypt3(d, s, prm.Q) == [ring.centre(v, prm.Q) for v in ring.pm(mu1, mu2, prm.Q)]
    r = scheme.relinearize(prm, d, evk)
    # R2: relinearisation changes the decryption only by a small error
    err = [ring.centre(x - y, prm.Q) for x, y in zip(harness.decrypt(r, s, prm.Q), harness.decrypt3(d, s, prm.Q))]
    assert max(abs(e) for e in err) < (1 << 20)
    out = scheme.rescale(prm, r, 40)
    got = harness.decode(harness.decrypt(out, s, prm.Q >> 40), N, D)
    assert np.abs(got - z1 * z2).max() <= 2.0 ** -20                         # north_star bound


def test_r5_degenerate_relin_ckks():
    N = 64
    prm = scheme.Params(N, 96, 96)
    g = synth.rng(55)
    d0, d1, d2 = (synth.uniform_big(g, N, 96) for _ in range(3))
    s = [int(v) for v in synth.ternary_hwt(g, N, 8)]
    zero = [0] * N
    evk_rand = (synth.uniform_big(g, N, 192), synth.uniform_big(g, N, 192))
    assert scheme.relinearize(prm, (d0, d1, zero), evk_rand) == (d0, d1)      # d2 = 0
    s2 = ring.pm([v % prm.PQ for v in s], [v % prm.PQ for v in s], prm.PQ)
    evk0 = ([(prm.P * v) % prm.PQ for v in s2], zero)                         # e' = 0, a' = 0
    o0, o1 = scheme.relinearize(prm, (d0, d1, d2), evk0)
    d2s2 = ring.pm(d2, [v % prm.Q for v in s2], prm.Q)
    assert o0 == ring.add(d0, d2s2, prm.Q) and o1 == d1                       # k_b = d2 s^2 exactly


# ---- R4/R5: BGV --------------------------------------------------------------------------------
@pytest.mark.parametrize("N,logQ,t,hwt", [(64, 80, 257, 16), (256, 120, 65537, None)])
def test_r4_bgv_exact(N, logQ, t, hwt):
    prm = scheme.Params(N, logQ, logQ, t)
    assert prm.Q % t == 1 and prm.Q % 2 == 1 and prm.P == prm.Q
    g = synth.rng(77 + N)
    s, evk = harness.keygen(prm, g, hwt=hwt)
    m1 = [int(v) for v in synth.uniform_mod(g, N, t)]
    m2 = [int(v) for v in synth.uniform_mod(g, N, t)]
    ct1, ct2 = harness.encrypt(prm, g, s, m1), harness.encrypt(prm, g, s, m2)
    assert harness.decrypt_bgv(ct1, s, prm) == m1
    d = scheme.he_mult(prm, ct1, ct2)
    want = ring.pm(m1, m2, t)
    assert [v % t for v in harness.decrypt3(d, s, prm.Q)] == want
    r = scheme.relinearize(prm, d, evk)
    assert harness.decrypt_bgv(r, s, prm) == want                             # exact mod t
    # R2: the switch error is a multiple of t and small
    err = [ring.centre(x - y, prm.Q) for x, y in zip(harness.decrypt(r, s, prm.Q), harness.decrypt3(d, s, prm.Q))]
    assert all(e % t == 0 for e in err) and max(abs(e) for e in err) < t * N * 64
    zero = [0] * N
    assert scheme.relinearize(prm, (d[0], d[1], zero), evk) == (d[0], d[1])


# ---- NEXT-1: coefficient-wise operations and the level drop (parity unpinned by the paper: names only) --------------------
def test_next1_elementwise_ops_are_the_ring_operations_and_decrypt_homomorphically():
    """ct_add / ct_sub / ct_negate: group laws on random data, and Dec(add) = Dec(ct1) + Dec(ct2) mod Q exactly (the
    decryption map c0 + c1 s is linear); BGV: plaintexts add mod t.  moddown: Dec(moddown(ct)) = Dec(ct) mod 2^logq'."""
    import numpy as np
    import synth
    from oracle import harness, scheme
    N, logQ, logP = 64, 100, 100
    prm = scheme.Params(N, logQ, logP, 0)
    g = synth.rng(31)
    s, _ = harness.keygen(prm, g, hwt=16)
    z1, z2 = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
    ct1 = harness.encrypt(prm, g, s, harness.encode(z1, N, 2.0 ** 30))
    ct2 = harness.encrypt(prm, g, s, harness.encode(z2, N, 2.0 ** 30))
    Q = prm.Q
    add, sub, neg = scheme.ct_add(prm, ct1, ct2), scheme.ct_sub(prm, ct1, ct2), scheme.ct_negate(prm, ct2)
    assert scheme.ct_sub(prm, add, ct2) == tuple(list(a) for a in ct1)
    assert scheme.ct_add(prm, ct1, neg) == sub
    assert scheme.ct_add(prm, ct2, neg) == tuple([0] * N for _ in range(2))
    d1, d2 = harness.decrypt(ct1, s, Q), harness.decrypt(ct2, s, Q)
    assert [x % Q for x in harness.decrypt(add, s, Q)] == [(a + b) % Q for a, b in zip(d1, d2)]
    assert np.max(np.abs(harness.decode(harness.decrypt(add, s, Q), N, 2.0 ** 30) - (z1 + z2))) < 1e-6
    assert np.max(np.abs(harness.decode(harness.decrypt(sub, s, Q), N, 2.0 ** 30) - (z1 - z2))) < 1e-6
    low = scheme.moddown(prm, ct1, 70)
    assert all(0 <= x < (1 << 70) for a in low for x in a)
    assert [x % (1 << 70) for x in harness.decrypt(low, s, 1 << 70)] == [x % (1 << 70) for x in d1]
    assert np.max(np.abs(harness.decode(harness.decrypt(low, s, 1 << 70), N, 2.0 ** 30) - z1)) < 1e-6
    # BGV: exact mod t
    prb = scheme.Params(N, 60, 60, 257)
    sb, _ = harness.keygen(prb, g, hwt=None)
    m1 = [int(v) for v in g.integers(0, 257, size=N)]
    m2 = [int(v) for v in g.integers(0, 257, size=N)]
    c1, c2 = harness.encrypt(prb, g, sb, m1), harness.encrypt(prb, g, sb, m2)
    assert harness.decrypt_bgv(scheme.ct_add(prb, c1, c2), sb, prb) == [(a + b) % 257 for a, b in zip(m1, m2)]
    assert harness.decrypt_bgv(scheme.ct_sub(prb, c1, c2), sb, prb) == [(a - b) % 257 for a, b in zip(m1, m2)]
    assert harness.decrypt_bgv(scheme.ct_negate(prb, c1), sb, prb) == [(-a) % 257 for a in m1]


# ---- NEXT-2: automorphism, rotation key switch (parity unpinned by the paper: names only) ---------------------------------
def test_next2_automorphism_is_the_substitution_and_rotation_permutes_the_slots():
    import numpy as np
    import synth
    from oracle import harness, ring, scheme
    N, M = 16, 97
    g = synth.rng(41)
    a = [int(v) for v in g.integers(0, M, size=N)]
    b = [int(v) for v in g.integers(0, M, size=N)]
    # sigma_k(X) = X^k reduced mod X^N + 1; sigma_1 = id; sigma_k sigma_j = sigma_{kj}; ring homomorphism
    X = [0, 1] + [0] * (N - 2)
    for k in (3, 5, 2 * N - 1):
        want = [0] * N
        want[k % N] = 1 if k < N else M - 1
        assert scheme.automorphism(X, k, M) == want
        assert scheme.automorphism(ring.pm(a, b, M), k, M) == ring.pm(scheme.automorphism(a, k, M), scheme.automorphism(b, k, M), M)
    assert scheme.automorphism(a, 1, M) == a
    assert scheme.automorphism(scheme.automorphism(a, 3, M), 5, M) == scheme.automorphism(a, 15, M)
    # direct evaluation: (sigma_k a)(x) = a(x^k) at a root of X^N + 1 mod 97 (x = 19^3 has order 32 = 2N)
    x = next(v for v in range(2, M) if pow(v, N, M) == M - 1)
    ev = lambda p, y: sum(c * pow(y, i, M) for i, c in enumerate(p)) % M
    assert ev(scheme.automorphism(a, 5, M), x) == ev(a, pow(x, 5, M))
    # end to end on CKKS: Dec(rotate(ct)) decodes to the permuted (and, for k = 2N - 1, conjugated) slots
    N, logQ, logP = 64, 100, 100
    prm = scheme.Params(N, logQ, logP, 0)
    s, _ = harness.keygen(prm, g, hwt=16)
    z = synth.unit_disk(g, N // 2)
    ct = harness.encrypt(prm, g, s, harness.encode(z, N, 2.0 ** 30))
    for k in (5, 25, 2 * N - 1):
        rk = harness.rotkeygen(prm, g, s, k)
        out = scheme.rotate(prm, ct, k, rk)
        got = harness.decode(harness.decrypt(out, s, prm.Q), N, 2.0 ** 30)
        src, conj = harness.slot_image(N, k)
        want = np.array([np.conj(z[i]) if c else z[i] for i, c in zip(src, conj)])
        assert np.max(np.abs(got - want)) < 1e-6
    src, conj = harness.slot_image(N, 2 * N - 1)
    assert src == list(range(N // 2)) and all(conj)
    # BGV: the plaintext polynomial is mapped by the same automorphism, exactly mod t
    prb = scheme.Params(N, 60, 60, 257)
    sb, _ = harness.keygen(prb, g, hwt=None)
    m = [int(v) for v in g.integers(0, 257, size=N)]
    cb = harness.encrypt(prb, g, sb, m)
    rkb = harness.rotkeygen(prb, g, sb, 5)
    assert harness.decrypt_bgv(scheme.rotate(prb, cb, 5, rkb), sb, prb) == scheme.automorphism(m, 5, 257)


# ---- NEXT-3: ciphertext x plaintext (parity unpinned by the paper: names only) ---------------------------------------------
def test_next3_mult_plain_multiplies_the_slots_and_is_exact_mod_t():
    import numpy as np
    import synth
    from oracle import harness, ring, scheme
    g = synth.rng(43)
    N, logQ, logP = 64, 120, 120
    prm = scheme.Params(N, logQ, logP, 0)
    s, _ = harness.keygen(prm, g, hwt=16)
    z, w = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
    ct = harness.encrypt(prm, g, s, harness.encode(z, N, 2.0 ** 30))
    m = [v % prm.Q for v in harness.encode(w, N, 2.0 ** 30)]
    out = scheme.mult_plain(prm, ct, m)
    # linearity of decryption: Dec(out) = Dec(ct) * m exactly in the ring
    d = [v % prm.Q for v in harness.decrypt(ct, s, prm.Q)]
    assert [v % prm.Q for v in harness.decrypt(out, s, prm.Q)] == ring.pm(d, m, prm.Q)
    got = harness.decode(harness.decrypt(scheme.rescale(prm, out, 30), s, 1 << (logQ - 30)), N, 2.0 ** 30)
    assert np.max(np.abs(got - z * w)) < 1e-6
    # the constant polynomial 1 is the identity, 0 annihilates
    one = [1] + [0] * (N - 1)
    assert scheme.mult_plain(prm, ct, one) == (list(ct[0]), list(ct[1]))
    assert scheme.mult_plain(prm, ct, [0] * N) == ([0] * N, [0] * N)
    prb = scheme.Params(N, 60, 60, 257)
    sb, _ = harness.keygen(prb, g, hwt=None)
    m1 = [int(v) for v in g.integers(0, 257, size=N)]
    m2 = [int(v) for v in g.integers(0, 257, size=N)]
    cb = harness.encrypt(prb, g, sb, m1)
    assert harness.decrypt_bgv(scheme.mult_plain(prb, cb, m2), sb, prb) == ring.pm(m1, m2, 257)


def test_next1_mul_monomial_is_the_signed_rotation_and_multiplies_slots_by_powers_of_the_roots():
    import numpy as np
    import synth
    from oracle import harness, scheme
    N, logQ = 64, 100
    prm = scheme.Params(N, logQ, logQ, 0)
    g = synth.rng(47)
    a = [int(v) for v in g.integers(0, 1 << 62, size=N)]
    Q = prm.Q
    for k in (0, 1, N // 2, N - 1, N, N + 5, 2 * N - 1):
        got = scheme.mul_monomial(prm, (a,), k)[0]
        want = [0] * N
        for i, x in enumerate(a):                     # X^k X^i = +-X^((i + k) mod N)
            j = (i + k) % (2 * N)
            want[j % N] = x % Q if j < N else (-x) % Q
        assert got == want
    # slots: (X^k m)(zeta_j) = zeta_j^k m(zeta_j); k = N/2 gives zeta_j^(N/2) = exp(i pi (2j+1)/2) = i (-1)^j
    s, _ = harness.keygen(prm, g, hwt=16)
    z = synth.unit_disk(g, N // 2)
    ct = harness.encrypt(prm, g, s, harness.encode(z, N, 2.0 ** 30))
    out = scheme.mul_monomial(prm, ct, N // 2)
    got = harness.decode(harness.decrypt(out, s, Q), N, 2.0 ** 30)
    want = np.array([1j * (-1) ** j * z[j] for j in range(N // 2)])
    assert np.max(np.abs(got - want)) < 1e-6


def test_next3_add_plain_and_mult_scalar_are_linear_under_decryption():
    """add_plain: Dec(ct + m) = Dec(ct) + m exactly mod Q (CKKS: slots add; BGV: plaintexts add mod t).  mult_scalar:
    k = 3 equals ct + ct + ct (the pinned ct_add), k = -1 the pinned ct_negate, k = 0 the zero ciphertext, Dec scales by k;
    both agree with the ring product by the constant polynomial (pm, pinned by P1-P4)."""
    import numpy as np
    import synth
    from oracle import harness, scheme
    from oracle.ring import pm
    N, logQ = 64, 100
    prm = scheme.Params(N, logQ, logQ, 0)
    g = synth.rng(37)
    s, _ = harness.keygen(prm, g, hwt=16)
    z1, z2 = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
    Q = prm.Q
    ct = harness.encrypt(prm, g, s, harness.encode(z1, N, 2.0 ** 30))
    m = [x % Q for x in harness.encode(z2, N, 2.0 ** 30)]
    ap = scheme.add_plain(prm, ct, m)
    d = harness.decrypt(ct, s, Q)
    assert [x % Q for x in harness.decrypt(ap, s, Q)] == [(a + b) % Q for a, b in zip(d, m)]
    assert np.max(np.abs(harness.decode(harness.decrypt(ap, s, Q), N, 2.0 ** 30) - (z1 + z2))) < 1e-6
    assert list(ap[1]) == list(ct[1])
    three = scheme.mult_scalar(prm, ct, 3)
    assert three == scheme.ct_add(prm, scheme.ct_add(prm, ct, ct), ct)
    assert scheme.mult_scalar(prm, ct, -1) == scheme.ct_negate(prm, ct)
    assert scheme.mult_scalar(prm, ct, 0) == tuple([0] * N for _ in range(2))
    for k in (7, -5, 2 ** 31 - 1, -(2 ** 31 - 1)):
        got = scheme.mult_scalar(prm, ct, k)
        const = [k % Q] + [0] * (N - 1)
        assert got == tuple(pm(a, const, Q) for a in ct)
        assert [x % Q for x in harness.decrypt(got, s, Q)] == [(x * k) % Q for x in d]
    assert np.max(np.abs(harness.decode(harness.decrypt(scheme.mult_scalar(prm, ct, -5), s, Q), N, 2.0 ** 30) + 5 * z1)) < 1e-5
    # BGV: exact mod t
    prb = scheme.Params(N, 60, 60, 257)
    sb, _ = harness.keygen(prb, g, hwt=None)
    m1 = [int(v) for v in g.integers(0, 257, size=N)]
    m2 = [int(v) for v in g.integers(0, 257, size=N)]
    c1 = harness.encrypt(prb, g, sb, m1)
    assert harness.decrypt_bgv(scheme.add_plain(prb, c1, m2), sb, prb) == [(a + b) % 257 for a, b in zip(m1, m2)]
    assert harness.decrypt_bgv(scheme.mult_scalar(prb, c1, 11), sb, prb) == [(a * 11) % 257 for a in m1]
    assert harness.decrypt_bgv(scheme.mult_scalar(prb, c1, -3), sb, prb) == [(-3 * a) % 257 for a in m1]
    assert scheme.mult_scalar(prb, c1, 3) == scheme.ct_add(prb, scheme.ct_add(prb, c1, c1), c1)


# ---- hand-worked pins of the rounding readings (tests/golden/relin_hand.txt) ---------------------------------------------
# The paper prints no formula for the divide-by-P of the key switch or for the BGV level drop;
# the readings are DESIGN.md 3 A3 / A10 / A20.  These values are worked out by hand in the golden file's comments, and a
# plausible mistake in each reading (truncation instead of round-half-up; r or k left un-centred) fails one of them.
def test_hand_ckks_divide_by_p_rounds_half_up():
    gold = _read_golden("relin_hand.txt")
    N, logQ, logP = gold["ckks_relin_params"]
    prm = scheme.Params(N, logQ, logP)
    zero, one = [0] * N, [1] + [0] * (N - 1)
    out = scheme.relinearize_ckks(prm, (zero, zero, one), (gold["ckks_relin_evk_b"], zero))   # x_b = b' itself
    assert out == (gold["ckks_relin_k_b"], zero)
    # the same through relinearize(), with d0 / d1 carried along mod Q
    d0, d1 = [15, 15, 1, 3], [2, 0, 9, 15]
    want0 = [(a + b) % prm.Q for a, b in zip(d0, gold["ckks_relin_k_b"])]
    assert scheme.relinearize(prm, (d0, d1, one), (gold["ckks_relin_evk_b"], zero)) == (want0, d1)


def test_hand_bgv_divide_by_p_centres_r_and_k():
    gold = _read_golden("relin_hand.txt")
    t, P, Q = gold["bgv_div_params"]
    assert scheme.make_modulus(4, t) == P == Q
    Pinv_t = pow(P % t, -1, t)
    got = [scheme._div_p_bgv(x, P, Q, t, Pinv_t) for x in gold["bgv_div_x"]]
    assert got == gold["bgv_div_out"]
    # through relinearize_bgv: N = 4, d2 = 1, so x_b = b', x_a = a' coefficient by coefficient
    prm = scheme.Params(4, 4, 4, t)
    xs, outs = gold["bgv_div_x"], gold["bgv_div_out"]
    zero, one = [0] * 4, [1, 0, 0, 0]
    assert scheme.relinearize_bgv(prm, (zero, zero, one), (xs[:4], xs[4:])) == (outs[:4], outs[4:])


def test_hand_bgv_modswitch_and_its_invariants():
    gold = _read_golden("relin_hand.txt")
    t, logQ, new_logQ = gold["bgv_modswitch_params"]
    prm = scheme.Params(4, logQ, logQ, t)
    cs, outs = gold["bgv_modswitch_c"], gold["bgv_modswitch_out"]
    for i in range(0, len(cs) - 3, 4):
        assert scheme.modswitch_bgv(prm, (cs[i:i + 4], cs[i:i + 4]), new_logQ) == (outs[i:i + 4], outs[i:i + 4])
    assert scheme.modswitch_bgv(prm, ([cs[-1]] * 4, [0] * 4), new_logQ) == ([outs[-1]] * 4, [0] * 4)
    # invariants at a larger size, every c: some representative c' + j Q' (|j| <= 1) is within (1 + t)/2 of c Q'/Q and is
    # = c (mod t) (Q = Q' = 1 mod t and the removed delta is a multiple of t)
    t, logQ, new_logQ = 257, 20, 13
    prm = scheme.Params(4, logQ, logQ, t)
    Q, Q2 = prm.Q, scheme.make_modulus(new_logQ, t)
    rnd = random.Random(4)
    for c in [0, 1, Q - 1, Q // 2, Q // 2 + 1] + [rnd.randrange(Q) for _ in range(300)]:
        cp = scheme.modswitch_bgv(prm, ([c] * 4, [c] * 4), new_logQ)[0][0]
        assert 0 <= cp < Q2
        assert any((cp + j * Q2 - c) % t == 0 and abs((cp + j * Q2) * Q - c * Q2) <= Q * (1 + t) // 2 for j in (-1, 0, 1))


@pytest.mark.parametrize("N,logQ,new_logQ,t,hwt", [(64, 120, 80, 257, 16), (256, 200, 120, 65537, None)])
def test_next4_modswitch_keeps_the_plaintext_and_shrinks_the_noise(N, logQ, new_logQ, t, hwt):
    """R4 for the level drop: Dec_Q'(modswitch(ct)) = m exactly mod t, the noise drops by about Q/Q', and a product formed
    and relinearised at the lower level still decrypts exactly (the evk there is generated for Q')."""
    prm = scheme.Params(N, logQ, logQ, t)
    g = synth.rng(N + t)
    s, evk = harness.keygen(prm, g, hwt=hwt)
    m1 = [int(v) for v in synth.uniform_mod(g, N, t)]
    m2 = [int(v) for v in synth.uniform_mod(g, N, t)]
    ct1, ct2 = harness.encrypt(prm, g, s, m1), harness.encrypt(prm, g, s, m2)
    prod = scheme.relinearize(prm, scheme.he_mult(prm, ct1, ct2), evk)
    assert harness.decrypt_bgv(prod, s, prm) == ring.pm(m1, m2, t)
    noise_hi = max(abs(v) for v in harness.decrypt(prod, s, prm.Q))
    low = scheme.modswitch_bgv(prm, prod, new_logQ)
    prm2 = scheme.Params(N, new_logQ, new_logQ, t)
    assert all(0 <= c < prm2.Q for comp in low for c in comp)
    assert harness.decrypt_bgv(low, s, prm2) == ring.pm(m1, m2, t)
    noise_lo = max(abs(v) for v in harness.decrypt(low, s, prm2.Q))
    assert noise_lo < (noise_hi >> (logQ - new_logQ - 1)) + t * (N + 1)
    # continue at the lower level: fresh key for Q', multiply by a switched fresh ciphertext
    g2 = synth.rng(N + t + 1)
    e2 = synth.gaussian_error(g2, N)
    a2 = synth.uniform_big(g2, N, (prm2.PQ - 1).bit_length() - 1)
    s2 = ring.pm([v % prm2.PQ for v in s], [v % prm2.PQ for v in s], prm2.PQ)
    a_s = harness.pm_secret(a2, s, prm2.PQ)
    evk2 = ([(-x + t * int(e) + prm2.P * y) % prm2.PQ for x, e, y in zip(a_s, e2, s2)], a2)
    m3 = [int(v) for v in synth.uniform_mod(g2, N, t)]
    ct3 = scheme.modswitch_bgv(prm, harness.encrypt(prm, g2, s, m3), new_logQ)
    assert harness.decrypt_bgv(ct3, s, prm2) == m3
    out = scheme.relinearize(prm2, scheme.he_mult(prm2, low, ct3), evk2)
    assert harness.decrypt_bgv(out, s, prm2) == ring.pm(ring.pm(m1, m2, t), m3, t)
