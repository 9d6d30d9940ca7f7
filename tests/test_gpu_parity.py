"""GPU parity: the CUDA path (through the C ABI, via the thin binding) against the CPU oracle, bit-exact.

Everything on the hot path is integer, so the bar is equality of every limb (BASELINE.json north_star).
Inputs are seeded and synthetic (synth/), shaped like the paper's workloads: random ciphertexts,
cnum per tensor, logN, logQ.  Full-size configs are checked on sampled coefficients that the oracle computes one
by one from the definition (Eq. 5-6), small ones element by element.
"""
import numpy as np
import pytest

import synth
from oracle import harness, ntt as ontt, ring, scheme
from oracle.limbs import from_limbs, to_limbs

pytestmark = pytest.mark.gpu

torch = pytest.importorskip("torch")

from gpu_util import coeff_from_limbs, limbs_np_to_tensor, polys_to_tensor, tensor_to_np, tensor_to_polys  # noqa: E402


def _lib():
    import paper_2607_05920_b200 as fhe
    return fhe


def _bitrev(i, bits):
    r = 0
    for b in range(bits):
        r |= ((i >> b) & 1) << (bits - 1 - b)
    return r


# ---- S1: decompose ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,logQ,Lin,mask", [(1024, 128, 4, 0), (1024, 128, 8, 0), (4096, 620, 20, 620), (256, 1240, 78, 0)])
def test_decompose_matches_python_mod(N, logQ, Lin, mask):
    fhe = _lib()
    ctx = fhe.Context(N, logQ, logQ)
    g = synth.rng(11)
    limbs = synth.uniform_limbs(g, (2,), N, 32 * Lin)
    K = ctx.K2
    q, _ = ctx.primes(K)
    res = tensor_to_np(ctx.fhe_debug_decompose(limbs_np_to_tensor(limbs), K, mask))
    for p in range(2):
        vals = from_limbs(limbs[p])
        if mask:
            vals = [v % (1 << mask) for v in vals]
        for j in (0, 1, K // 2, K - 1):
            want = np.array([v % q[j] for v in vals], dtype=np.uint32)
            assert np.array_equal(res[p, j], want), (p, j)


# ---- S2 / S4: NTT against the oracle's Eq. 8 with the library's own (q, psi) -----------------------------------
@pytest.mark.parametrize("N", [256, 1024, 8192, 16384, 65536])
def test_ntt_forward_is_eq8_bitreversed_and_inverse_roundtrips(N):
    fhe = _lib()
    ctx = fhe.Context(N, 64, 64)
    K = min(3, ctx.K2)
    q, psi = ctx.primes(K)
    g = synth.rng(5)
    x = np.stack([g.integers(0, q[j], size=N, dtype=np.uint64).astype(np.uint32) for j in range(K)])[None]
    d = limbs_np_to_tensor(x.copy())
    ctx.fhe_debug_ntt(d, False)
    f = tensor_to_np(d)
    bits = N.bit_length() - 1
    rev = np.array([_bitrev(i, bits) for i in range(N)])
    for j in range(K):
        want = ontt.ntt_forward(x[0, j].astype(np.uint64), q[j], psi[j])   # natural order, Eq. 8
        assert np.array_equal(f[0, j][rev].astype(np.uint64), want), j
    ctx.fhe_debug_ntt(d, True)
    assert np.array_equal(tensor_to_np(d), x)


# ---- fhe_polymul ---------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("N,logQ,batch", [(256, 64, 3), (1024, 128, 2), (1024, 218, 2), (2048, 61, 1)])
def test_polymul_small_full(N, logQ, batch):
    fhe = _lib()
    ctx = fhe.Context(N, logQ, 32)
    g = synth.rng(100 + N + logQ)
    a = synth.uniform_limbs(g, (batch,), N, logQ)
    b = synth.uniform_limbs(g, (batch,), N, logQ)
    out = tensor_to_np(ctx.fhe_polymul(limbs_np_to_tensor(a), limbs_np_to_tensor(b)))
    for i in range(batch):
        want = ring.pm(from_limbs(a[i]), from_limbs(b[i]), 1 << logQ)
        assert from_limbs(out[i]) == want


def test_polymul_extremes_all_q_minus_1_and_zero():
    """P5 closed form (a = b = Q-1 everywhere reaches both ends of the CRT range) and the zero polynomial."""
    fhe = _lib()
    N, logQ = 1024, 218
    ctx = fhe.Context(N, logQ, 32)
    Q = 1 << logQ
    a = to_limbs([Q - 1] * N, ctx.L)[None]
    z = np.zeros_like(a)
    out = tensor_to_np(ctx.fhe_polymul(limbs_np_to_tensor(a), limbs_np_to_tensor(a)))
    assert from_limbs(out[0]) == [(2 * k + 2 - N) % Q for k in range(N)]
    out = tensor_to_np(ctx.fhe_polymul(limbs_np_to_tensor(a), limbs_np_to_tensor(z)))
    assert not out.any()


def test_polymul_c2_shape():
    """configs[1]: N = 2^13, 218-bit coefficients (7 limbs), a slice of the batch of 64 checked in full against the
    oracle's own NTT route, the rest on sampled coefficients from the definition."""
    fhe = _lib()
    N, logQ, batch = 1 << 13, 218, 64
    ctx = fhe.Context(N, logQ, 32)
    assert ctx.L == 7
    g = synth.rng(2)
    a = synth.uniform_limbs(g, (batch,), N, logQ)
    b = synth.uniform_limbs(g, (batch,), N, logQ)
    out = tensor_to_np(ctx.fhe_polymul(limbs_np_to_tensor(a), limbs_np_to_tensor(b)))
    Q = 1 << logQ
    for i in (0, 63):
        assert from_limbs(out[i]) == ring.pm(from_limbs(a[i]), from_limbs(b[i]), Q)
    rnd = np.random.default_rng(7)
    for i in range(1, 63, 5):
        ai, bi = from_limbs(a[i]), from_limbs(b[i])
        for k in [0, N - 1] + [int(v) for v in rnd.integers(0, N, size=3)]:
            assert coeff_from_limbs(out[i], k) == ring.pm_coeff(ai, bi, k, Q)


# ---- configs[0]: tiny CKKS, every limb, plus the decryption bound -----------------------------------------------------
def _ckks_setup(N, logQ, logP, B, seed, delta_bits=40):
    prm = scheme.Params(N, logQ, logP, 0)
    g = synth.rng(seed)
    s, evk = harness.keygen(prm, g, hwt=64)
    cts1, cts2, zs = [], [], []
    for _ in range(B):
        z1, z2 = synth.unit_disk(g, N // 2), synth.unit_disk(g, N // 2)
        cts1.append(harness.encrypt(prm, g, s, harness.encode(z1, N, 2.0 ** delta_bits)))
        cts2.append(harness.encrypt(prm, g, s, harness.encode(z2, N, 2.0 ** delta_bits)))
        zs.append((z1, z2))
    return prm, s, evk, cts1, cts2, zs


def test_c1_tiny_ckks_full_pipeline():
    fhe = _lib()
    N, logQ, logP, B = 1 << 10, 128, 128, 2
    prm, s, evk, cts1, cts2, zs = _ckks_setup(N, logQ, logP, B, seed=0)
    ctx = fhe.Context(N, logQ, logP)
    assert (ctx.L, ctx.L_PQ) == (4, 8)
    ctx.fhe_set_evk(polys_to_tensor(list(evk), ctx.L_PQ))
    d1, d2 = polys_to_tensor(cts1, ctx.L), polys_to_tensor(cts2, ctx.L)
    d3 = ctx.fhe_he_mult(d1, d2)
    want3 = [scheme.he_mult(prm, cts1[i], cts2[i]) for i in range(B)]
    assert tensor_to_polys(d3) == [[list(p) for p in w] for w in want3]
    r2 = ctx.fhe_relinearize(d3)
    want2 = [scheme.relinearize(prm, want3[i], evk) for i in range(B)]
    assert tensor_to_polys(r2) == [[list(p) for p in w] for w in want2]
    rs = ctx.fhe_rescale(r2, 40)
    wantr = [scheme.rescale(prm, want2[i], 40) for i in range(B)]
    got_rs = tensor_to_polys(rs)
    assert got_rs == [[list(p) for p in w] for w in wantr]
    fused = ctx.fhe_mult_relin_rescale(d1, d2, 40)
    assert torch.equal(fused, rs)
    # decryption bound (north_star): |decode(Dec(.)) - z z'| <= 2^-20 at Delta = 2^40, from the GPU ciphertext
    for i in range(B):
        mu = harness.decrypt(tuple(got_rs[i]), s, 1 << (logQ - 40))
        z = harness.decode(mu, N, 2.0 ** 40)
        assert np.max(np.abs(z - zs[i][0] * zs[i][1])) <= 2.0 ** -20


@pytest.mark.parametrize("p_bits", [1, 31, 32, 33, 64, 127])
def test_rescale_shift_amounts(p_bits):
    fhe = _lib()
    N, logQ = 256, 128
    ctx = fhe.Context(N, logQ, 64)
    prm = scheme.Params(N, logQ, 64, 0)
    g = synth.rng(p_bits)
    ct = synth.uniform_limbs(g, (3, 2), N, logQ)
    ct[0, 0, :, :5] = 0xFFFFFFFF                     # all-ones coefficients: the rounding carry runs to the top
    got = tensor_to_polys(ctx.fhe_rescale(limbs_np_to_tensor(ct), p_bits))
    for i in range(3):
        want = scheme.rescale(prm, (from_limbs(ct[i, 0]), from_limbs(ct[i, 1])), p_bits)
        assert got[i] == [list(w) for w in want]
