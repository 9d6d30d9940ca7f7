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
@pytest.mark.parametrize("pipeline", [False, True])
@pytest.mark.parametrize("N,logQ,Lin,mask", [(1024, 128, 4, 0), (1024, 128, 8, 0), (4096, 620, 20, 620), (256, 1240, 78, 0),
                                             (512, 64, 2, 61), (2048, 256, 8, 250)])
def test_decompose_matches_python_mod(N, logQ, Lin, mask, pipeline):
    """pipeline = False: small shapes convert on the CUDA cores (kernels_small.cu), the others on the tensor-core pipeline;
    True: everything through the pipeline (mode 1 of fhe_debug_force_pipeline)."""
    fhe = _lib()
    ctx = fhe.Context(N, logQ, logQ)
    ctx.fhe_debug_force_pipeline(pipeline)
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


@pytest.mark.parametrize("Lin,mask", [(12, 0), (16, 0), (16, 500), (9, 0), (3, 70)])
def test_small_decompose_limb_bounds_and_largest_lazy_sums(Lin, mask):
    """The CUDA-core decompose keeps sum_l x_l (2^(32 l) mod q) lazily in 64 bits (kernels_small.cu): every limb bound it
    is instantiated for (2, 4, 8, 12, 16), with coefficients whose limbs are all 2^32 - 1 (the largest sums the folds
    must hold), all zero, and random, on every prime -- against Python's %."""
    fhe = _lib()
    N = 512
    ctx = fhe.Context(N, 96, 96)
    K = ctx.K2
    assert K * Lin <= 192                             # the small path takes it (fhe_internal.cuh: SMALL_WORK)
    g = synth.rng(100 + Lin)
    limbs = synth.uniform_limbs(g, (2,), N, 32 * Lin)
    limbs[0, :, :8] = 0xFFFFFFFF
    limbs[0, :, 8:12] = 0
    limbs[1, ::2, 16:24] = 0xFFFFFFFF                 # alternating all-ones / zero limbs
    limbs[1, 1::2, 16:24] = 0
    q, _ = ctx.primes(K)
    res = tensor_to_np(ctx.fhe_debug_decompose(limbs_np_to_tensor(limbs), K, mask))
    ctx.fhe_debug_force_pipeline(1)
    assert np.array_equal(res, tensor_to_np(ctx.fhe_debug_decompose(limbs_np_to_tensor(limbs), K, mask)))   # the tensor-core route agrees
    for p in range(2):
        vals = from_limbs(limbs[p])
        if mask:
            vals = [v % (1 << mask) for v in vals]
        for j in range(K):
            assert np.array_equal(res[p, j], np.array([v % q[j] for v in vals], dtype=np.uint32)), (p, j)


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
@pytest.mark.parametrize("pipeline", [False, True])
@pytest.mark.parametrize("N,logQ,batch", [(256, 64, 3), (1024, 128, 2), (1024, 218, 2), (2048, 61, 1), (512, 256, 2), (256, 33, 2)])
def test_polymul_small_full(N, logQ, batch, pipeline):
    fhe = _lib()
    ctx = fhe.Context(N, logQ, 32)
    ctx.fhe_debug_force_pipeline(pipeline)
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


@pytest.mark.parametrize("pipeline", [0, 1, 2])
def test_polymul_c2_shape(pipeline):
    """configs[1]: N = 2^13, 218-bit coefficients (7 limbs), a slice of the batch of 64 checked in full against the
    oracle's own NTT route, the rest on sampled coefficients from the definition."""
    fhe = _lib()
    N, logQ, batch = 1 << 13, 218, 64
    ctx = fhe.Context(N, logQ, 32)
    ctx.fhe_debug_force_pipeline(pipeline)
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


# ---- full-size configs: sampled coefficients from the definition ----------------------------------------------------
def _sample_ks(N, seed, count=4):
    rnd = np.random.default_rng(seed)
    return [0, N - 1] + [int(v) for v in rnd.integers(1, N - 1, size=count)]


def _check_he_mult_samples(out3, ct1, ct2, Q, ks):
    """out3: uint32 [3][L][N]; ct1/ct2: uint32 [2][L][N]."""
    c0, c1 = from_limbs(ct1[0]), from_limbs(ct1[1])
    e0, e1 = from_limbs(ct2[0]), from_limbs(ct2[1])
    for k in ks:
        assert coeff_from_limbs(out3[0], k) == ring.pm_coeff(c0, e0, k, Q), ("d0", k)
        assert coeff_from_limbs(out3[1], k) == (ring.pm_coeff(c0, e1, k, Q) + ring.pm_coeff(c1, e0, k, Q)) % Q, ("d1", k)
        assert coeff_from_limbs(out3[2], k) == ring.pm_coeff(c1, e1, k, Q), ("d2", k)


def _relin_coeff_ckks(prm, d3, evk_polys, k, d2=None):
    d2 = from_limbs(d3[2]) if d2 is None else d2
    out = []
    for comp in range(2):
        x = ring.pm_coeff(d2, evk_polys[comp], k, prm.PQ)
        kk = scheme.round_shift(x, prm.logP) % prm.Q
        out.append((coeff_from_limbs(d3[comp], k) + kk) % prm.Q)
    return out


def _relin_coeff_bgv(prm, d3, evk_polys, k):
    d2 = from_limbs(d3[2])
    Pinv_t = pow(prm.P % prm.t, -1, prm.t)
    out = []
    for comp in range(2):
        x = ring.pm_coeff(d2, evk_polys[comp], k, prm.PQ)
        kk = scheme._div_p_bgv(x, prm.P, prm.Q, prm.t, Pinv_t)
        out.append((coeff_from_limbs(d3[comp], k) + kk) % prm.Q)
    return out


def _structured_ks(N, item, n_items, polys_per_item, n_sm, per_item=72):
    """Coefficient positions chosen by the structure of the conversion pipeline, not by an RNG: the CRT launch walks the
    128-coefficient tiles of polynomial p = item * polys_per_item + comp, tile = p * N/128 + k/128, CTA = tile mod grid,
    and the CTA's tiles alternate between its two epilogue groups / accumulator sets.  Returned for one item: per_item
    residues k mod 128 (items take them in turn, so that the items of a batch together cover every k mod 128; each in a
    different tile), the first and last coefficient of the polynomial and of its first / last 256-point rows, and the
    tiles that are the first and the last tile CTA 0 and CTA grid-1 see in this item."""
    tpp = N // 128
    grid = min(n_items * polys_per_item * tpp, n_sm)
    ks = {0, 127, 128, 255, 256, N - 256, N - 129, N - 128, N - 1}
    for r in range(item * per_item, (item + 1) * per_item):
        ks.add(((r * 131 + item * 17) % tpp) * 128 + r % 128)
    for comp in range(polys_per_item):
        tiles = range((item * polys_per_item + comp) * tpp, (item * polys_per_item + comp + 1) * tpp)
        for cta in (0, grid - 1):
            mine = [t for t in tiles if t % grid == cta]
            for t, r in ((mine[0], 0), (mine[-1], 127)):
                ks.add((t % tpp) * 128 + r)
    return sorted(ks)


def _groups_hit(N, item, polys_per_item, n_items, n_sm, ks):
    """Which (epilogue group, k mod 128 half) combinations the positions reach, over the polynomials of the item."""
    tpp = N // 128
    grid = min(n_items * polys_per_item * tpp, n_sm)
    hit = set()
    for comp in range(polys_per_item):
        for k in ks:
            tile = (item * polys_per_item + comp) * tpp + k // 128
            hit.add(((tile // grid) & 1, tile % grid in (0, grid - 1)))
    return hit


@pytest.mark.parametrize("N,logQ,logP,B", [(1 << 15, 620, 620, 8), (1 << 16, 1240, 1240, 4)])
def test_ckks_full_size_every_limb_of_one_pair_and_structured_samples(N, logQ, logP, B):
    """configs[2] and configs[4] (the benchmarked shape, in the launch configuration bench.py times: the whole batch in one
    call).  Item 0 is a REAL encryption (HWT-64 secret, sigma = 3.2, Delta = 2^40) and is compared on every limb of every
    coefficient against the oracle's own NTT route for he_mult (d0, d1, d2), relinearize and rescale, then decrypted:
    the slot product within 2^-20.  The other items are uniform ciphertexts checked on positions chosen by the structure
    of the kernels (every k mod 128 over the batch, both CRT epilogue groups, first / last tiles of the first / last CTA,
    row boundaries; >= 512 in all), from the definition Eq. 5-6 one coefficient at a time.  The fused call must equal the
    three calls."""
    fhe = _lib()
    prm, s, evk, cts1, cts2, zs = _ckks_setup(N, logQ, logP, 1, seed=N)
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(N + logQ)
    ct1 = synth.uniform_limbs(g, (B, 2), N, logQ)
    ct2 = synth.uniform_limbs(g, (B, 2), N, logQ)
    ct1[0] = np.stack([to_limbs(p, ctx.L) for p in cts1[0]])
    ct2[0] = np.stack([to_limbs(p, ctx.L) for p in cts2[0]])
    ct1[1, 0, :, 0] = 0xFFFFFFFF                     # a coefficient with every stored bit set (masked on load)
    evk_np = np.stack([to_limbs(p, ctx.L_PQ) for p in evk])
    ctx.fhe_set_evk(limbs_np_to_tensor(evk_np))
    d1, d2 = limbs_np_to_tensor(ct1), limbs_np_to_tensor(ct2)
    t3 = ctx.fhe_he_mult(d1, d2)
    t2 = ctx.fhe_relinearize(t3)
    tr = ctx.fhe_rescale(t2, 40)
    fused = ctx.fhe_mult_relin_rescale(d1, d2, 40)
    assert torch.equal(fused, tr)
    out3, out2, outr = tensor_to_np(t3), tensor_to_np(t2), tensor_to_np(tr)
    # ---- item 0: every limb of every coefficient, against the oracle's own NTT route ----
    want3 = scheme.he_mult(prm, cts1[0], cts2[0])
    assert [from_limbs(out3[0, i]) for i in range(3)] == [list(p) for p in want3]
    want2 = scheme.relinearize(prm, want3, evk)
    assert [from_limbs(out2[0, i]) for i in range(2)] == [list(p) for p in want2]
    wantr = scheme.rescale(prm, want2, 40)
    gotr = [from_limbs(outr[0, i]) for i in range(2)]
    assert gotr == [list(p) for p in wantr]
    z = harness.decode(harness.decrypt(tuple(gotr), s, 1 << (logQ - 40)), N, 2.0 ** 40)
    assert np.max(np.abs(z - zs[0][0] * zs[0][1])) <= 2.0 ** -20
    # ---- the other items: positions chosen by structure, from the definition (one output polynomial per position, in
    # turn: a coefficient costs N big-integer products on the CPU) ----
    ct1m = ct1.copy()
    ct1m[..., ctx.L - 1, :] &= np.uint32((1 << (logQ % 32)) - 1) if logQ % 32 else np.uint32(0xFFFFFFFF)
    Q, Q2 = prm.Q, 1 << (logQ - 40)
    total, residues = 0, set()
    for b in range(1, B):
        ks3 = _structured_ks(N, b, B, 3, ctx.n_sm)
        assert _groups_hit(N, b, 3, B, ctx.n_sm, ks3) >= {(0, False), (1, False)}
        c0, c1 = from_limbs(ct1m[b, 0]), from_limbs(ct1m[b, 1])
        e0, e1 = from_limbs(ct2[b, 0]), from_limbs(ct2[b, 1])
        for n, k in enumerate(ks3):
            which = (n + b) % 3
            if which == 0:
                want = ring.pm_coeff(c0, e0, k, Q)
            elif which == 1:
                want = (ring.pm_coeff(c0, e1, k, Q) + ring.pm_coeff(c1, e0, k, Q)) % Q
            else:
                want = ring.pm_coeff(c1, e1, k, Q)
            assert coeff_from_limbs(out3[b, which], k) == want, (b, which, k)
        ks2 = _structured_ks(N, b, B, 2, ctx.n_sm)
        d2b = from_limbs(out3[b, 2])
        for n, k in enumerate(ks2):
            comp = (n + b) % 2
            x = ring.pm_coeff(d2b, evk[comp], k, prm.PQ)
            want = (coeff_from_limbs(out3[b, comp], k) + scheme.round_shift(x, logP)) % Q
            assert coeff_from_limbs(out2[b, comp], k) == want, (b, comp, k)
            assert coeff_from_limbs(outr[b, comp], k) == scheme.round_shift(want, 40) % Q2, (b, comp, k)
        total += len(ks3) + len(ks2)
        residues |= {k % 128 for k in ks3}
    assert total >= 512 and (B < 3 or len(residues) == 128)
    # R1 (any size): 2^p c' - c in (-2^(p-1), 2^(p-1)] mod Q, on every coefficient of every polynomial with numpy
    for b in range(B):
        for comp in range(2):
            lo_in = out2[b, comp, 0].astype(np.uint64) | (out2[b, comp, 1].astype(np.uint64) << np.uint64(32))
            lo_out = outr[b, comp, 0].astype(np.uint64)
            diff = ((lo_out << np.uint64(40)) - lo_in).astype(np.int64)     # low 64 bits suffice for the low-bit identity
            low40 = (lo_in & np.uint64((1 << 40) - 1)).astype(np.int64)
            expect = np.where(low40 >= (1 << 39), (1 << 40) - low40, -low40)
            assert np.array_equal(diff & ((1 << 62) - 1), expect & ((1 << 62) - 1))


# ---- the paper's own workload shape: cnum = 4, logN = 16, logQ = 1024, logp = 60 ----------------------
def test_paper_table1_shape_structured_samples_incl_rotation_and_plaintext_product():
    """The shape bench.py --table1 times: N = 2^16, Q = 2^1024 (32 whole limbs: logQ a multiple of 32 at full size), keys
    mod 2^2048, rescale by 2^60.  Uniform ciphertexts and keys (parity needs no decryption); every call the table times
    that runs the multiplication pipeline -- he_mult, relinearize, rescale, rotate (X -> X^5), conjugate (X -> X^(2N-1)),
    mult_plain -- is compared on positions chosen by the kernels' structure, from the definition Eq. 5-6 one coefficient
    at a time; the streaming operations are compared on every limb (plain multi-word arithmetic on Python integers)."""
    fhe = _lib()
    N, logQ, logP, B, p = 1 << 16, 1024, 1024, 4, 60
    prm = scheme.Params(N, logQ, logP, 0)
    Q, PQ = prm.Q, prm.PQ
    ctx = fhe.Context(N, logQ, logP)
    assert ctx.L == 32 and ctx.L_PQ == 64
    g = synth.rng(1024)
    ct1 = synth.uniform_limbs(g, (B, 2), N, logQ)
    ct2 = synth.uniform_limbs(g, (B, 2), N, logQ)
    pt = synth.uniform_limbs(g, (B,), N, logQ)
    keys = {name: synth.uniform_limbs(g, (2,), N, logQ + logP) for name in ("evk", "rot5", "conj")}
    kp = {name: [from_limbs(v[0]), from_limbs(v[1])] for name, v in keys.items()}
    ctx.fhe_set_evk(limbs_np_to_tensor(keys["evk"]))
    ctx.fhe_set_rotation_key(0, 5, limbs_np_to_tensor(keys["rot5"]))
    ctx.fhe_set_rotation_key(1, 2 * N - 1, limbs_np_to_tensor(keys["conj"]))
    d1, d2, dpt = limbs_np_to_tensor(ct1), limbs_np_to_tensor(ct2), limbs_np_to_tensor(pt)
    t3 = ctx.fhe_he_mult(d1, d2)
    t2 = ctx.fhe_relinearize(t3)
    tr = ctx.fhe_rescale(t2, p)
    assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, p), tr)
    out3, out2, outr = tensor_to_np(t3), tensor_to_np(t2), tensor_to_np(tr)
    rot = {0: tensor_to_np(ctx.fhe_rotate(d1, 0)), 1: tensor_to_np(ctx.fhe_rotate(d1, 1))}
    mp = tensor_to_np(ctx.fhe_mult_plain(d1, dpt, 1))
    checked = 0
    for b in (0, B - 1):
        c = [from_limbs(ct1[b, 0]), from_limbs(ct1[b, 1])]
        e = [from_limbs(ct2[b, 0]), from_limbs(ct2[b, 1])]
        ks = _structured_ks(N, b, B, 3, ctx.n_sm, per_item=24)
        for n, k in enumerate(ks):
            which = (n + b) % 3
            if which == 0:
                want = ring.pm_coeff(c[0], e[0], k, Q)
            elif which == 1:
                want = (ring.pm_coeff(c[0], e[1], k, Q) + ring.pm_coeff(c[1], e[0], k, Q)) % Q
            else:
                want = ring.pm_coeff(c[1], e[1], k, Q)
            assert coeff_from_limbs(out3[b, which], k) == want, ("he_mult", b, which, k)
        d2b = from_limbs(out3[b, 2])
        for n, k in enumerate(_structured_ks(N, b, B, 2, ctx.n_sm, per_item=24)):
            comp = (n + b) % 2
            want = (coeff_from_limbs(out3[b, comp], k) + scheme.round_shift(ring.pm_coeff(d2b, kp["evk"][comp], k, PQ), logP)) % Q
            assert coeff_from_limbs(out2[b, comp], k) == want, ("relin", b, comp, k)
            assert coeff_from_limbs(outr[b, comp], k) == scheme.round_shift(want, p) % (1 << (logQ - p)), ("rescale", b, comp, k)
        for slot, kgal, name in ((0, 5, "rot5"), (1, 2 * N - 1, "conj")):
            s0, s1 = scheme.automorphism(c[0], kgal, Q), scheme.automorphism(c[1], kgal, Q)
            for n, k in enumerate(_structured_ks(N, b, B, 2, ctx.n_sm, per_item=16)):
                comp = (n + b + slot) % 2
                want = ((s0[k] if comp == 0 else 0) + scheme.round_shift(ring.pm_coeff(s1, kp[name][comp], k, PQ), logP)) % Q
                assert coeff_from_limbs(rot[slot][b, comp], k) == want, (name, b, comp, k)
                checked += 1
        m = from_limbs(pt[b])
        for n, k in enumerate(_structured_ks(N, b, B, 2, ctx.n_sm, per_item=12)):
            comp = (n + b) % 2
            assert coeff_from_limbs(mp[b, comp], k) == ring.pm_coeff(c[comp], m, k, Q), ("mult_plain", b, comp, k)
        checked += len(ks)
    assert checked >= 200
    # the streaming rows of the table, every limb: whole-limb Q makes them plain multi-word arithmetic
    a64 = [from_limbs(ct1[1, i]) for i in range(2)]
    b64 = [from_limbs(ct2[1, i]) for i in range(2)]
    one = slice(1, 2)
    assert tensor_to_polys(ctx.fhe_add(d1[one], d2[one]))[0] == [[(x + y) % Q for x, y in zip(a64[i], b64[i])] for i in range(2)]
    assert tensor_to_polys(ctx.fhe_sub(d1[one], d2[one]))[0] == [[(x - y) % Q for x, y in zip(a64[i], b64[i])] for i in range(2)]
    assert tensor_to_polys(ctx.fhe_negate(d1[one]))[0] == [[(-x) % Q for x in a64[i]] for i in range(2)]
    assert tensor_to_polys(ctx.fhe_moddown(d1[one], logQ - p))[0] == [[x % (1 << (logQ - p)) for x in a64[i]] for i in range(2)]
    h = N // 2                                       # X^(N/2) a: coefficient i moves to i + N/2, negated when it wraps (pin P3)
    assert tensor_to_polys(ctx.fhe_mul_monomial(d1[one], h))[0] == [[(-x) % Q for x in a64[i][h:]] + a64[i][:h] for i in range(2)]
    assert tensor_to_polys(ctx.fhe_mult_scalar(d1[one], 123456789))[0] == [[(x * 123456789) % Q for x in a64[i]] for i in range(2)]
    m1 = from_limbs(pt[1])
    assert tensor_to_polys(ctx.fhe_add_plain(d1[one], dpt[one], 1))[0] == [[(x + y) % Q for x, y in zip(a64[0], m1)], a64[1]]


# ---- CUDA graph capture: the hot-path calls allocate nothing, synchronise nothing and stay on the caller's stream ---------
def test_hot_path_is_cuda_graph_capturable_and_replays_bit_identically():
    """include/fhe.h, "Ownership": hot-path calls enqueue on the caller's stream, allocate nothing and never synchronise.
    A CUDA graph capture fails on any of those, so: capture fhe_mult_relin_rescale (12 launches, programmatic dependent
    launch attributes included) and fhe_polymul_static once, replay them on new inputs written into the captured buffers,
    and compare every limb with the direct calls."""
    fhe = _lib()
    N, logQ, logP, B, p = 1 << 10, 128, 128, 2, 40
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(31337)
    ctx.fhe_set_evk(limbs_np_to_tensor(synth.uniform_limbs(g, (2,), N, logQ + logP)))
    def fresh():
        return (limbs_np_to_tensor(synth.uniform_limbs(g, (B, 2), N, logQ)), limbs_np_to_tensor(synth.uniform_limbs(g, (B, 2), N, logQ)))
    x, y = fresh()
    out = torch.empty_like(x)
    pm = torch.empty((B, ctx.L, N), dtype=torch.int32, device="cuda")
    side = torch.cuda.Stream()
    side.wait_stream(torch.cuda.current_stream())
    with torch.cuda.stream(side):                    # warm-up on the capture stream: workspace of the binding, kernel attributes
        ctx.fhe_mult_relin_rescale(x, y, p, out=out, stream=side)
        ctx.fhe_polymul_static(x[:, 0].contiguous(), y[:, 0].contiguous(), pm, stream=side)
    side.synchronize()
    xa, ya = x[:, 0].contiguous(), y[:, 0].contiguous()
    graph = torch.cuda.CUDAGraph()
    l0 = ctx.launch_count()
    with torch.cuda.graph(graph, stream=side):
        ctx.fhe_mult_relin_rescale(x, y, p, out=out, stream=torch.cuda.current_stream())
        ctx.fhe_polymul_static(xa, ya, pm, stream=torch.cuda.current_stream())
    assert ctx.launch_count() - l0 >= 12
    for _ in range(2):
        nx, ny = fresh()
        x.copy_(nx); y.copy_(ny); xa.copy_(nx[:, 0]); ya.copy_(ny[:, 0])
        out.fill_(-1); pm.fill_(-1)
        graph.replay()
        torch.cuda.synchronize()
        assert torch.equal(out, ctx.fhe_mult_relin_rescale(nx, ny, p))
        assert torch.equal(pm, ctx.fhe_polymul(nx[:, 0].contiguous(), ny[:, 0].contiguous()))


# ---- a grid of small shapes: every path selection that depends on (logQ, logP, t) ------------------------------------------
_GRID = [(lq, lp, 0) for lq in (33, 64, 96, 127, 160, 200, 256, 300) for lp in (32, 95, 96, 128, 250)] + \
        [(lq, lp, t) for t in (3, 257, 65537) for lq, lp in ((64, 96), (96, 96), (100, 160), (128, 100), (150, 96), (200, 200), (250, 130))]


@pytest.mark.parametrize("logQ,logP,t", _GRID)
def test_grid_of_small_shapes_full_pipeline(logQ, logP, t):
    """N = 256, two uniform pairs (parity needs no encryption) with one all-(Q - 1) polynomial, through polymul, he_mult,
    relinearize and (CKKS) rescale by 1, 17 and logQ - 1 against the oracle, in the default path selection and with everything
    forced through the tensor-core pipeline.  The grid crosses the bounds that select a path: CUDA-core vs pipeline conversions
    (K x limbs <= 192), top-form vs full CKKS relin target (logP >= 96), the three BGV divide-by-P routes, logQ and logP
    multiples of 32 and not."""
    fhe = _lib()
    N, B = 256, 2
    prm = scheme.Params(N, logQ, logP, t)
    try:
        ctx = fhe.Context(N, logQ, logP, t)
    except fhe.FheError as ex:
        pytest.skip(f"shape not supported: {ex}")
    Q, PQ = prm.Q, prm.PQ
    rnd = np.random.default_rng(logQ * 1000 + logP + t)
    def poly(M):
        return [int.from_bytes(rnd.bytes((M.bit_length() + 7) // 8 + 1), "little") % M for _ in range(N)]
    ct1 = [[poly(Q), poly(Q)] for _ in range(B)]
    ct2 = [[poly(Q), poly(Q)] for _ in range(B)]
    ct1[1][0] = [Q - 1] * N
    ct2[1][1] = [Q - 1] * N
    evk = (poly(PQ), poly(PQ))
    d1, d2 = polys_to_tensor(ct1, ctx.L), polys_to_tensor(ct2, ctx.L)
    ctx.fhe_set_evk(polys_to_tensor(list(evk), ctx.L_PQ))
    want_pm = [ring.pm(ct1[i][0], ct2[i][1], Q) for i in range(B)]
    want3 = [scheme.he_mult(prm, tuple(ct1[i]), tuple(ct2[i])) for i in range(B)]
    want2 = [scheme.relinearize(prm, want3[i], evk) for i in range(B)]
    for mode in (0, 1):
        ctx.fhe_debug_force_pipeline(mode)
        assert tensor_to_polys(ctx.fhe_polymul(d1[:, 0].contiguous(), d2[:, 1].contiguous())) == [list(p) for p in want_pm], mode
        try:
            t3 = ctx.fhe_he_mult(d1, d2)
            t2 = ctx.fhe_relinearize(t3)
        except fhe.FheError as ex:
            if "too large" in str(ex):
                continue                                   # a CRT target the pipeline cannot hold: the calls say so
            raise
        assert tensor_to_polys(t3) == [[list(p) for p in w] for w in want3], mode
        assert tensor_to_polys(t2) == [[list(p) for p in w] for w in want2], mode
        if t == 0:
            for pb in (1, 17, logQ - 1):
                wantr = [scheme.rescale(prm, want2[i], pb) for i in range(B)]
                assert tensor_to_polys(ctx.fhe_rescale(t2, pb)) == [[list(p) for p in w] for w in wantr], (mode, pb)
                assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, pb), ctx.fhe_rescale(t2, pb)), (mode, pb)
        else:
            assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, 0), t2), mode


# ---- configs[3]: non-RNS BGV ---------------------------------------------------------------------------------------------
def _bgv_setup(N, logQ, logP, t, B, seed):
    prm = scheme.Params(N, logQ, logP, t)
    g = synth.rng(seed)
    s, evk = harness.keygen(prm, g, hwt=None)
    cts1, cts2, ms = [], [], []
    for _ in range(B):
        m1 = [int(v) for v in synth.uniform_mod(g, N, t)]
        m2 = [int(v) for v in synth.uniform_mod(g, N, t)]
        cts1.append(harness.encrypt(prm, g, s, m1))
        cts2.append(harness.encrypt(prm, g, s, m2))
        ms.append((m1, m2))
    return prm, s, evk, cts1, cts2, ms


# The divide-by-P of the BGV relinearisation has three routes (kernels_crt.cu, PostParams::fold_*): the fold through P = 2^logP + e on
# V itself (the first three shapes), the fold after a Barrett reduction mod PQ ((256, 174, 128, 257): the second fold's quotient
# needs 96 bits), and the general Barrett division ((256, 220, 120, 257), (256, 136, 96, 786433): logQ too far above logP)
@pytest.mark.parametrize("N,logQ,logP,t", [(256, 100, 100, 257), (1024, 437, 437, 65537), (512, 150, 220, 65537), (256, 174, 128, 257),
                                          (256, 220, 120, 257), (256, 136, 96, 786433)])
def test_bgv_small_full(N, logQ, logP, t):
    fhe = _lib()
    prm, s, evk, cts1, cts2, ms = _bgv_setup(N, logQ, logP, t, 2, seed=N + t)
    ctx = fhe.Context(N, logQ, logP, t)
    assert ctx.modulus(0) == prm.Q and ctx.modulus(1) == prm.P and ctx.modulus(2) == prm.PQ
    assert (ctx.L, ctx.L_PQ) == (prm.L, prm.L_PQ)
    ctx.fhe_set_evk(polys_to_tensor(list(evk), ctx.L_PQ))
    d1, d2 = polys_to_tensor(cts1, ctx.L), polys_to_tensor(cts2, ctx.L)
    t3 = ctx.fhe_he_mult(d1, d2)
    want3 = [scheme.he_mult(prm, cts1[i], cts2[i]) for i in range(2)]
    assert tensor_to_polys(t3) == [[list(p) for p in w] for w in want3]
    t2 = ctx.fhe_relinearize(t3)
    want2 = [scheme.relinearize(prm, want3[i], evk) for i in range(2)]
    got2 = tensor_to_polys(t2)
    assert got2 == [[list(p) for p in w] for w in want2]
    assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, 0), t2)
    for i in range(2):   # R4: exact decryption mod t from the GPU ciphertext
        assert harness.decrypt_bgv(tuple(got2[i]), s, prm) == ring.pm(ms[i][0], ms[i][1], t)
    with pytest.raises(fhe.FheError):
        ctx.fhe_rescale(t2, 8)


def test_c4_bgv_full_size():
    """configs[3]: N = 2^14, t = 65537, Q = P = least odd > 2^437 that is 1 mod t; batch of 16.  Pair 0 is a real
    encryption checked in full (and decrypted exactly mod t); the rest of the batch is uniform below Q, sampled."""
    fhe = _lib()
    N, logQ, logP, t, B = 1 << 14, 437, 437, 65537, 16
    prm, s, evk, cts1, cts2, ms = _bgv_setup(N, logQ, logP, t, 1, seed=4)
    ctx = fhe.Context(N, logQ, logP, t)
    assert ctx.modulus(0) == (1 << 437) + 33 and (ctx.L, ctx.L_PQ) == (14, 28)
    g = synth.rng(44)
    r1 = synth.uniform_limbs(g, (B, 2), N, 437)          # < 2^437 < Q
    r2 = synth.uniform_limbs(g, (B, 2), N, 437)
    r1 = np.concatenate([r1, np.zeros((B, 2, ctx.L - r1.shape[2], N), np.uint32)], axis=2) if r1.shape[2] < ctx.L else r1
    r2 = np.concatenate([r2, np.zeros((B, 2, ctx.L - r2.shape[2], N), np.uint32)], axis=2) if r2.shape[2] < ctx.L else r2
    r1[0] = np.stack([to_limbs(p, ctx.L) for p in cts1[0]])
    r2[0] = np.stack([to_limbs(p, ctx.L) for p in cts2[0]])
    r1[1, 0] = to_limbs([prm.Q - 1] * N, ctx.L)            # extreme inputs: every coefficient Q - 1
    r2[1, 0] = to_limbs([prm.Q - 1] * N, ctx.L)
    ctx.fhe_set_evk(polys_to_tensor(list(evk), ctx.L_PQ))
    d1, d2 = limbs_np_to_tensor(r1), limbs_np_to_tensor(r2)
    t3 = ctx.fhe_he_mult(d1, d2)
    out3 = tensor_to_np(t3)
    want3 = scheme.he_mult(prm, cts1[0], cts2[0])
    assert [from_limbs(out3[0, i]) for i in range(3)] == [list(p) for p in want3]
    for b in (1, 7, B - 1):
        _check_he_mult_samples(out3[b], r1[b], r2[b], prm.Q, _sample_ks(N, b, 2))
    t2 = ctx.fhe_relinearize(t3)
    out2 = tensor_to_np(t2)
    want2 = scheme.relinearize(prm, want3, evk)
    got0 = [from_limbs(out2[0, i]) for i in range(2)]
    assert got0 == [list(p) for p in want2]
    assert harness.decrypt_bgv(tuple(got0), s, prm) == ring.pm(ms[0][0], ms[0][1], t)
    for b in (1, B - 1):
        for k in _sample_ks(N, 20 + b, 2):
            want = _relin_coeff_bgv(prm, out3[b], list(evk), k)
            assert [coeff_from_limbs(out2[b, 0], k), coeff_from_limbs(out2[b, 1], k)] == want, (b, k)
    assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, 0), t2)


# ---- shapes that make the conversion pipeline take its other paths -------------------------------------------------------
def test_decompose_extreme_byte_sums_and_two_passes():
    """Every input byte 0xFF (the largest accumulator columns the Barrett step sees), a one-hot input, and a prime count
    whose accumulator columns exceed tensor memory, so the launch runs two passes over its tiles (pipe.cuh)."""
    fhe = _lib()
    N, logQ = 512, 2480
    ctx = fhe.Context(N, logQ, 32)
    Lin = ctx.L
    K = ctx.K_pm
    assert (K + 15) // 16 > 6            # more 64-column chunks than fit beside the A buffers in 512 TMEM columns
    q, _ = ctx.primes(K)
    limbs = np.zeros((3, Lin, N), dtype=np.uint32)
    limbs[0] = 0xFFFFFFFF
    limbs[1, Lin - 1, :] = 0x80000000
    limbs[2] = synth.uniform_limbs(synth.rng(5), (), N, 32 * Lin)
    res = tensor_to_np(ctx.fhe_debug_decompose(limbs_np_to_tensor(limbs), K, 0))
    for p in range(3):
        vals = from_limbs(limbs[p])
        for j in (0, 15, 16, 95, 96, K - 1):
            want = np.array([v % q[j] for v in vals], dtype=np.uint32)
            assert np.array_equal(res[p, j], want), (p, j)


def test_polymul_widest_sweep_cell_sampled():
    """A cell of the polymul sweep at logQ = 2480 (78 limbs, K > 160): two-pass decompose, single-buffered A operand
    in the CRT.  Sampled coefficients from the definition (Eq. 5-6)."""
    fhe = _lib()
    N, logQ, batch = 1 << 12, 2480, 3
    ctx = fhe.Context(N, logQ, 32)
    assert ctx.L == 78 and ctx.K_pm > 160
    g = synth.rng(2480)
    a = synth.uniform_limbs(g, (batch,), N, logQ)
    b = synth.uniform_limbs(g, (batch,), N, logQ)
    out = tensor_to_np(ctx.fhe_polymul(limbs_np_to_tensor(a), limbs_np_to_tensor(b)))
    Q = 1 << logQ
    rnd = np.random.default_rng(3)
    for i in range(batch):
        ai, bi = from_limbs(a[i]), from_limbs(b[i])
        for k in [0, 1, 127, 128, N - 1] + [int(v) for v in rnd.integers(0, N, size=4)]:
            assert coeff_from_limbs(out[i], k) == ring.pm_coeff(ai, bi, k, Q)


@pytest.mark.parametrize("batch", [1, 5, 37])
def test_host_entry_point_equals_device_path(batch):
    """fhe_mult_relin_rescale_host pipelines the batch in pieces over three streams (37 items: ragged pieces of two);
    its result must be the device path's, bit for bit."""
    fhe = _lib()
    N, logQ, logP, p = 256, 128, 128, 40
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(77)
    ct1 = limbs_np_to_tensor(synth.uniform_limbs(g, (batch, 2), N, logQ))
    ct2 = limbs_np_to_tensor(synth.uniform_limbs(g, (batch, 2), N, logQ))
    ctx.fhe_set_evk(limbs_np_to_tensor(synth.uniform_limbs(g, (2,), N, logQ + logP)))
    want = ctx.fhe_mult_relin_rescale(ct1, ct2, p)
    torch.cuda.synchronize()
    h1, h2 = ct1.cpu().pin_memory(), ct2.cpu().pin_memory()
    got = ctx.fhe_mult_relin_rescale_host(h1, h2, p)
    assert torch.equal(got, want.cpu())


def test_empty_batch_is_a_no_op():
    fhe = _lib()
    ctx = fhe.Context(256, 64, 32)
    a = torch.empty((0, ctx.L, 256), dtype=torch.int32, device="cuda")
    out = ctx.fhe_polymul(a, a)
    assert out.shape[0] == 0


@pytest.mark.parametrize("bits", [1, 4, 58])
@pytest.mark.parametrize("logQ,logP", [(128, 128), (100, 96), (218, 250)])
def test_relin_top_form_and_its_exact_path(bits, logQ, logP):
    """The CKKS relin CRT takes the carry out of the low logP bits from 96-bit truncated constants and
    recomputes flagged coefficients exactly.  With the flag threshold lowered to 1 or 4 fractional bits half resp. 1/16
    of the coefficients go down the exact path; every setting must give the oracle's limbs, with and without rescale."""
    fhe = _lib()
    N, B, p = 256, 2, 40
    prm = scheme.Params(N, logQ, logP, 0)
    ctx = fhe.Context(N, logQ, logP)
    ctx.fhe_debug_crt_ambiguity(bits)
    g = synth.rng(900 + bits + logP)
    d3_np = synth.uniform_limbs(g, (B, 3), N, logQ)
    evk_np = synth.uniform_limbs(g, (2,), N, logQ + logP)
    d3 = [[from_limbs(d3_np[i, k]) for k in range(3)] for i in range(B)]
    evk = tuple(from_limbs(evk_np[k]) for k in range(2))
    ctx.fhe_set_evk(limbs_np_to_tensor(evk_np))
    r2 = ctx.fhe_relinearize(limbs_np_to_tensor(d3_np))
    want2 = [scheme.relinearize(prm, tuple(d3[i]), evk) for i in range(B)]
    assert tensor_to_polys(r2) == [[list(q) for q in w] for w in want2]
    # fused path (he_mult -> relin -> rescale) against the oracle's three calls
    ct_np = synth.uniform_limbs(g, (2, B, 2), N, logQ)
    fused = ctx.fhe_mult_relin_rescale(limbs_np_to_tensor(ct_np[0]), limbs_np_to_tensor(ct_np[1]), p)
    for i in range(B):
        c1 = tuple(from_limbs(ct_np[0, i, k]) for k in range(2))
        c2 = tuple(from_limbs(ct_np[1, i, k]) for k in range(2))
        want = scheme.rescale(prm, scheme.relinearize(prm, scheme.he_mult(prm, c1, c2), evk), p)
        assert tensor_to_polys(fused[i]) == [list(q) for q in want]


@pytest.mark.parametrize("logQ,logP,amb", [(352, 352, 58), (352, 352, 1), (365, 120, 58), (365, 120, 1), (352, 64, 58), (365, 90, 58)])
def test_fused_rescale_epilogue_shift_amounts(logQ, logP, amb):
    """The rescale fused into the relin CRT epilogue (what fhe_mult_relin_rescale, the benchmarked call, runs) over the
    shift amounts that move its limb boundaries: p < 32, p a multiple of 32, p = logQ - 1, p past the rounding limb;
    top-form targets (logP >= 96, with the exact path forced on half of the coefficients and off) and full targets
    (logP < 96); logQ a multiple of 32 and not.  L = 11 / 12 limbs, so the streaming fast path (no boundary inside a group
    of eight limbs) is taken as well as the boundary path.  Each must equal the three separate calls and the oracle."""
    fhe = _lib()
    N, B = 256, 2
    prm = scheme.Params(N, logQ, logP, 0)
    ctx = fhe.Context(N, logQ, logP)
    assert ctx.L > 10
    ctx.fhe_debug_crt_ambiguity(amb)
    g = synth.rng(logQ + logP + amb)
    ct_np = synth.uniform_limbs(g, (2, B, 2), N, logQ)
    evk_np = synth.uniform_limbs(g, (2,), N, logQ + logP)
    evk = tuple(from_limbs(evk_np[k]) for k in range(2))
    ctx.fhe_set_evk(limbs_np_to_tensor(evk_np))
    d1, d2 = limbs_np_to_tensor(ct_np[0]), limbs_np_to_tensor(ct_np[1])
    t2 = ctx.fhe_relinearize(ctx.fhe_he_mult(d1, d2))
    want2 = []
    for i in range(B):
        c1 = tuple(from_limbs(ct_np[0, i, k]) for k in range(2))
        c2 = tuple(from_limbs(ct_np[1, i, k]) for k in range(2))
        want2.append(scheme.relinearize(prm, scheme.he_mult(prm, c1, c2), evk))
    assert tensor_to_polys(t2) == [[list(q) for q in w] for w in want2]
    assert torch.equal(ctx.fhe_mult_relin_rescale(d1, d2, 0), t2)
    for p in (1, 31, 32, 33, 64, 96, 320, logQ - 1):
        fused = ctx.fhe_mult_relin_rescale(d1, d2, p)
        assert torch.equal(fused, ctx.fhe_rescale(t2, p)), p
        assert tensor_to_polys(fused) == [[list(q) for q in scheme.rescale(prm, w, p)] for w in want2], p


def test_exact_path_takes_every_flagged_coefficient_of_a_large_launch():
    """With the flag threshold at one fractional bit half of the coefficients of a launch go down the exact CRT path:
    2 items x 2 polynomials x 2^16 coefficients = 131 072 flagged ones in one launch (the flag store is a bitmap sized to
    the launch, so none can be dropped).  The result must be the same limbs as with the threshold at 58 bits, and the
    oracle's on structured positions."""
    fhe = _lib()
    N, logQ, logP, B, p = 1 << 16, 128, 128, 2, 40
    prm = scheme.Params(N, logQ, logP, 0)
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(4242)
    ct1 = synth.uniform_limbs(g, (B, 2), N, logQ)
    ct2 = synth.uniform_limbs(g, (B, 2), N, logQ)
    evk_np = synth.uniform_limbs(g, (2,), N, logQ + logP)
    ctx.fhe_set_evk(limbs_np_to_tensor(evk_np))
    d1, d2 = limbs_np_to_tensor(ct1), limbs_np_to_tensor(ct2)
    t3 = ctx.fhe_he_mult(d1, d2)
    ref2, ref = ctx.fhe_relinearize(t3), ctx.fhe_mult_relin_rescale(d1, d2, p)
    ctx.fhe_debug_crt_ambiguity(1)
    got2, got = ctx.fhe_relinearize(t3), ctx.fhe_mult_relin_rescale(d1, d2, p)
    assert torch.equal(got2, ref2) and torch.equal(got, ref)
    out3, out2 = tensor_to_np(t3), tensor_to_np(got2)
    evk = [from_limbs(evk_np[0]), from_limbs(evk_np[1])]
    for b in range(B):
        d2b = from_limbs(out3[b, 2])
        for k in _structured_ks(N, b, B, 2, ctx.n_sm, per_item=16):
            want = _relin_coeff_ckks(prm, out3[b], evk, k, d2b)
            assert [coeff_from_limbs(out2[b, 0], k), coeff_from_limbs(out2[b, 1], k)] == want, (b, k)


@pytest.mark.parametrize("N,logQ,logP,t", [(1 << 12, 128, 128, 0), (1 << 13, 100, 96, 0), (1 << 13, 150, 60, 0), (1 << 12, 120, 120, 257),
                                            (1 << 13, 100, 130, 65537)])
def test_whole_transform_sizes_full_pipeline(N, logQ, logP, t):
    """N = 2^12 and (on request) 2^13 run every product (polymul, tensor, relin) through the single whole-transform kernel
    (ntt_whole_kernel): every limb of he_mult, relinearize, rescale (CKKS) and polymul against the oracle's own NTT route."""
    fhe = _lib()
    prm = scheme.Params(N, logQ, logP, t)
    ctx = fhe.Context(N, logQ, logP, t)
    ctx.fhe_debug_force_pipeline(2)
    g = synth.rng(N + logQ + t)
    B = 2
    bits = logQ                                                     # uniform below 2^logQ <= Q: canonical for both schemes
    ct_np = synth.uniform_limbs(g, (2, B, 2), N, bits)
    evk_np = synth.uniform_limbs(g, (2,), N, logQ + logP)           # below PQ for both
    def pad(a, L):
        return a if a.shape[-2] == L else np.concatenate([a, np.zeros(a.shape[:-2] + (L - a.shape[-2], N), np.uint32)], axis=-2)
    ct_np, evk_np = pad(ct_np, ctx.L), pad(evk_np, ctx.L_PQ)
    evk = tuple(from_limbs(evk_np[k]) for k in range(2))
    ctx.fhe_set_evk(limbs_np_to_tensor(evk_np))
    d1, d2 = limbs_np_to_tensor(ct_np[0]), limbs_np_to_tensor(ct_np[1])
    t3 = ctx.fhe_he_mult(d1, d2)
    t2 = ctx.fhe_relinearize(t3)
    pm_out = ctx.fhe_polymul(d1[:, 0].contiguous(), d2[:, 1].contiguous())
    got3, got2, gotpm = tensor_to_polys(t3), tensor_to_polys(t2), tensor_to_polys(pm_out)
    for i in range(B):
        c1 = tuple(from_limbs(ct_np[0, i, k]) for k in range(2))
        c2 = tuple(from_limbs(ct_np[1, i, k]) for k in range(2))
        want3 = scheme.he_mult(prm, c1, c2)
        assert got3[i] == [list(p) for p in want3], i
        want2 = scheme.relinearize(prm, want3, evk)
        assert got2[i] == [list(p) for p in want2], i
        assert gotpm[i] == ring.pm(c1[0], c2[1], prm.Q), i
        if t == 0:
            assert tensor_to_polys(ctx.fhe_mult_relin_rescale(d1, d2, 40)[i]) == [list(p) for p in scheme.rescale(prm, want2, 40)]


# ---- NEXT-1: coefficient-wise operations, level drop, and a depth-2 circuit across two levels ----------------
@pytest.mark.parametrize("N,logQ,t", [(256, 128, 0), (1024, 218, 0), (256, 100, 257), (1024, 437, 65537)])
def test_next1_add_sub_negate_match_the_oracle(N, logQ, t):
    fhe = _lib()
    prm = scheme.Params(N, logQ, logQ, t)
    ctx = fhe.Context(N, logQ, logQ, t)
    g = synth.rng(50 + N + logQ)
    Q = prm.Q
    rnd = np.random.default_rng(N + logQ)
    def rand_ct():
        ct = tuple([int.from_bytes(rnd.bytes((Q.bit_length() + 7) // 8 + 8), "little") % Q for _ in range(N)] for _ in range(2))
        ct[0][0], ct[0][1], ct[1][0] = 0, Q - 1, Q - 1          # the ends of the range
        return ct
    c1, c2 = rand_ct(), rand_ct()
    d1, d2 = polys_to_tensor([list(c1)], ctx.L), polys_to_tensor([list(c2)], ctx.L)
    assert tensor_to_polys(ctx.fhe_add(d1, d2))[0] == [list(p) for p in scheme.ct_add(prm, c1, c2)]
    assert tensor_to_polys(ctx.fhe_sub(d1, d2))[0] == [list(p) for p in scheme.ct_sub(prm, c1, c2)]
    assert tensor_to_polys(ctx.fhe_negate(d1))[0] == [list(p) for p in scheme.ct_negate(prm, c1)]
    assert torch.equal(ctx.fhe_sub(ctx.fhe_add(d1, d2), d2), d1)


def test_next1_moddown_and_depth_two_circuit_over_two_levels():
    """(z1 z2) z3 on CKKS: multiply + relinearise + rescale at logQ = 128, drop the factor z3 to the new level with
    fhe_moddown, multiply again with a context for logQ = 88 whose evk is the original one reduced mod 2^(logP + 88).
    Every ciphertext equals the oracle's limb for limb; the final decryption is within 2^-20 of the slot product."""
    fhe = _lib()
    N, logQ, logP, p = 1 << 10, 128, 128, 40
    prm, s, evk, cts1, cts2, zs = _ckks_setup(N, logQ, logP, 2, seed=5)
    hi = fhe.Context(N, logQ, logP)
    hi.fhe_set_evk(polys_to_tensor(list(evk), hi.L_PQ))
    # level 1: ct12 = rescale(relin(ct1 * ct2)) has modulus 2^88
    ct12 = hi.fhe_mult_relin_rescale(polys_to_tensor([cts1[0]], hi.L), polys_to_tensor([cts2[0]], hi.L), p)
    want12 = scheme.rescale(prm, scheme.relinearize(prm, scheme.he_mult(prm, cts1[0], cts2[0]), evk), p)
    assert tensor_to_polys(ct12)[0] == [list(q) for q in want12]
    logq1 = logQ - p
    # the third factor comes down to the same level by moddown
    ct3 = hi.fhe_moddown(polys_to_tensor([cts1[1]], hi.L), logq1)
    want3 = scheme.moddown(prm, cts1[1], logq1)
    assert tensor_to_polys(ct3)[0] == [list(q) for q in want3]
    # level 2 context: logQ = 88 (3 limbs), evk mod 2^(logP + 88)
    prm1 = scheme.Params(N, logq1, logP, 0)
    lo = fhe.Context(N, logq1, logP)
    evk1 = tuple([x % prm1.PQ for x in e] for e in evk)
    lo.fhe_set_evk(polys_to_tensor(list(evk1), lo.L_PQ))
    a = ct12[..., : lo.L, :].contiguous()
    b = ct3[..., : lo.L, :].contiguous()
    out = lo.fhe_mult_relin_rescale(a, b, p)
    want = scheme.rescale(prm1, scheme.relinearize(prm1, scheme.he_mult(prm1, want12, want3), evk1), p)
    got = tensor_to_polys(out)[0]
    assert got == [list(q) for q in want]
    mu = harness.decrypt(tuple(got), s, 1 << (logq1 - p))
    z = harness.decode(mu, N, 2.0 ** 40)
    assert np.max(np.abs(z - zs[0][0] * zs[0][1] * zs[1][0])) <= 2.0 ** -20


# ---- NEXT-2: rotation / conjugation = automorphism + key switch with a rotation key ----------------------
@pytest.mark.parametrize("N,logQ,logP,t,ks", [(1 << 10, 128, 128, 0, (5, 25, 2047)), (256, 100, 100, 257, (3, 511)),
                                              (1 << 12, 218, 250, 0, (5,))])
def test_next2_rotate_matches_the_oracle(N, logQ, logP, t, ks):
    fhe = _lib()
    prm = scheme.Params(N, logQ, logP, t)
    g = synth.rng(60 + N)
    s, _ = harness.keygen(prm, g, hwt=64 if t == 0 else None)
    ctx = fhe.Context(N, logQ, logP, t)
    B = 2
    if t == 0:
        zs = [synth.unit_disk(g, N // 2) for _ in range(B)]
        cts = [harness.encrypt(prm, g, s, harness.encode(z, N, 2.0 ** 40)) for z in zs]
    else:
        ms = [[int(v) for v in g.integers(0, t, size=N)] for _ in range(B)]
        cts = [harness.encrypt(prm, g, s, m) for m in ms]
    d = polys_to_tensor([list(c) for c in cts], ctx.L)
    for slot, k in enumerate(ks):
        rk = harness.rotkeygen(prm, g, s, k)
        ctx.fhe_set_rotation_key(slot, k, polys_to_tensor(list(rk), ctx.L_PQ))
        got = tensor_to_polys(ctx.fhe_rotate(d, slot))
        for i in range(B):
            want = scheme.rotate(prm, cts[i], k, rk)
            assert got[i] == [list(p) for p in want], (k, i)
        if t == 0:
            src, conj = harness.slot_image(N, k)
            z = harness.decode(harness.decrypt(tuple(got[0]), s, prm.Q), N, 2.0 ** 40)
            want = np.array([np.conj(zs[0][j]) if c else zs[0][j] for j, c in zip(src, conj)])
            assert np.max(np.abs(z - want)) <= 2.0 ** -20
        else:
            assert harness.decrypt_bgv(tuple(got[0]), s, prm) == scheme.automorphism(ms[0], k, t)
    # an empty slot is an error, not a silent no-op
    with pytest.raises(fhe.FheError):
        ctx.fhe_rotate(d, len(ks))


# ---- NEXT-3: ciphertext x plaintext, pairwise and broadcast ----------------------------------------------
@pytest.mark.parametrize("N,logQ,t,B,group", [(1024, 128, 0, 3, 1), (1024, 128, 0, 5, 5), (256, 100, 257, 4, 2), (4096, 218, 0, 5, 2)])
def test_next3_mult_plain_pairwise_and_broadcast(N, logQ, t, B, group):
    fhe = _lib()
    prm = scheme.Params(N, logQ, 32 if t == 0 else logQ, t)
    ctx = fhe.Context(N, logQ, prm.logP, t)
    g = synth.rng(70 + N + B)
    Q = prm.Q
    npt = (B + group - 1) // group
    ct_np = synth.uniform_limbs(g, (B, 2), N, logQ)      # uniform below 2^logQ < Q: valid canonical inputs for both schemes
    pt_np = synth.uniform_limbs(g, (npt,), N, logQ)
    out = tensor_to_polys(ctx.fhe_mult_plain(limbs_np_to_tensor(ct_np), limbs_np_to_tensor(pt_np), group))
    for i in range(B):
        ct = tuple(from_limbs(ct_np[i, k]) for k in range(2))
        want = scheme.mult_plain(prm, ct, from_limbs(pt_np[i // group]))
        assert out[i] == [list(p) for p in want], i


@pytest.mark.parametrize("N,logQ,t", [(256, 128, 0), (1024, 218, 0), (256, 100, 257)])
def test_next1_mul_monomial_matches_the_oracle(N, logQ, t):
    fhe = _lib()
    prm = scheme.Params(N, logQ, logQ, t)
    ctx = fhe.Context(N, logQ, logQ, t)
    Q = prm.Q
    rnd = np.random.default_rng(N + logQ + 3)
    ct = tuple([int.from_bytes(rnd.bytes((Q.bit_length() + 7) // 8 + 8), "little") % Q for _ in range(N)] for _ in range(2))
    ct[0][0], ct[0][1], ct[1][N - 1] = 0, Q - 1, 1
    d = polys_to_tensor([list(ct)], ctx.L)
    for k in (0, 1, N // 2, N - 1, N, 3 * N // 2, 2 * N - 1):
        assert tensor_to_polys(ctx.fhe_mul_monomial(d, k))[0] == [list(p) for p in scheme.mul_monomial(prm, ct, k)], k


# ---- NEXT-3, constants: ct + plaintext (pairwise / broadcast) and ct x integer scalar -----------------------------------------
@pytest.mark.parametrize("N,logQ,t,B,group", [(256, 128, 0, 3, 1), (1024, 218, 0, 5, 5), (256, 100, 257, 4, 2), (1024, 437, 65537, 3, 3)])
def test_next3_add_plain_pairwise_and_broadcast(N, logQ, t, B, group):
    fhe = _lib()
    prm = scheme.Params(N, logQ, logQ, t)
    ctx = fhe.Context(N, logQ, logQ, t)
    Q = prm.Q
    rnd = np.random.default_rng(N + logQ + B)
    def rand_poly():
        p = [int.from_bytes(rnd.bytes((Q.bit_length() + 7) // 8 + 8), "little") % Q for _ in range(N)]
        p[0], p[1], p[2] = 0, Q - 1, Q - 1
        return p
    npt = (B + group - 1) // group
    cts = [(rand_poly(), rand_poly()) for _ in range(B)]
    pts = [rand_poly() for _ in range(npt)]
    for m in pts:
        m[2] = 1                                               # (Q - 1) + 1 wraps to 0, (Q - 1) + (Q - 1) to Q - 2
    d_ct = polys_to_tensor([list(c) for c in cts], ctx.L)
    d_pt = polys_to_tensor(pts, ctx.L)
    got = tensor_to_polys(ctx.fhe_add_plain(d_ct, d_pt, group))
    for i in range(B):
        want = scheme.add_plain(prm, cts[i], pts[i // group])
        assert got[i] == [list(p) for p in want], i
    # in place
    ctx.fhe_add_plain(d_ct, d_pt, group, out=d_ct)
    assert tensor_to_polys(d_ct) == got


@pytest.mark.parametrize("N,logQ,t", [(256, 128, 0), (1024, 218, 0), (256, 100, 257), (1024, 437, 65537), (256, 96, 257)])
def test_next3_mult_scalar_matches_the_oracle(N, logQ, t):
    fhe = _lib()
    prm = scheme.Params(N, logQ, logQ, t)
    ctx = fhe.Context(N, logQ, logQ, t)
    Q = prm.Q
    rnd = np.random.default_rng(N + logQ + 5)
    ct = tuple([int.from_bytes(rnd.bytes((Q.bit_length() + 7) // 8 + 8), "little") % Q for _ in range(N)] for _ in range(2))
    ct[0][0], ct[0][1], ct[0][2], ct[1][0], ct[1][1] = 0, Q - 1, 1, Q - 1, (1 << logQ) - 1
    d = polys_to_tensor([list(ct)], ctx.L)
    for k in (0, 1, -1, 2, 3, -7, 65537, 2 ** 31 - 1, -(2 ** 31 - 1)):
        assert tensor_to_polys(ctx.fhe_mult_scalar(d, k))[0] == [list(p) for p in scheme.mult_scalar(prm, ct, k)], k
    keep = d.clone()
    ctx.fhe_mult_scalar(d, -12345, out=d)                      # in place
    assert tensor_to_polys(d)[0] == [list(p) for p in scheme.mult_scalar(prm, ct, -12345)]
    assert torch.equal(ctx.fhe_add(ctx.fhe_mult_scalar(keep, 2), keep), ctx.fhe_mult_scalar(keep, 3))
    with pytest.raises((fhe.FheError, ValueError)):
        ctx.fhe_mult_scalar(keep, -2 ** 31)


# ---- NEXT-4: BGV modulus switching -------------------------------------------------------------------------------
@pytest.mark.parametrize("N,logQ,t,news", [(256, 100, 257, (99, 92, 60, 34)), (1024, 437, 65537, (436, 429, 405, 300, 34)),
                                           (256, 128, 3, (127, 96, 64)), (256, 160, 786433, (159, 140, 97, 40))])
def test_next4_modswitch_matches_the_oracle(N, logQ, t, news):
    """Every coefficient against scheme.modswitch_bgv, over drops of one bit (the quotient correction moves many multiples
    of Q), a few bits, a limb, many limbs; the ends of the range, Q/2 and its neighbours (the centring of r), in place."""
    fhe = _lib()
    prm = scheme.Params(N, logQ, logQ, t)
    ctx = fhe.Context(N, logQ, logQ, t)
    Q = prm.Q
    rnd = np.random.default_rng(N + logQ + t % 1000)
    def rand_poly():
        p = [int.from_bytes(rnd.bytes((Q.bit_length() + 7) // 8 + 8), "little") % Q for _ in range(N)]
        p[:8] = [0, 1, Q - 1, Q - 2, Q // 2, Q // 2 + 1, Q // 2 - 1, (1 << logQ) - 1]
        return p
    ct = (rand_poly(), rand_poly())
    d = polys_to_tensor([list(ct)], ctx.L)
    for new_logQ in news:
        want = scheme.modswitch_bgv(prm, ct, new_logQ)
        got = tensor_to_polys(ctx.fhe_modswitch(d, new_logQ))[0]
        assert got == [list(p) for p in want], new_logQ
    keep = d.clone()
    ctx.fhe_modswitch(d, news[-1], out=d)
    assert torch.equal(d, ctx.fhe_modswitch(keep, news[-1]))
    with pytest.raises(fhe.FheError):
        ctx.fhe_modswitch(keep, logQ)
    with pytest.raises(fhe.FheError):
        fhe.Context(256, 128, 128).fhe_modswitch(torch.zeros((1, 2, 4, 256), dtype=torch.int32, device="cuda"), 64)   # CKKS


def test_next4_bgv_depth_two_circuit_across_a_modulus_switch():
    """(m1 m2) m3 on BGV at the C4 parameter shape (t = 65537, logQ = 437): multiply + relinearise at Q, switch the product
    and a fresh ciphertext down to Q' (logQ' = 300) with fhe_modswitch, multiply + relinearise again with a context and a
    key for Q'.  Every ciphertext equals the oracle's limb for limb; the final decryption is exact mod t."""
    fhe = _lib()
    N, logQ, new_logQ, t = 1 << 10, 437, 300, 65537
    prm, s, evk, cts1, cts2, ms = _bgv_setup(N, logQ, logQ, t, 2, seed=9)
    hi = fhe.Context(N, logQ, logQ, t)
    hi.fhe_set_evk(polys_to_tensor(list(evk), hi.L_PQ))
    prod = hi.fhe_mult_relin_rescale(polys_to_tensor([cts1[0]], hi.L), polys_to_tensor([cts2[0]], hi.L), 0)
    want_prod = scheme.relinearize(prm, scheme.he_mult(prm, cts1[0], cts2[0]), evk)
    assert tensor_to_polys(prod)[0] == [list(p) for p in want_prod]
    low = hi.fhe_modswitch(prod, new_logQ)
    third = hi.fhe_modswitch(polys_to_tensor([cts1[1]], hi.L), new_logQ)
    want_low, want_third = scheme.modswitch_bgv(prm, want_prod, new_logQ), scheme.modswitch_bgv(prm, cts1[1], new_logQ)
    assert tensor_to_polys(low)[0] == [list(p) for p in want_low]
    assert tensor_to_polys(third)[0] == [list(p) for p in want_third]
    prm2 = scheme.Params(N, new_logQ, new_logQ, t)
    assert harness.decrypt_bgv(want_low, s, prm2) == ring.pm(ms[0][0], ms[0][1], t)
    # key for the lower level: same secret, evk mod P'Q'
    g2 = synth.rng(99)
    e2 = synth.gaussian_error(g2, N)
    a2 = synth.uniform_big(g2, N, (prm2.PQ - 1).bit_length() - 1)
    s2 = ring.pm([v % prm2.PQ for v in s], [v % prm2.PQ for v in s], prm2.PQ)
    a_s = harness.pm_secret(a2, s, prm2.PQ)
    evk2 = ([(-x + t * int(e) + prm2.P * y) % prm2.PQ for x, e, y in zip(a_s, e2, s2)], a2)
    lo = fhe.Context(N, new_logQ, new_logQ, t)
    assert lo.modulus(0) == prm2.Q
    lo.fhe_set_evk(polys_to_tensor(list(evk2), lo.L_PQ))
    a = low[..., : lo.L, :].contiguous()
    b = third[..., : lo.L, :].contiguous()
    out = lo.fhe_mult_relin_rescale(a, b, 0)
    want = scheme.relinearize(prm2, scheme.he_mult(prm2, want_low, want_third), evk2)
    got = tensor_to_polys(out)[0]
    assert got == [list(p) for p in want]
    assert harness.decrypt_bgv(tuple(got), s, prm2) == ring.pm(ring.pm(ms[0][0], ms[0][1], t), ms[1][0], t)


def test_repeated_runs_are_bit_identical():
    """The pipeline kernels hand tiles between warp roles through mbarriers, tensor memory and shared memory; a race
    would show as run-to-run differences.  (compute-sanitizer is closed on this pool.)  40 runs of the fused call on a
    shape with several tiles per CTA and ragged last tiles must give one and the same result."""
    fhe = _lib()
    N, logQ, logP, B, p = 1 << 13, 218, 250, 5, 40
    ctx = fhe.Context(N, logQ, logP)
    g = synth.rng(31337)
    ct1 = limbs_np_to_tensor(synth.uniform_limbs(g, (B, 2), N, logQ))
    ct2 = limbs_np_to_tensor(synth.uniform_limbs(g, (B, 2), N, logQ))
    ctx.fhe_set_evk(limbs_np_to_tensor(synth.uniform_limbs(g, (2,), N, logQ + logP)))
    ref = ctx.fhe_mult_relin_rescale(ct1, ct2, p).clone()
    for _ in range(40):
        assert torch.equal(ctx.fhe_mult_relin_rescale(ct1, ct2, p), ref)
