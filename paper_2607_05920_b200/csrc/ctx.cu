// ctx.cu -- fhe_ctx_create: host precomputation of every table the kernels read (section 5.2),
// uploaded once.  Nothing here runs on the hot path.
#include <cstring>
#include <new>

#include "bigu.hpp"
#include "fhe_internal.cuh"

namespace fhe {

static std::string g_create_err;

// ---- word-sized number theory ------------------------------------------------------------------------------------
static inline uint32_t mulmod(uint32_t a, uint32_t b, uint32_t m) { return (uint32_t)((uint64_t)a * b % m); }
static uint32_t powmod(uint32_t a, uint64_t e, uint32_t m) {
  uint32_t r = 1 % m;
  a %= m;
  while (e) {
    if (e & 1) r = mulmod(r, a, m);
    a = mulmod(a, a, m);
    e >>= 1;
  }
  return r;
}
static bool is_prime32(uint32_t n) {   // deterministic Miller-Rabin for n < 2^32 (bases 2, 7, 61)
  if (n < 2) return false;
  for (uint32_t p : {2u, 3u, 5u, 7u, 11u, 13u, 17u, 19u, 23u, 29u, 31u, 37u}) {
    if (n % p == 0) return n == p;
  }
  uint32_t d = n - 1, r = 0;
  while ((d & 1) == 0) { d >>= 1; ++r; }
  for (uint32_t a : {2u, 7u, 61u}) {
    uint32_t x = powmod(a, d, n);
    if (x == 1 || x == n - 1) continue;
    bool comp = true;
    for (uint32_t i = 1; i < r; ++i) {
      x = mulmod(x, x, n);
      if (x == n - 1) { comp = false; break; }
    }
    if (comp) return false;
  }
  return true;
}
static uint32_t bitrev(uint32_t x, uint32_t bits) {
  uint32_t r = 0;
  for (uint32_t i = 0; i < bits; ++i) r |= ((x >> i) & 1u) << (bits - 1 - i);
  return r;
}
static inline uint32_t shoup(uint32_t w, uint32_t q) { return (uint32_t)(((uint64_t)w << 32) / q); }

template <class T>
static cudaError_t upload(Context* c, T** dptr, const std::vector<T>& h) {
  void* p = nullptr;
  size_t bytes = h.size() * sizeof(T);
  cudaError_t e = cudaMalloc(&p, bytes ? bytes : 16);
  if (e != cudaSuccess) return e;
  c->allocs.push_back(p);
  *dptr = (T*)p;
  if (bytes) e = cudaMemcpy(p, h.data(), bytes, cudaMemcpyHostToDevice);
  return e;
}

// modulus 2^log (t == 0) or the least odd integer > 2^log that is 1 mod t: 2^log + modulus_offset(log, t)
uint64_t modulus_offset(uint32_t log, uint64_t t) {
  if (t == 0) return 0;
  uint32_t tt = (uint32_t)t;
  uint32_t two = powmod(2, log, tt);
  uint32_t c0 = (uint32_t)(((uint64_t)1 + tt - two) % tt);   // (1 - 2^log) mod t
  uint64_t c = c0 == 0 ? tt : c0;
  if ((c & 1) == 0) c += tt;                                  // t odd: flips parity
  return c;
}
static BigU make_modulus(uint32_t log, uint64_t t) {
  BigU m = BigU::pow2(log);
  if (t == 0) return m;
  m.add(BigU(modulus_offset(log, t)));
  return m;
}

// smallest K such that the product of the first K primes exceeds bound; extends the prime list on demand
static uint32_t primes_for(std::vector<uint32_t>& primes, const BigU& bound) {
  BigU M((uint64_t)1);
  uint32_t K = 0;
  uint32_t cand = primes.empty() ? 0x40000001u - (1u << 17) : primes.back() - (1u << 17);   // q < 2^30: lazy butterflies keep values in [0, 4q)
  while (BigU::cmp(M, bound) <= 0) {
    if (K == primes.size()) {
      while (!is_prime32(cand)) cand -= (1u << 17);
      primes.push_back(cand);
      cand -= (1u << 17);
    }
    M.mul_small(primes[K]);
    ++K;
  }
  return K;
}

// value as `n` little-endian bytes
static std::vector<uint8_t> bytes_of(const BigU& x, size_t n) {
  std::vector<uint8_t> o(n, 0);
  for (size_t i = 0; i < n; ++i) o[i] = (uint8_t)(x.limb(i / 4) >> (8 * (i % 4)));
  return o;
}

// CRT constants for the basis q_0..q_{K-1} and the target T (pow2: T = 2^(32 Lraw) with Lraw = ceil(width_bits/32);
// else T = Tmod odd).  See fhe_internal.cuh (CrtTarget) and kernels_crt.cu for how the image is consumed.
// decompose constant image [KBimg / 16][cols][16 bytes]: byte cc of (2^(8 kb) m_j) mod q_j at column 4 j + cc (m_j = 1: plain)
static std::vector<uint8_t> dec_image(const Context* c, uint32_t K, const std::vector<uint2>* mult) {
  std::vector<uint8_t> img((size_t)c->dec_KBimg * c->dec_cols, 0);
  for (uint32_t j = 0; j < K; ++j) {
    const uint32_t q = c->h_q[j];
    uint32_t cur = mult ? (*mult)[j].x % q : 1u;
    for (uint32_t kb = 0; kb < c->dec_KBimg; ++kb) {
      for (uint32_t cc = 0; cc < 4; ++cc)
        img[((size_t)(kb / 16) * c->dec_cols + 4 * j + cc) * 16 + kb % 16] = (uint8_t)(cur >> (8 * cc));
      cur = mulmod(cur, 256u, q);
    }
  }
  return img;
}

static cudaError_t build_target(Context* c, CrtTarget& tg, uint32_t K, bool pow2, uint32_t width_bits,
                                const BigU& Tmod, uint32_t post_limbs, bool scaled_image = false) {
  tg.K = K;
  tg.KB = (4 * K + 31) / 32 * 32;
  uint32_t clogK = 0;
  while ((1u << clogK) < K + 1) ++clogK;
  const uint32_t vbits = pow2 ? width_bits : (Tmod.bits() + 32 + clogK + 1);   // V < (K+1) 2^32 T
  tg.Lraw = (vbits + 31) / 32;
  const uint32_t nbytes = 4 * tg.Lraw;
  const uint32_t ncols = CRT_ALPHA_COLS + nbytes;
  tg.Lx = std::max(tg.Lraw + 1, post_limbs);
  constexpr uint32_t NC = 64;                                           // pipe::NC
  tg.nchunks = (ncols + NC - 1) / NC;
  const BigU T = pow2 ? BigU::pow2(32 * tg.Lraw) : Tmod;
  BigU M((uint64_t)1);
  for (uint32_t i = 0; i < K; ++i) M.mul_small(c->h_q[i]);
  const size_t img_cols = (size_t)tg.nchunks * NC;                      // image [KB / 16][img_cols][16 bytes] (pipe.cuh)
  std::vector<uint8_t> img((size_t)tg.KB * img_cols, 0);
  auto put = [&](uint32_t kb, uint32_t col, uint8_t v) {
    img[((size_t)(kb / 16) * img_cols + col) * 16 + kb % 16] = v;
  };
  std::vector<uint2> scale(K);
  for (uint32_t i = 0; i < K; ++i) {
    const uint32_t q = c->h_q[i];
    BigU Mi = M;
    if (Mi.divmod_small(q) != 0) return cudaErrorUnknown;
    const uint32_t inv = powmod(Mi.mod_small(q), q - 2, q);            // (M/q_i)^-1 mod q_i
    const std::vector<uint8_t> W = bytes_of(pow2 ? Mi.low_bits(32 * tg.Lraw) : BigU::mod(Mi, T), nbytes);
    const uint64_t F = (1ull << ALPHA_SHIFT) / q;                       // < 2^19: three bytes
    for (uint32_t b = 0; b < 4; ++b) {                                  // byte b of y_i weighs 2^(8 b)
      for (uint32_t e = b; e < nbytes; ++e) put(4 * i + b, CRT_ALPHA_COLS + e, W[e - b]);
      for (uint32_t cc = 0; cc < 3; ++cc) put(4 * i + b, b + cc, (uint8_t)(F >> (8 * cc)));
    }
    const uint32_t ninv = powmod(c->N % q, q - 2, q);
    const uint32_t r32 = (uint32_t)((1ull << 32) % q);
    const uint32_t sc = mulmod(mulmod(ninv, inv, q), r32, q);
    scale[i] = make_uint2(sc, shoup(sc, q));
  }
  std::vector<uint32_t> negM(tg.Lraw, 0u);
  {
    BigU Mt = pow2 ? M.low_bits(32 * tg.Lraw) : BigU::mod(M, T);
    BigU neg;
    if (!Mt.is_zero()) { neg = T; neg.sub(Mt); }
    neg.to_limbs(negM.data(), negM.size());
  }
  cudaError_t e = upload(c, &tg.d_B, img);
  if (e != cudaSuccess) return e;
  if ((e = upload(c, &tg.d_negM, negM)) != cudaSuccess) return e;
  if (scaled_image) {                                                   // the second factor's decompose carries the final constant
    const std::vector<uint8_t> di = dec_image(c, K, &scale);
    if ((e = upload(c, &tg.d_decB_scaled, di)) != cudaSuccess) return e;
  }
  if (pow2 && K <= SMALL_K && tg.Lraw <= SMALL_LIMBS) {                 // limb form of the constants for the CUDA-core CRT
    std::vector<uint32_t> wl((size_t)(K + 1) * tg.Lraw, 0u);
    for (uint32_t i = 0; i < K; ++i) {
      BigU Mi = M;
      Mi.divmod_small(c->h_q[i]);
      Mi.low_bits(32 * tg.Lraw).to_limbs(wl.data() + (size_t)i * tg.Lraw, tg.Lraw);
    }
    for (uint32_t l = 0; l < tg.Lraw; ++l) wl[(size_t)K * tg.Lraw + l] = negM[l];
    if ((e = upload(c, &tg.d_Wlimbs, wl)) != cudaSuccess) return e;
  }
  return upload(c, &tg.d_scale, scale);
}

// bits [lo, lo + n) of x
static BigU bit_range(const BigU& x, uint32_t lo, uint32_t n) {
  BigU r;
  r.v.assign((n + 31) / 32, 0u);
  for (uint32_t i = 0; i < n; ++i)
    if (x.bit(lo + i)) r.v[i / 32] |= 1u << (i % 32);
  r.trim();
  return r;
}

// The CKKS relin target in its "top" form (fhe_internal.cuh): image columns 0..7 alpha, 8..31 the byte
// positions of sum_i y_i Wt_i (Wt_i = top TOP_BITS bits of W_i mod 2^logP), 32.. those of sum_i y_i Wh_i mod 2^(32 L)
// (Wh_i = W_i >> logP).  The negM table is [Nt (TOP_LIMBS) | Nh (L)].  The full constants go along for the exact path.
static cudaError_t build_target_top(Context* c, CrtTarget& tg, uint32_t K, uint32_t logP, uint32_t logQ) {
  constexpr uint32_t NC = 64;
  const uint32_t L = (logQ + 31) / 32;
  tg.K = K;
  tg.KB = (4 * K + 31) / 32 * 32;
  tg.top = true;
  tg.Lraw = TOP_LIMBS + L;
  tg.Lx = tg.Lraw + 1;
  tg.Lfull = (logP + logQ + 31) / 32;
  const uint32_t hbytes = 4 * L, tbytes = TOP_BITS / 8;
  const uint32_t ncols = CRT_ALPHA_COLS + 4 * TOP_LIMBS + hbytes;
  tg.nchunks = (ncols + NC - 1) / NC;
  BigU M((uint64_t)1);
  for (uint32_t i = 0; i < K; ++i) M.mul_small(c->h_q[i]);
  const size_t img_cols = (size_t)tg.nchunks * NC;
  std::vector<uint8_t> img((size_t)tg.KB * img_cols, 0);
  auto put = [&](uint32_t kb, uint32_t col, uint8_t v) { img[((size_t)(kb / 16) * img_cols + col) * 16 + kb % 16] = v; };
  std::vector<uint2> scale(K);
  std::vector<uint32_t> wfull((size_t)K * tg.Lfull, 0u);
  for (uint32_t i = 0; i < K; ++i) {
    const uint32_t q = c->h_q[i];
    BigU Mi = M;
    if (Mi.divmod_small(q) != 0) return cudaErrorUnknown;
    const uint32_t inv = powmod(Mi.mod_small(q), q - 2, q);            // (M/q_i)^-1 mod q_i
    const BigU W = Mi.low_bits(logP + logQ);
    W.to_limbs(wfull.data() + (size_t)i * tg.Lfull, tg.Lfull);
    const std::vector<uint8_t> Wt = bytes_of(bit_range(W, logP - TOP_BITS, TOP_BITS), tbytes);
    const std::vector<uint8_t> Wh = bytes_of(bit_range(W, logP, logQ), hbytes);
    const uint64_t F = (1ull << ALPHA_SHIFT) / q;
    for (uint32_t b = 0; b < 4; ++b) {                                  // byte b of y_i weighs 2^(8 b)
      for (uint32_t cc = 0; cc < 3; ++cc) put(4 * i + b, b + cc, (uint8_t)(F >> (8 * cc)));
      for (uint32_t e = 0; e < tbytes; ++e) put(4 * i + b, CRT_ALPHA_COLS + b + e, Wt[e]);
      for (uint32_t e = b; e < hbytes; ++e) put(4 * i + b, CRT_ALPHA_COLS + 4 * TOP_LIMBS + e, Wh[e - b]);
    }
    const uint32_t ninv = powmod(c->N % q, q - 2, q);
    const uint32_t r32 = (uint32_t)((1ull << 32) % q);
    const uint32_t sc = mulmod(mulmod(ninv, inv, q), r32, q);
    scale[i] = make_uint2(sc, shoup(sc, q));
  }
  std::vector<uint32_t> negM(tg.Lraw, 0u), negfull(tg.Lfull, 0u);
  {
    const BigU T = BigU::pow2(logP + logQ);
    BigU Mt = M.low_bits(logP + logQ), neg;
    if (!Mt.is_zero()) { neg = T; neg.sub(Mt); }
    neg.to_limbs(negfull.data(), negfull.size());
    bit_range(neg, logP - TOP_BITS, TOP_BITS).to_limbs(negM.data(), TOP_LIMBS);
    bit_range(neg, logP, logQ).to_limbs(negM.data() + TOP_LIMBS, L);
  }
  cudaError_t e = upload(c, &tg.d_B, img);
  if (e != cudaSuccess) return e;
  if ((e = upload(c, &tg.d_negM, negM)) != cudaSuccess) return e;
  if ((e = upload(c, &tg.d_Wfull, wfull)) != cudaSuccess) return e;
  if ((e = upload(c, &tg.d_negMfull, negfull)) != cudaSuccess) return e;
  return upload(c, &tg.d_scale, scale);
}

static uint64_t mu1_of(const BigU& m) {   // floor(2^(bits(m)+62) / m), in (2^62, 2^63]
  BigU q, r;
  BigU::divmod(BigU::pow2(m.bits() + 62), m, q, r);
  return (uint64_t)q.limb(0) | ((uint64_t)q.limb(1) << 32);
}

static fhe_status fail(Context* c, fhe_status st, const std::string& msg) {
  if (c) c->err = msg;
  g_create_err = msg;
  return st;
}

static void destroy(Context* c) {
  if (!c) return;
  for (void* p : c->allocs) cudaFree(p);
  if (c->d_evk_hat) cudaFree(c->d_evk_hat);
  for (int i = 0; i < Context::MAX_ROT_KEYS; ++i) if (c->d_rot_hat[i]) cudaFree(c->d_rot_hat[i]);
  for (auto& e : c->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  if (c->s_h2d) cudaStreamDestroy(c->s_h2d);
  if (c->s_d2h) cudaStreamDestroy(c->s_d2h);
  if (c->ev_start) cudaEventDestroy(c->ev_start);
  for (int i = 0; i < Context::HOST_PIECES; ++i) {
    if (c->ev_in[i]) cudaEventDestroy(c->ev_in[i]);
    if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
  }
  delete c;
}

static fhe_status create(Context** out, uint32_t N, uint32_t logQ, uint32_t logP, uint64_t t) {
  if (!out) return fail(nullptr, FHE_ERR_ARG, "out is NULL");
  *out = nullptr;
  if (N < 256 || N > 65536 || (N & (N - 1))) return fail(nullptr, FHE_ERR_UNSUPPORTED, "N must be a power of two in [2^8, 2^16]");
  if (logQ < 32 || logQ > 2560 || logP < 1 || logP > 2560) return fail(nullptr, FHE_ERR_UNSUPPORTED, "logQ in [32,2560], logP in [1,2560]");
  if (logQ + logP + 2 > 3328) return fail(nullptr, FHE_ERR_UNSUPPORTED, "logQ + logP too large (evk wider than 3326 bits)");
  if (t != 0 && ((t & 1) == 0 || t < 3 || t >= (1ull << 31))) return fail(nullptr, FHE_ERR_UNSUPPORTED, "BGV t must be odd, 3 <= t < 2^31");
  Context* c = new (std::nothrow) Context();
  if (!c) return fail(nullptr, FHE_ERR_NOMEM, "host allocation failed");
  c->N = N; c->logQ = logQ; c->logP = logP; c->t = t;
  while ((1u << c->logN) < N) ++c->logN;
  int dev = 0;
  cudaError_t e = cudaGetDevice(&dev);
  c->device = dev;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&c->n_sm, cudaDevAttrMultiProcessorCount, dev);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_start, cudaEventDisableTiming);
  for (int i = 0; i < Context::HOST_PIECES && e == cudaSuccess; ++i) {
    e = cudaEventCreateWithFlags(&c->ev_in[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming);
  }
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); destroy(c); return fail(nullptr, FHE_ERR_CUDA, "no CUDA device: " + m); }

  const BigU Q = make_modulus(logQ, t), P = make_modulus(logP, t);
  const BigU PQ = BigU::mul(P, Q);
  auto bits_m1 = [](const BigU& m) { BigU x = m; x.sub(BigU((uint64_t)1)); return x.bits(); };
  c->bitsQ = bits_m1(Q); c->bitsP = bits_m1(P); c->bitsPQ = bits_m1(PQ);
  c->L = (c->bitsQ + 31) / 32; c->L_P = (c->bitsP + 31) / 32; c->L_PQ = (c->bitsPQ + 31) / 32;
  c->h_Q.assign(c->L + 2, 0); Q.to_limbs(c->h_Q.data(), c->L + 2);
  c->h_P.assign(c->L_P + 2, 0); P.to_limbs(c->h_P.data(), c->L_P + 2);
  c->h_PQ.assign(c->L_PQ + 2, 0); PQ.to_limbs(c->h_PQ.data(), c->L_PQ + 2);

  // ---- primes: 30-bit, = 1 (mod 2^17), descending from 2^30; bounds DESIGN.md 3-A5 ------------
  {
    BigU NQ2 = BigU::mul(Q, Q); NQ2.mul_small(N);
    BigU b_pm = NQ2; b_pm.mul_small(4);
    BigU b_t = NQ2; b_t.mul_small(8);
    BigU b_r = BigU::mul(Q, PQ); b_r.mul_small(N); b_r.mul_small(4);
    c->K_pm = primes_for(c->h_q, b_pm);
    c->K1 = primes_for(c->h_q, b_t);
    c->K2 = primes_for(c->h_q, b_r);
    c->Kmax = (uint32_t)c->h_q.size();
  }
  const uint32_t Kmax = c->Kmax;

  // ---- per-prime constants and twiddle tables ---------------------------------------------------------------------
  std::vector<uint32_t> qn(Kmax);
  std::vector<uint2> qmu(Kmax);
  std::vector<uint4> qsmall(Kmax);
  std::vector<uint2> scale_plain(Kmax);
  // decompose constants: widest input is the evk (L_PQ limbs) or what fhe_debug_decompose may pass (MAX_LIMBS_IN)
  c->dec_KBimg = (4 * MAX_LIMBS_IN + 31) / 32 * 32;
  c->dec_cols = (Kmax + 15) / 16 * DEC_NC;               // image [dec_KBimg / 16][dec_cols][16 bytes] (pipe.cuh)
  c->h_psi.resize(Kmax);
  std::vector<uint2> twf((size_t)Kmax * N);             // the one twiddle table: the inverse stages read it mirrored (kernels_ntt.cu, bf_inv)
  std::vector<uint32_t> pw(N);
  for (uint32_t j = 0; j < Kmax; ++j) {
    const uint32_t q = c->h_q[j];
    uint32_t inv = 1;                                  // q^-1 mod 2^32 by Newton iteration
    for (int it = 0; it < 5; ++it) inv *= 2u - q * inv;
    qn[j] = 0u - inv;
    qmu[j] = make_uint2(q, (uint32_t)((1ull << 53) / q));
    qsmall[j] = make_uint4(q, (uint32_t)((1ull << 32) % q), (uint32_t)((1ull << 61) / q), (uint32_t)((1ull << ALPHA_SHIFT) / q));
    uint32_t psi = 0;
    for (uint32_t g = 2; g < 2000 && !psi; ++g) {
      uint32_t cand = powmod(g, (q - 1) / (2 * N), q);
      if (powmod(cand, N, q) == q - 1) psi = cand;     // order exactly 2N
    }
    if (!psi) { destroy(c); return fail(nullptr, FHE_ERR_UNSUPPORTED, "no primitive root found"); }
    c->h_psi[j] = psi;
    pw[0] = 1;
    for (uint32_t k = 1; k < N; ++k) pw[k] = mulmod(pw[k - 1], psi, q);
    for (uint32_t k = 0; k < N; ++k) {
      uint32_t r = bitrev(k, c->logN);
      twf[(size_t)j * N + k] = make_uint2(pw[r], shoup(pw[r], q));
    }
    uint32_t ninv = powmod(N % q, q - 2, q);
    scale_plain[j] = make_uint2(ninv, shoup(ninv, q));
  }
#define UP(dst, vec)                                                                                   \
  if ((e = upload(c, &c->dst, vec)) != cudaSuccess) {                                                  \
    std::string m = cudaGetErrorString(e); destroy(c); return fail(nullptr, FHE_ERR_CUDA, "upload failed: " + m); }
  UP(d_q, c->h_q) UP(d_qinv_neg, qn) UP(d_qmu, qmu) UP(d_qsmall, qsmall) UP(d_tw_fwd, twf)
  {
    const uint32_t kd = Kmax < SMALL_DEC_K ? Kmax : SMALL_DEC_K;
    std::vector<uint32_t> pw32((size_t)kd * SMALL_LIMBS);
    for (uint32_t j = 0; j < kd; ++j) {
      const uint32_t q = c->h_q[j], c32 = (uint32_t)((1ull << 32) % q);
      uint32_t v = 1;
      for (uint32_t l = 0; l < SMALL_LIMBS; ++l) { pw32[(size_t)j * SMALL_LIMBS + l] = v; v = mulmod(v, c32, q); }
    }
    UP(d_pow32q, pw32)
  }
  const std::vector<uint8_t> decB = dec_image(c, Kmax, nullptr);
  UP(d_scale_plain, scale_plain) UP(d_decB, decB)

  // ---- CRT targets -------------------------------------------------------------------------------------------------
  const bool ckks = (t == 0);
  if ((e = build_target(c, c->tgt_pm, c->K_pm, ckks, logQ, Q, c->L + 2, true)) != cudaSuccess ||
      (e = build_target(c, c->tgt_tensor, c->K1, ckks, logQ, Q, c->L + 2, true)) != cudaSuccess ||
      (e = (ckks && logP >= TOP_BITS) ? build_target_top(c, c->tgt_relin, c->K2, logP, logQ)
                                      : build_target(c, c->tgt_relin, c->K2, ckks, logQ + logP, PQ, c->L_PQ + 2)) != cudaSuccess) {
    std::string m = cudaGetErrorString(e); destroy(c); return fail(nullptr, FHE_ERR_CUDA, "CRT table build failed: " + m);
  }

  // ---- post-processing parameters -----------------------------------------------------------------------------------
  PostParams pp;
  memset(&pp, 0, sizeof(pp));
  pp.L = c->L; pp.L_PQ = c->L_PQ; pp.L_P = c->L_P; pp.logQ = logQ; pp.logP = logP;
  pp.bitsQ = Q.bits(); pp.bitsP = P.bits(); pp.bitsPQ = PQ.bits();   // significant bits of the moduli themselves
  if (!ckks) {
    std::vector<uint32_t> hQ(c->L + 2), hP(c->L_P + 2), hPQ(c->L_PQ + 2);
    Q.to_limbs(hQ.data(), hQ.size()); P.to_limbs(hP.data(), hP.size()); PQ.to_limbs(hPQ.data(), hPQ.size());
    UP(d_Qlimbs, hQ) UP(d_Plimbs, hP) UP(d_PQlimbs, hPQ)
    BigU mu, r;
    BigU::divmod(BigU::pow2(32 * c->L_PQ), P, mu, r);
    std::vector<uint32_t> hmu(mu.v.size() + 1, 0u);
    mu.to_limbs(hmu.data(), hmu.size());
    UP(d_muP, hmu)
    pp.muP_limbs = (uint32_t)mu.v.size();
    pp.g_limbs = c->L_PQ - c->L_P;
    pp.scratch_limbs = (pp.g_limbs + 1) + pp.muP_limbs + 1;   // product q1 * mu of the divide-by-P (kernels_crt.cu)
    const uint32_t tt = (uint32_t)t;
    std::vector<uint32_t> p32(c->L_P + 2);
    uint32_t cur = 1 % tt, b32 = (uint32_t)((1ull << 32) % tt);
    for (uint32_t i = 0; i < c->L_P; ++i) { p32[i] = cur; cur = mulmod(cur, b32, tt); }
    p32[c->L_P] = P.mod_small(tt);                       // slot L_P holds P mod t
    UP(d_pow32_t, p32)
    pp.d_Q = c->d_Qlimbs; pp.d_P = c->d_Plimbs; pp.d_PQ = c->d_PQlimbs; pp.d_muP = c->d_muP; pp.d_pow32_t = c->d_pow32_t;
    pp.mu1_Q = mu1_of(Q); pp.mu1_PQ = mu1_of(PQ);
    {
      const uint64_t eP = modulus_offset(logP, t);
      uint32_t be = 0;
      while (be < 64 && (eP >> be)) ++be;
      pp.eP = (uint32_t)eP;
      pp.fold_div = (eP >> 32) == 0 && logP >= 96 && be + pp.bitsQ + 1 <= logP + 60 ? 1u : 0u;
      if (pp.scratch_limbs < c->L_PQ + 4 - (logP >> 5) + 2) pp.scratch_limbs = c->L_PQ + 4 - (logP >> 5) + 2;   // A of V itself: Lx - wq limbs, Lx <= L_PQ + 4
      pp.mu_t = tt < (1u << 31) ? ~0ull / tt : 0ull;
      const uint64_t eQ = modulus_offset(logQ, t);
      pp.eQ = (uint32_t)eQ;
      pp.fold_modq = eQ < (1ull << 22) && logQ >= 64 ? 1u : 0u;
      {
        // V < 2^(bitsPQ + 40): A = V >> logP has at most ba bits, the second fold's quotient j at most bj, the quotient's own
        // excess over 2^logQ at most bx
        uint32_t bq2 = 0;
        while (bq2 < 64 && (eQ >> bq2)) ++bq2;
        const int ba = (int)pp.bitsPQ + 40 - (int)logP, bj = ba + (int)be - (int)logP, bx = ba - (int)logQ;
        pp.fold_full = pp.fold_div && pp.fold_modq && bj <= 95 && (bj <= 0 || bj + (int)be < (int)logP) && bx + (int)bq2 <= 63 ? 1u : 0u;
      }
    }
    pp.t = tt; pp.Pinv_t = powmod(P.mod_small(tt), (uint64_t)tt - 2, tt);
    // t need not be prime: fall back to a search-free extended Euclid if Fermat fails
    if (mulmod(pp.Pinv_t, P.mod_small(tt), tt) != 1 % tt) {
      int64_t a = P.mod_small(tt), b = tt, x0 = 1, x1 = 0;
      while (b) { int64_t qq = a / b, tmp = a - qq * b; a = b; b = tmp; tmp = x0 - qq * x1; x0 = x1; x1 = tmp; }
      if (a != 1) { destroy(c); return fail(nullptr, FHE_ERR_UNSUPPORTED, "gcd(P, t) != 1"); }
      pp.Pinv_t = (uint32_t)((x0 % (int64_t)tt + tt) % tt);
    }
  }
#undef UP
  c->post_pm = pp;     c->post_pm.mode = ckks ? POST_CKKS_MASK : POST_BGV_MODQ;
  c->post_tensor = c->post_pm;
  c->post_relin = pp;  c->post_relin.mode = ckks ? POST_CKKS_RELIN : POST_BGV_RELIN;
  // A target whose constant matrix or accumulators exceed shared / tensor memory disables the calls that need it
  // (FHE_ERR_UNSUPPORTED from those calls); the context is refused only when not even the plain product fits.
  c->fit_pm = crt_target_fits(c->tgt_pm, c->post_pm);
  c->fit_tensor = crt_target_fits(c->tgt_tensor, c->post_tensor);
  c->fit_relin = crt_target_fits(c->tgt_relin, c->post_relin);
  if (!c->fit_pm) {
    destroy(c);
    return fail(nullptr, FHE_ERR_UNSUPPORTED, "parameters too large for the conversion pipeline (TMEM columns / shared memory)");
  }
  e = cudaDeviceSynchronize();
  if (e != cudaSuccess) { std::string m = cudaGetErrorString(e); destroy(c); return fail(nullptr, FHE_ERR_CUDA, m); }
  *out = c;
  return FHE_OK;
}

}  // namespace fhe

using namespace fhe;

extern "C" {

// fhe_ctx stays an incomplete type: an fhe_ctx* is a fhe::Context* in disguise.

fhe_status fhe_ctx_create(fhe_ctx** out, uint32_t N, uint32_t logQ, uint32_t logP, uint64_t t) {
  try {
    return create(reinterpret_cast<Context**>(out), N, logQ, logP, t);
  } catch (const std::bad_alloc&) {
    g_create_err = "host allocation failed";
    return FHE_ERR_NOMEM;
  } catch (...) {
    g_create_err = "unexpected host exception";
    return FHE_ERR_ARG;
  }
}
void fhe_ctx_destroy(fhe_ctx* ctx) { destroy(reinterpret_cast<Context*>(ctx)); }

fhe_status fhe_ctx_info(const fhe_ctx* ctx, fhe_info* o) {
  if (!ctx || !o) return FHE_ERR_ARG;
  const Context* c = reinterpret_cast<const Context*>(ctx);
  o->N = c->N; o->logQ = c->logQ; o->logP = c->logP; o->t = c->t; o->bitsQ = c->bitsQ; o->bitsPQ = c->bitsPQ;
  o->L = c->L; o->L_PQ = c->L_PQ; o->K_pm = c->K_pm; o->K1 = c->K1; o->K2 = c->K2; o->n_sm = (uint32_t)c->n_sm;
  return FHE_OK;
}
const char* fhe_last_error(const fhe_ctx* ctx) {
  if (!ctx) return g_create_err.c_str();
  return reinterpret_cast<const Context*>(ctx)->err.c_str();
}
fhe_status fhe_get_modulus(const fhe_ctx* ctx, int which, uint32_t* h, uint32_t n) {
  if (!ctx || !h) return FHE_ERR_ARG;
  const Context* c = reinterpret_cast<const Context*>(ctx);
  const std::vector<uint32_t>& v = which == 0 ? c->h_Q : which == 1 ? c->h_P : c->h_PQ;
  if (which < 0 || which > 2) return FHE_ERR_ARG;
  size_t need = v.size();
  while (need && v[need - 1] == 0) --need;
  if (n < need) return FHE_ERR_ARG;
  for (uint32_t i = 0; i < n; ++i) h[i] = i < v.size() ? v[i] : 0u;
  return FHE_OK;
}
fhe_status fhe_debug_primes(const fhe_ctx* ctx, uint32_t* h_q, uint32_t* h_psi, uint32_t count) {
  if (!ctx || !h_q || !h_psi) return FHE_ERR_ARG;
  const Context* c = reinterpret_cast<const Context*>(ctx);
  if (count > c->Kmax) return FHE_ERR_ARG;
  for (uint32_t i = 0; i < count; ++i) { h_q[i] = c->h_q[i]; h_psi[i] = c->h_psi[i]; }
  return FHE_OK;
}
uint64_t fhe_debug_launch_count(const fhe_ctx* ctx) {
  return ctx ? reinterpret_cast<const Context*>(ctx)->launches : 0;
}
fhe_status fhe_debug_timing(fhe_ctx* ctx, int enable) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = reinterpret_cast<Context*>(ctx);
  for (auto& e : c->events) { cudaEventDestroy(e.a); cudaEventDestroy(e.b); }
  c->events.clear();
  c->timing = enable != 0;
  return FHE_OK;
}
fhe_status fhe_debug_timing_read(fhe_ctx* ctx, int kernel_class, double* ms_total, uint64_t* launches) {
  if (!ctx || !ms_total || !launches || kernel_class < 0 || kernel_class >= KC_COUNT) return FHE_ERR_ARG;
  Context* c = reinterpret_cast<Context*>(ctx);
  double tot = 0;
  uint64_t n = 0;
  for (auto& e : c->events) {
    if (e.cls != kernel_class) continue;
    cudaError_t st = cudaEventSynchronize(e.b);
    float ms = 0;
    if (st == cudaSuccess) st = cudaEventElapsedTime(&ms, e.a, e.b);
    if (st != cudaSuccess) { c->err = cudaGetErrorString(st); return FHE_ERR_CUDA; }
    tot += ms;
    ++n;
  }
  *ms_total = tot;
  *launches = n;
  return FHE_OK;
}

}  // extern "C"
