// kernels_elem.cu -- NEXT-1: the coefficient-wise ciphertext operations the paper lists by name
// (add_pairwise_into, sub_pairwise_into, negate_pairwise_into) and the level drop
// (moddownBy_pairwise_into) on limb-major polynomials [L][N] with canonical coefficients in [0, Q).
// HBM-bound streaming kernels: one thread per coefficient, so every limb access of a warp is one 128-byte line; the
// carry / borrow runs along the limbs inside the thread.
//   CKKS (Q = 2^logQ):  the sum / difference wraps mod 2^(32 L) by itself; the top limb is masked.
//   BGV  (odd Q):       a + b in [0, 2Q): subtract Q when >= Q; a - b: add Q on borrow; -a = Q - a for a != 0.
//                       The comparison with Q needs all limbs, so the coefficient is kept in a local array.
#include "fhe_internal.cuh"

namespace fhe {

constexpr uint32_t ELEM_MAX_LIMBS = 88;   // logQ <= 2560 (+ one limb for an odd Q just above 2^logQ)

enum ElemOp : int { EL_ADD = 0, EL_SUB = 1, EL_NEG = 2, EL_MODDOWN = 3 };

__device__ __forceinline__ uint32_t top_mask32(uint32_t bits) { return (bits & 31) ? ((1u << (bits & 31)) - 1u) : 0xFFFFFFFFu; }

template <int OP>
__global__ void __launch_bounds__(256)
elem_ckks_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ a, const uint32_t* __restrict__ b, uint32_t N,
                 uint32_t L, uint32_t bits) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const size_t base = (size_t)poly * L * N + n;
  const uint32_t Lb = (bits + 31) / 32, tm = top_mask32(bits);     // limbs that hold bits; the rest of the L limbs are zero
  uint32_t carry = OP == EL_NEG ? 1u : 0u;                          // -a = ~a + 1
  auto limb = [&](uint32_t l) {
    uint32_t v = 0;
    if (l < Lb) {
      const uint32_t x = a[base + (size_t)l * N];
      if (OP == EL_ADD) {
        const uint64_t s = (uint64_t)x + b[base + (size_t)l * N] + carry;
        v = (uint32_t)s; carry = (uint32_t)(s >> 32);
      } else if (OP == EL_SUB) {
        const uint64_t d = (uint64_t)x - b[base + (size_t)l * N] - carry;   // >= -2^32: the borrow is the sign
        v = (uint32_t)d; carry = (uint32_t)(d >> 63);
      } else if (OP == EL_NEG) {
        const uint64_t s = (uint64_t)(~x) + carry;
        v = (uint32_t)s; carry = (uint32_t)(s >> 32);
      } else {
        v = x;
      }
      if (l == Lb - 1) v &= tm;
    }
    out[base + (size_t)l * N] = v;
  };
  if constexpr (OP == EL_MODDOWN) {                                 // measured: a deeper unroll helps the copy, hurts add / sub
#pragma unroll 8
    for (uint32_t l = 0; l < L; ++l) limb(l);
  } else {
    for (uint32_t l = 0; l < L; ++l) limb(l);
  }
}

template <int OP>
__global__ void __launch_bounds__(256)
elem_bgv_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ a, const uint32_t* __restrict__ b,
                const uint32_t* __restrict__ Q, uint32_t N, uint32_t L) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const size_t base = (size_t)poly * L * N + n;
  uint32_t r[ELEM_MAX_LIMBS];
  if (OP == EL_ADD) {
    uint32_t carry = 0;
    for (uint32_t l = 0; l < L; ++l) {
      const uint64_t s = (uint64_t)a[base + (size_t)l * N] + b[base + (size_t)l * N] + carry;
      r[l] = (uint32_t)s; carry = (uint32_t)(s >> 32);
    }
    bool ge = carry != 0;                                           // sum >= 2^(32 L) > Q
    if (!ge) {
      ge = true;
      for (uint32_t l = L; l-- > 0;) { const uint32_t q = __ldg(Q + l); if (r[l] != q) { ge = r[l] > q; break; } }
    }
    uint32_t borrow = 0;
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = r[l];
      if (ge) { const uint32_t q = __ldg(Q + l); const uint32_t d = v - q, d2 = d - borrow; borrow = (v < q) | (d < borrow); v = d2; }
      out[base + (size_t)l * N] = v;
    }
  } else {                                                          // a - b (EL_NEG: 0 - a)
    uint32_t borrow = 0;
    for (uint32_t l = 0; l < L; ++l) {
      const uint32_t x = OP == EL_NEG ? 0u : a[base + (size_t)l * N];
      const uint32_t y = OP == EL_NEG ? a[base + (size_t)l * N] : b[base + (size_t)l * N];
      const uint32_t d = x - y, d2 = d - borrow;
      borrow = (x < y) | (d < borrow);
      r[l] = d2;
    }
    uint32_t carry = 0;
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = r[l];
      if (borrow) { const uint64_t s = (uint64_t)v + __ldg(Q + l) + carry; v = (uint32_t)s; carry = (uint32_t)(s >> 32); }
      out[base + (size_t)l * N] = v;
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// NEXT-2: Galois automorphism sigma_k: a(X) -> a(X^k) mod (X^N + 1), k odd (rotation of the CKKS slots; k = 2N - 1 is
// the conjugation).  Coefficient i moves to position i k mod 2N, with a sign flip when that is
// >= N.  Gather form: out[n] = a[i] for i' = n k^-1 mod 2N < N (i = i'), else -a[i' - N].  Ciphertext component 0 goes
// to slot 0 of the triple, component 1 to slot 2, slot 1 is zeroed: the key switch adds (round(sigma(c1) rk / P)) to
// (sigma(c0), 0).  Reads are a permutation (one 32-byte sector per word); the kernel is a small part of a rotation.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
automorphism_kernel(uint32_t* __restrict__ out3, const uint32_t* __restrict__ in2, const uint32_t* __restrict__ Q, uint32_t N,
                    uint32_t L, uint32_t bits, uint32_t kinv, uint32_t ckks) {
  const uint32_t bpp = N / 256;
  const uint32_t item = blockIdx.x / (3 * bpp), rem = blockIdx.x % (3 * bpp), slot = rem / bpp;
  const uint32_t n = (rem % bpp) * 256 + threadIdx.x;
  uint32_t* dst = out3 + ((size_t)item * 3 + slot) * L * N + n;
  if (slot == 1) {
    for (uint32_t l = 0; l < L; ++l) dst[(size_t)l * N] = 0;
    return;
  }
  const uint32_t ip = (uint32_t)(((uint64_t)n * kinv) & (2 * N - 1));
  const bool neg = ip >= N;
  const uint32_t* src = in2 + ((size_t)item * 2 + (slot ? 1 : 0)) * L * N + (neg ? ip - N : ip);
  if (!neg) {
    for (uint32_t l = 0; l < L; ++l) dst[(size_t)l * N] = src[(size_t)l * N];
    return;
  }
  if (ckks) {                                                       // -a mod 2^bits: two's complement, top limb masked
    const uint32_t Lb = (bits + 31) / 32, tm = top_mask32(bits);
    uint32_t carry = 1;
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = 0;
      if (l < Lb) {
        const uint64_t s = (uint64_t)(~src[(size_t)l * N]) + carry;
        v = (uint32_t)s; carry = (uint32_t)(s >> 32);
        if (l == Lb - 1) v &= tm;
      }
      dst[(size_t)l * N] = v;
    }
  } else {                                                          // Q - a, and 0 stays 0
    uint32_t any = 0;
    for (uint32_t l = 0; l < L; ++l) any |= src[(size_t)l * N];
    uint32_t borrow = 0;
    for (uint32_t l = 0; l < L; ++l) {
      const uint32_t q = any ? __ldg(Q + l) : 0u, y = src[(size_t)l * N];
      const uint32_t d = q - y, d2 = d - borrow;
      borrow = (q < y) | (d < borrow);
      dst[(size_t)l * N] = d2;
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Multiplication by the monomial X^k, 0 <= k < 2N: a signed rotation of the coefficients (X^N = -1).  k = N/2 is the
// multiplication by the imaginary unit of the CKKS slots (imult_pairwise_into), k = 3N/2 its inverse.
// out[n] = a[n - k] for n >= k (mod 2N bookkeeping below), negated when the index wraps an odd number of times.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
monomial_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ in, const uint32_t* __restrict__ Q, uint32_t N,
                uint32_t L, uint32_t bits, uint32_t k, uint32_t ckks) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const uint32_t ip = (n + 2 * N - k) & (2 * N - 1);                // source index mod 2N: X^k X^ip = X^n
  const bool neg = ip >= N;
  const uint32_t* src = in + (size_t)poly * L * N + (neg ? ip - N : ip);
  uint32_t* dst = out + (size_t)poly * L * N + n;
  if (!neg) {
    for (uint32_t l = 0; l < L; ++l) dst[(size_t)l * N] = src[(size_t)l * N];
  } else if (ckks) {
    const uint32_t Lb = (bits + 31) / 32, tm = top_mask32(bits);
    uint32_t carry = 1;
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = 0;
      if (l < Lb) {
        const uint64_t s = (uint64_t)(~src[(size_t)l * N]) + carry;
        v = (uint32_t)s; carry = (uint32_t)(s >> 32);
        if (l == Lb - 1) v &= tm;
      }
      dst[(size_t)l * N] = v;
    }
  } else {
    uint32_t any = 0;
    for (uint32_t l = 0; l < L; ++l) any |= src[(size_t)l * N];
    uint32_t borrow = 0;
    for (uint32_t l = 0; l < L; ++l) {
      const uint32_t q = any ? __ldg(Q + l) : 0u, y = src[(size_t)l * N];
      const uint32_t d = q - y, d2 = d - borrow;
      borrow = (q < y) | (d < borrow);
      dst[(size_t)l * N] = d2;
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// NEXT-3, constants (addconst / multconst: names only; reading in DESIGN.md 3).
//   add_plain:   out = (c0 + m, c1): ciphertext i gets plaintext polynomial i / group added to component 0; component 1 is
//                copied (skipped in place).
//   mult_scalar: every coefficient times the integer k, |k| < 2^31.  x |k| has L + 1 limbs.  CKKS: the low logQ bits,
//                two's complement for k < 0.  BGV: Q = 2^logQ + e with 0 < e < 2^(logQ - 33) (the least odd integer above
//                2^logQ that is 1 mod t, checked by the caller), so floor(x |k| / Q) is h = floor(x |k| / 2^logQ) or
//                h - 1 (x |k| / 2^logQ - x |k| / Q < 2^31 e / 2^logQ < 1): r = x |k| - h Q, + Q when negative; Q - r for
//                k < 0 and r != 0.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
add_plain_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ ct, const uint32_t* __restrict__ pt,
                 const uint32_t* __restrict__ Q, uint32_t N, uint32_t L, uint32_t bits, uint32_t group, uint32_t ckks) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const size_t base = (size_t)poly * L * N + n;
  if (poly & 1) {                                                   // component 1
    if (out != ct)
      for (uint32_t l = 0; l < L; ++l) out[base + (size_t)l * N] = ct[base + (size_t)l * N];
    return;
  }
  const uint32_t* m = pt + (size_t)((poly >> 1) / group) * L * N + n;
  uint32_t carry = 0;
  if (ckks) {                                                       // streams: the sum wraps mod 2^(32 L), the top limb is masked
    const uint32_t Lb = (bits + 31) / 32, tm = top_mask32(bits);
#pragma unroll 8
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = 0;
      if (l < Lb) {
        const uint64_t s = (uint64_t)ct[base + (size_t)l * N] + m[(size_t)l * N] + carry;
        v = (uint32_t)s; carry = (uint32_t)(s >> 32);
        if (l == Lb - 1) v &= tm;
      }
      out[base + (size_t)l * N] = v;
    }
    return;
  }
  uint32_t r[ELEM_MAX_LIMBS];
  for (uint32_t l = 0; l < L; ++l) {
    const uint64_t s = (uint64_t)ct[base + (size_t)l * N] + m[(size_t)l * N] + carry;
    r[l] = (uint32_t)s; carry = (uint32_t)(s >> 32);
  }
  bool ge = carry != 0;
  if (!ge) {
    ge = true;
    for (uint32_t l = L; l-- > 0;) { const uint32_t q = __ldg(Q + l); if (r[l] != q) { ge = r[l] > q; break; } }
  }
  uint32_t borrow = 0;
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t v = r[l];
    if (ge) { const uint32_t q = __ldg(Q + l); const uint32_t d = v - q, d2 = d - borrow; borrow = (v < q) | (d < borrow); v = d2; }
    out[base + (size_t)l * N] = v;
  }
}

__global__ void __launch_bounds__(256)
mult_scalar_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ in, const uint32_t* __restrict__ Q, uint32_t N,
                   uint32_t L, uint32_t bits, uint32_t kabs, uint32_t kneg, uint32_t ckks) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const size_t base = (size_t)poly * L * N + n;
  uint32_t carry = 0;
  if (ckks) {                                                       // streams: product limb, two's complement, mask
    const uint32_t Lb = (bits + 31) / 32, tm = top_mask32(bits);
    uint32_t c1 = kneg;                                             // -v = ~v + 1
#pragma unroll 8
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = 0;
      if (l < Lb) {
        const uint64_t pr = (uint64_t)in[base + (size_t)l * N] * kabs + carry;
        v = (uint32_t)pr; carry = (uint32_t)(pr >> 32);
        if (kneg) { const uint64_t s = (uint64_t)(~v) + c1; v = (uint32_t)s; c1 = (uint32_t)(s >> 32); }
        if (l == Lb - 1) v &= tm;
      }
      out[base + (size_t)l * N] = v;
    }
    return;
  }
  uint32_t r[ELEM_MAX_LIMBS + 1];
  for (uint32_t l = 0; l < L; ++l) {
    const uint64_t s = (uint64_t)in[base + (size_t)l * N] * kabs + carry;
    r[l] = (uint32_t)s; carry = (uint32_t)(s >> 32);
  }
  r[L] = carry;
  const uint32_t w = bits >> 5, sh = bits & 31;                     // h = bits [logQ, logQ + 32) of the product
  uint32_t h = r[w] >> sh;
  if (sh && w + 1 <= L) h |= r[w + 1] << (32 - sh);
  // r -= h Q over L + 1 limbs (Q has L limbs); the result is in (-Q, Q): its sign is the final borrow
  uint64_t mc = 0;
  uint32_t borrow = 0;
  for (uint32_t l = 0; l <= L; ++l) {
    const uint64_t pq = (l < L ? (uint64_t)__ldg(Q + l) * h : 0ull) + mc;
    const uint32_t sub = (uint32_t)pq; mc = pq >> 32;
    const uint32_t v = r[l], d = v - sub, d2 = d - borrow;
    borrow = (v < sub) | (d < borrow);
    r[l] = d2;
  }
  if (borrow) {                                                     // negative: add Q back once
    uint32_t c2 = 0;
    for (uint32_t l = 0; l < L; ++l) { const uint64_t s = (uint64_t)r[l] + __ldg(Q + l) + c2; r[l] = (uint32_t)s; c2 = (uint32_t)(s >> 32); }
  }
  uint32_t any = 0;
  for (uint32_t l = 0; l < L; ++l) any |= r[l];
  const bool flip = kneg && any;
  uint32_t b2 = 0;
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t v = r[l];
    if (flip) { const uint32_t q = __ldg(Q + l); const uint32_t d = q - v, d2 = d - b2; b2 = (q < v) | (d < b2); v = d2; }
    out[base + (size_t)l * N] = v;
  }
}

// ------------------------------------------------------------------------------------------------------------------
// NEXT-4: BGV modulus switch (named only; reading DESIGN.md 3, A20).  Q = 2^logQ + e, Q' = 2^b + e'
// (both the least odd integer above the power of two that is 1 mod t, so e, e' < 2 t < 2^32).  Per coefficient c in [0, Q):
//     x = c Q',   r = x mod Q centred,   k = (-r Q^-1) mod t centred = (-r) mod t centred (Q = 1 mod t),
//     c' = ((x - r)/Q - k) mod Q'.
// The division by Q uses its shape instead of a general Barrett step:  x = h0 2^logQ + xl  gives  x = h0 Q + (xl - h0 e),
// and when z = xl - h0 e is negative, y = -z = j 2^logQ + yl = j Q + (yl - j e) moves j (< 2^35) or j + 1 more multiples of Q
// across; |j e| < 2^67 < Q (logQ >= 96 is required), so the remainder lands in [0, Q) without a loop.
// One thread per coefficient with the numbers in local arrays: a level drop happens once per multiplication depth, the
// kernel needs no tuning beyond coalesced limb accesses.
// ------------------------------------------------------------------------------------------------------------------
constexpr uint32_t MS_H = ELEM_MAX_LIMBS + 2, MS_X = 2 * ELEM_MAX_LIMBS + 6;

__global__ void __launch_bounds__(128)
modswitch_bgv_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ in, uint32_t N, uint32_t L, uint32_t logQ,
                     uint32_t e, uint32_t b, uint32_t e2, uint32_t t, uint64_t mu_t) {
  const uint32_t bpp = N / 128;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * 128 + threadIdx.x;
  const size_t base = (size_t)poly * L * N + n;
  const uint32_t wq = logQ >> 5, bq = logQ & 31, Lq = (logQ + 31) / 32;     // Q's power of two: limb wq, bit bq
  const uint32_t ws = b >> 5, bs = b & 31, L2 = b / 32 + 1;                 // Q' has b + 1 bits
  const uint32_t nx = L + L2 + 2;
  uint32_t x[MS_X], h[MS_H];
  for (uint32_t l = 0; l < nx; ++l) x[l] = 0;
  // ---- x = c e' + (c << b) ----
  {
    uint32_t carry = 0, cprev = 0, carry2 = 0;
    for (uint32_t l = 0; l <= L; ++l) {
      const uint32_t cl = l < L ? in[base + (size_t)l * N] : 0u;
      const uint64_t pr = (uint64_t)cl * e2 + carry + x[l];       // x[l] may already hold a limb of the shifted copy
      x[l] = (uint32_t)pr; carry = (uint32_t)(pr >> 32);
      const uint32_t v = bs ? (cl << bs) | (cprev >> (32 - bs)) : cl;
      cprev = cl;
      const uint64_t s = (uint64_t)x[l + ws] + v + carry2;        // ws >= 1: never the limb the product has just written
      x[l + ws] = (uint32_t)s; carry2 = (uint32_t)(s >> 32);
    }
    for (uint32_t l = L + 1; carry && l < nx; ++l) { const uint64_t s = (uint64_t)x[l] + carry; x[l] = (uint32_t)s; carry = (uint32_t)(s >> 32); }
    for (uint32_t l = L + ws + 1; carry2 && l < nx; ++l) { const uint64_t s = (uint64_t)x[l] + carry2; x[l] = (uint32_t)s; carry2 = (uint32_t)(s >> 32); }
  }
  // ---- h0 = x >> logQ (b + 2 bits), xl = x mod 2^logQ (left in x[0 .. Lq)) ----
  const uint32_t nh = (b + 2) / 32 + 1;
  for (uint32_t i = 0; i < nh; ++i) {
    const uint32_t lo = wq + i < nx ? x[wq + i] : 0u, hi = wq + i + 1 < nx ? x[wq + i + 1] : 0u;
    h[i] = bq ? (lo >> bq) | (hi << (32 - bq)) : lo;
  }
  h[nh] = 0;
  if (bq) x[Lq - 1] &= (1u << bq) - 1u;
  const uint32_t nz = (Lq > nh + 1 ? Lq : nh + 1) + 1;             // limbs of z = xl - h0 e (signed)
  for (uint32_t l = Lq; l < nz; ++l) x[l] = 0;
  uint32_t borrow = 0;
  {
    uint32_t mc = 0;
    for (uint32_t l = 0; l < nz; ++l) {
      const uint64_t pr = (l < nh ? (uint64_t)h[l] * e : 0ull) + mc;
      const uint32_t sub = (uint32_t)pr; mc = (uint32_t)(pr >> 32);
      const uint32_t v = x[l], d = v - sub, d2 = d - borrow;
      borrow = (v < sub) | (d < borrow);
      x[l] = d2;
    }
  }
  // ---- remainder in [0, Q) (x[0 .. Lq]) and quotient (h) ----
  uint64_t hdec = 0;                                               // what comes off h0
  if (borrow) {
    uint32_t c1 = 1;                                               // y = -z
    for (uint32_t l = 0; l < nz; ++l) { const uint64_t s = (uint64_t)(~x[l]) + c1; x[l] = (uint32_t)s; c1 = (uint32_t)(s >> 32); }
    const uint32_t j0 = wq < nz ? x[wq] : 0u, j1 = wq + 1 < nz ? x[wq + 1] : 0u, j2 = wq + 2 < nz ? x[wq + 2] : 0u;
    const uint64_t j = bq ? ((uint64_t)(j0 >> bq) | ((uint64_t)j1 << (32 - bq)) | ((uint64_t)j2 << (64 - bq))) : ((uint64_t)j0 | ((uint64_t)j1 << 32));
    if (bq) x[Lq - 1] &= (1u << bq) - 1u;                          // yl
    for (uint32_t l = Lq; l <= Lq; ++l) x[l] = 0;
    // w = yl - j e over Lq + 1 limbs (j e < 2^67)
    const uint64_t p0 = (uint64_t)(uint32_t)j * e, p1 = (j >> 32) * e + (p0 >> 32);
    const uint32_t je[3] = {(uint32_t)p0, (uint32_t)p1, (uint32_t)(p1 >> 32)};
    uint32_t bw = 0, any = 0;
    for (uint32_t l = 0; l <= Lq; ++l) {
      const uint32_t sub = l < 3 ? je[l] : 0u, v = x[l], d = v - sub, d2 = d - bw;
      bw = (v < sub) | (d < bw);
      x[l] = d2; any |= d2;
    }
    if (!bw && any) {                                              // w > 0: one more multiple, remainder Q - w
      hdec = j + 1;
      uint32_t b2 = 0;
      for (uint32_t l = 0; l <= Lq; ++l) {
        const uint32_t ql = (l == 0 ? e : 0u) + (l == wq ? 1u << bq : 0u), v = x[l], d = ql - v, d2 = d - b2;
        b2 = (ql < v) | (d < b2);
        x[l] = d2;
      }
    } else {                                                       // w <= 0: remainder -w
      hdec = j;
      uint32_t c2 = 1;
      for (uint32_t l = 0; l <= Lq; ++l) { const uint64_t s = (uint64_t)(~x[l]) + c2; x[l] = (uint32_t)s; c2 = (uint32_t)(s >> 32); }
    }
  }
  // ---- centre the remainder: r = rem - Q when 2 rem > Q (Q odd: no tie) ----
  bool negr;
  {
    int cmp = 0;
    for (uint32_t l = Lq + 1; l-- > 0 && cmp == 0;) {
      const uint32_t two = (x[l] << 1) | (l ? x[l - 1] >> 31 : 0u);
      const uint32_t ql = (l == 0 ? e : 0u) + (l == wq ? 1u << bq : 0u);
      if (two != ql) cmp = two > ql ? 1 : -1;
    }
    // bit 32 (Lq + 1) of 2 rem: rem < Q < 2^(32 Lq + 32 - 1) so x[Lq] < 2^31 and nothing is shifted out
    negr = cmp > 0;
  }
  uint32_t rt = 0;                                                 // rem mod t, then r mod t
  for (uint32_t l = Lq + 1; l-- > 0;) rt = horner_mod(rt, x[l], t, mu_t);
  if (negr) rt = rt ? rt - 1 : t - 1;                              // r = rem - Q, Q = 1 (mod t)
  const uint32_t k = rt ? t - rt : 0u;                             // (-r) mod t
  const bool kneg = k > t / 2;                                     // centred: k - t
  const uint32_t kmag = kneg ? t - k : k;
  // ---- v = h0 - hdec + [negr] - k_centred, then mod Q' ----
  int64_t cc = (int64_t)(negr ? 1 : 0) + (kneg ? (int64_t)kmag : -(int64_t)kmag);
  {
    uint32_t bw = 0;
    for (uint32_t l = 0; l <= nh; ++l) {                           // h -= hdec (hdec <= h0)
      const uint32_t sub = l == 0 ? (uint32_t)hdec : l == 1 ? (uint32_t)(hdec >> 32) : 0u, v = h[l], d = v - sub, d2 = d - bw;
      bw = (v < sub) | (d < bw);
      h[l] = d2;
    }
    for (uint32_t l = 0; l <= nh; ++l) { const int64_t s = (int64_t)h[l] + cc; h[l] = (uint32_t)s; cc = s >> 32; }
  }
  auto q2limb = [&](uint32_t l) { return (l == 0 ? e2 : 0u) + (l == ws ? 1u << bs : 0u); };
  if (cc < 0) {                                                    // negative: + Q'
    uint32_t c3 = 0;
    for (uint32_t l = 0; l <= nh; ++l) { const uint64_t s = (uint64_t)h[l] + q2limb(l) + c3; h[l] = (uint32_t)s; c3 = (uint32_t)(s >> 32); }
  } else {
    bool ge = true;                                                // v >= Q' ?
    for (uint32_t l = nh + 1; l-- > 0;) { const uint32_t ql = q2limb(l); if (h[l] != ql) { ge = h[l] > ql; break; } }
    if (ge) {
      uint32_t b3 = 0;
      for (uint32_t l = 0; l <= nh; ++l) { const uint32_t ql = q2limb(l), v = h[l], d = v - ql, d2 = d - b3; b3 = (v < ql) | (d < b3); h[l] = d2; }
    }
  }
  for (uint32_t l = 0; l < L; ++l) out[base + (size_t)l * N] = l <= nh ? h[l] : 0u;
}

cudaError_t launch_modswitch(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logQ, uint32_t e, uint32_t e2,
                             uint32_t npoly, cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  if (c->L > ELEM_MAX_LIMBS) return cudaErrorInvalidValue;
  const uint32_t t = (uint32_t)c->t;
  const uint64_t mu_t = ~0ull / t;                                 // floor((2^64 - 1) / t): at most 1 below floor(2^64 / t)
  LaunchTimer lt(c, KC_RESCALE, s);
  modswitch_bgv_kernel<<<(c->N / 128) * npoly, 128, 0, s>>>(d_out, d_in, c->N, c->L, c->logQ, e, new_logQ, e2, t, mu_t);
  return cudaGetLastError();
}

cudaError_t launch_add_plain(Context* c, uint32_t* d_out, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                             uint32_t group, cudaStream_t s) {
  if (!batch) return cudaSuccess;
  if (c->L > ELEM_MAX_LIMBS) return cudaErrorInvalidValue;
  LaunchTimer lt(c, KC_RESCALE, s);
  add_plain_kernel<<<(c->N / 256) * 2 * batch, 256, 0, s>>>(d_out, d_ct, d_pt, c->d_Qlimbs, c->N, c->L, c->logQ, group, c->t == 0 ? 1u : 0u);
  return cudaGetLastError();
}

cudaError_t launch_mult_scalar(Context* c, uint32_t* d_out, const uint32_t* d_in, int32_t k, uint32_t npoly, cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  if (c->L > ELEM_MAX_LIMBS) return cudaErrorInvalidValue;
  const uint32_t kabs = k < 0 ? (uint32_t)(-(int64_t)k) : (uint32_t)k;
  LaunchTimer lt(c, KC_RESCALE, s);
  mult_scalar_kernel<<<(c->N / 256) * npoly, 256, 0, s>>>(d_out, d_in, c->d_Qlimbs, c->N, c->L, c->logQ, kabs, k < 0 ? 1u : 0u, c->t == 0 ? 1u : 0u);
  return cudaGetLastError();
}

cudaError_t launch_monomial(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t k, uint32_t npoly, cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  LaunchTimer lt(c, KC_RESCALE, s);
  monomial_kernel<<<(c->N / 256) * npoly, 256, 0, s>>>(d_out, d_in, c->d_Qlimbs, c->N, c->L, c->logQ, k, c->t == 0 ? 1u : 0u);
  return cudaGetLastError();
}

cudaError_t launch_automorphism(Context* c, uint32_t* d_out3, const uint32_t* d_in2, uint32_t k, uint32_t batch, cudaStream_t s) {
  if (!batch) return cudaSuccess;
  const uint32_t twoN = 2 * c->N;
  uint32_t kinv = 1;                                                // k^-1 mod 2N (k odd): Newton iteration mod 2^32, then reduce
  for (int it = 0; it < 5; ++it) kinv *= 2u - k * kinv;
  kinv &= twoN - 1;
  LaunchTimer lt(c, KC_RESCALE, s);
  automorphism_kernel<<<(c->N / 256) * 3 * batch, 256, 0, s>>>(d_out3, d_in2, c->d_Qlimbs, c->N, c->L, c->logQ, kinv, c->t == 0 ? 1u : 0u);
  return cudaGetLastError();
}

cudaError_t launch_elem(Context* c, int op, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly,
                        uint32_t bits, cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  if (c->L > ELEM_MAX_LIMBS) return cudaErrorInvalidValue;
  const uint32_t grid = (c->N / 256) * npoly;
  LaunchTimer lt(c, KC_RESCALE, s);
  if (c->t == 0) {
    switch (op) {
      case EL_ADD: elem_ckks_kernel<EL_ADD><<<grid, 256, 0, s>>>(d_out, d_a, d_b, c->N, c->L, bits); break;
      case EL_SUB: elem_ckks_kernel<EL_SUB><<<grid, 256, 0, s>>>(d_out, d_a, d_b, c->N, c->L, bits); break;
      case EL_NEG: elem_ckks_kernel<EL_NEG><<<grid, 256, 0, s>>>(d_out, d_a, d_a, c->N, c->L, bits); break;
      case EL_MODDOWN: elem_ckks_kernel<EL_MODDOWN><<<grid, 256, 0, s>>>(d_out, d_a, d_a, c->N, c->L, bits); break;
      default: return cudaErrorInvalidValue;
    }
  } else {
    switch (op) {
      case EL_ADD: elem_bgv_kernel<EL_ADD><<<grid, 256, 0, s>>>(d_out, d_a, d_b, c->d_Qlimbs, c->N, c->L); break;
      case EL_SUB: elem_bgv_kernel<EL_SUB><<<grid, 256, 0, s>>>(d_out, d_a, d_b, c->d_Qlimbs, c->N, c->L); break;
      case EL_NEG: elem_bgv_kernel<EL_NEG><<<grid, 256, 0, s>>>(d_out, d_a, d_a, c->d_Qlimbs, c->N, c->L); break;
      default: return cudaErrorInvalidValue;
    }
  }
  return cudaGetLastError();
}

}  // namespace fhe
