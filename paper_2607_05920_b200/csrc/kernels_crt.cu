// kernels_crt.cu -- S5 CRT reconstruction + reduction mod Q, S6(e,f) divide-by-P + add, S7 rescale.
//
// Reconstruction uses the direct form of the CRT (Eq. 1) instead of the paper's Garner recurrence
// (Eq. 16-17): with y_i = x_i (M/q_i)^-1 mod q_i (the constant is folded into the inverse NTT),
//     X = sum_i y_i (M/q_i) - alpha M,   alpha = round(sum_i y_i / q_i),
// gives the centred representative |X| < M/2 directly.  M is chosen > 4 * (largest possible |X|), so
// frac(sum y_i/q_i) is within 1/4 of an integer and a 2^-22-accurate fixed-point sum decides alpha exactly
// (DESIGN.md 5).  The sum is a dot product of (K+1) words with (K+1) constant multi-digit vectors, evaluated on
// 26-bit digits so that products accumulate in uint64 without carries.
#include <algorithm>

#include "fhe_internal.cuh"
#include "pipe.cuh"

namespace fhe {

constexpr int TC = 128;   // coefficients (= threads) per block

// ---- multi-limb helpers on a shared-memory column: limb l of this thread's number is p[l * TC] ---------------------
struct Col {
  uint32_t* p;
  __device__ __forceinline__ uint32_t get(uint32_t l) const { return p[l * TC]; }
  __device__ __forceinline__ void set(uint32_t l, uint32_t v) const { p[l * TC] = v; }
};

// x += 2^bit, over limbs [0, nl) (carry out of limb nl-1 is dropped)
__device__ __forceinline__ void col_add_pow2(Col x, uint32_t bit, uint32_t nl) {
  uint32_t l = bit >> 5;
  uint32_t add = 1u << (bit & 31);
  while (l < nl && add) {
    uint32_t v = x.get(l), s = v + add;
    x.set(l, s);
    add = s < v ? 1u : 0u;
    ++l;
  }
}
// bits [sh + 32 l, sh + 32 l + 32) of x (x has nl limbs; beyond reads as 0)
__device__ __forceinline__ uint32_t col_bits(Col x, uint32_t sh, uint32_t l, uint32_t nl) {
  uint32_t w = (sh >> 5) + l, b = sh & 31;
  uint32_t lo = w < nl ? x.get(w) : 0u;
  if (b == 0) return lo;
  uint32_t hi = (w + 1) < nl ? x.get(w + 1) : 0u;
  return (lo >> b) | (hi << (32 - b));
}
__host__ __device__ __forceinline__ uint32_t top_mask(uint32_t bits) { return (bits & 31) ? ((1u << (bits & 31)) - 1u) : 0xFFFFFFFFu; }

// x >= m ?  (x: nl limbs in the column, m: nl limbs in global memory)
__device__ __forceinline__ bool col_ge(Col x, const uint32_t* __restrict__ m, uint32_t nl) {
  for (uint32_t l = nl; l-- > 0;) {
    uint32_t a = x.get(l), b = __ldg(m + l);
    if (a != b) return a > b;
  }
  return true;
}
// x -= m over nl limbs (wraps)
__device__ __forceinline__ void col_sub(Col x, const uint32_t* __restrict__ m, uint32_t nl) {
  uint32_t borrow = 0;
  _Pragma("unroll 4")
  for (uint32_t l = 0; l < nl; ++l) {
    uint32_t a = x.get(l), b = __ldg(m + l);
    uint32_t d = a - b, d2 = d - borrow;
    borrow = (a < b) | (d < borrow);
    x.set(l, d2);
  }
}
// x += m over nl limbs (wraps)
__device__ __forceinline__ void col_add(Col x, const uint32_t* __restrict__ m, uint32_t nl) {
  uint32_t carry = 0;
  _Pragma("unroll 4")
  for (uint32_t l = 0; l < nl; ++l) {
    uint64_t s = (uint64_t)x.get(l) + __ldg(m + l) + carry;
    x.set(l, (uint32_t)s);
    carry = (uint32_t)(s >> 32);
  }
}
// x -= k * m over nx limbs (wraps mod 2^(32 nx)); m has nm limbs, k is 64-bit
__device__ __forceinline__ void col_submul64(Col x, const uint32_t* __restrict__ m, uint32_t nm, uint64_t k, uint32_t nx) {
  const uint32_t k0 = (uint32_t)k, k1 = (uint32_t)(k >> 32);
  // product limbs p_l = sum k0*m[l] + k1*m[l-1], streamed with a 96-bit carry
  uint64_t acc_lo = 0; uint32_t acc_hi = 0;  // acc = acc_hi * 2^64 + acc_lo
  uint32_t borrow = 0;
  _Pragma("unroll 4")
  for (uint32_t l = 0; l < nx; ++l) {
    uint64_t t0 = (l < nm) ? (uint64_t)k0 * __ldg(m + l) : 0ull;
    uint64_t t1 = (l >= 1 && l - 1 < nm) ? (uint64_t)k1 * __ldg(m + l - 1) : 0ull;
    uint64_t s = acc_lo + t0; acc_hi += (s < acc_lo); acc_lo = s;
    s = acc_lo + t1; acc_hi += (s < acc_lo); acc_lo = s;
    uint32_t pl = (uint32_t)acc_lo;
    acc_lo = (acc_lo >> 32) | ((uint64_t)acc_hi << 32); acc_hi = 0;
    uint32_t a = x.get(l);
    uint32_t d = a - pl, d2 = d - borrow;
    borrow = (a < pl) | (d < borrow);
    x.set(l, d2);
  }
}
// V (nx limbs, V < 2^(bits+40)) -> V mod m in place, m with `bits` significant bits, mu1 = floor(2^(bits+62)/m)
__device__ __forceinline__ void col_barrett1(Col x, uint32_t nx, const uint32_t* __restrict__ m, uint32_t nm,
                                             uint32_t bits, uint64_t mu1) {
  const uint32_t sh = bits - 24;
  uint64_t vt = (uint64_t)col_bits(x, sh, 0, nx) | ((uint64_t)col_bits(x, sh, 1, nx) << 32);
  uint64_t qh = __umul64hi(vt, mu1) >> 22;
  col_submul64(x, m, nm, qh, nx);
  // remainder in [0, 2m): at most two corrections (one expected)
  for (int it = 0; it < 2; ++it) {
    bool hi_nz = false;
    for (uint32_t l = nm; l < nx; ++l) hi_nz |= (x.get(l) != 0);
    if (hi_nz || col_ge(x, m, nm)) col_sub(x, m, nx);
  }
}

// V (nx limbs, V < 2^(k + 40)) -> V mod M in place, M = 2^k + e with e < 2^22 (the BGV moduli: the least odd integer above the
// power of two that is 1 mod t): V = A 2^k + B is congruent to B - A e, and A e < 2^63 is a two-word number, so the reduction is
// one masked copy, one subtraction and at most one addition of M instead of a Barrett step with the limbs of M.
__device__ __forceinline__ void col_fold_mod(Col x, uint32_t nx, uint32_t k, uint32_t e) {
  const uint32_t wq = k >> 5, bq = k & 31, nm = wq + 1;
  const uint32_t a0 = x.get(wq), a1 = wq + 1 < nx ? x.get(wq + 1) : 0u, a2 = wq + 2 < nx ? x.get(wq + 2) : 0u;
  const uint64_t A = bq ? ((uint64_t)(a0 >> bq) | ((uint64_t)a1 << (32 - bq)) | ((uint64_t)a2 << (64 - bq))) : ((uint64_t)a0 | ((uint64_t)a1 << 32));
  x.set(wq, bq ? a0 & ((1u << bq) - 1u) : 0u);
  for (uint32_t l = nm; l < nx; ++l) x.set(l, 0u);
  const uint64_t s = A * e;
  uint32_t borrow = 0;
  _Pragma("unroll 4")
  for (uint32_t l = 0; l < nm; ++l) {
    const uint32_t sub = l == 0 ? (uint32_t)s : l == 1 ? (uint32_t)(s >> 32) : 0u, v = x.get(l), d = v - sub, d2 = d - borrow;
    borrow = (v < sub) | (d < borrow);
    x.set(l, d2);
    if (l >= 1 && !borrow) break;                                  // nothing left to propagate
  }
  if (borrow) {                                                    // negative: + M once (A e < 2^63 < M)
    uint32_t carry = 0;
    _Pragma("unroll 4")
    for (uint32_t l = 0; l < nm; ++l) {
      const uint64_t sum = (uint64_t)x.get(l) + ((l == 0 ? e : 0u) + (l == wq ? 1u << bq : 0u)) + carry;
      x.set(l, (uint32_t)sum);
      carry = (uint32_t)(sum >> 32);
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// CRT epilogue of the conversion pipeline (pipe.cuh).  The loaders stage the residues y[i][n] as the A operand (word i =
// column i), the tensor cores contract them with the constant image B: column 8 + e receives
// S_e = sum_{i,b} y_ib * byte_{e-b}(W_i), columns 0..5 the byte sums of sum_i y_i floor(2^48 / q_i) (-> alpha).  Here:
//   column sums  P_l = S_4l + 2^8 S_4l+1 + 2^16 S_4l+2 + 2^24 S_4l+3 + alpha negM_l  (< 2^52): four mad.wide per limb,
//                independent across the eight limbs of a call
//   CKKS relin   everything that is ADDED to V before the shifts is added to the column sums first -- the polynomial d
//                (d0 or d1) at bit position s1, the rounding 2^(logP-1) of the divide by P, the rounding 2^(s1+p-1) of the
//                rescale (s1 = logP, or 0 for the top form, which hands V >> logP over directly) -- so that ONE carry chain
//                (two dependent instructions per limb) yields the limbs of  total = V + 2^(logP-1) + (d << s1) + 2^(s1+p-1)
//                and the output limb m is bits [s1 + p + 32 m, +32) of it, one funnel shift.  Carries out of bit
//                s1 + logQ only reach bits the final reduction mod 2^(logQ-p) drops, so (d + k) needs no reduction mod
//                2^logQ between the two roundings: the result is the one of the three separate steps (A3/A4).
//   CKKS mask    the limbs of V below logQ, top limb masked (tensor / polymul)
//   BGV          the limbs go to this thread's column xs[.][etid] in shared memory and the multi-limb Barrett
//                reductions run on the column (post()).
// The polynomial added by the relin modes is prefetched into a shared-memory column with cp.async while the tile's
// MMAs run.  MODE / TOP / RESC are template parameters: the hot loops carry no mode branches.
// ------------------------------------------------------------------------------------------------------------------
struct CrtParams {
  uint32_t* out; size_t out_outer, out_inner;
  const uint32_t* add; size_t add_outer, add_inner;   // relin modes; else nullptr
  const uint32_t* negM;                               // [Lraw]
  uint32_t Lraw, Lx, nl, ntab;                        // nl = limbs of V the chunks cover; ntab = entries of the negM table
  uint32_t amb_bits; uint32_t* flags;                 // top-form relin target (fhe_internal.cuh): flag bitmap of the exact path
  uint32_t xs_off, adds_off, scratch_off;             // word offsets inside the scratch: negM table at 0, then the columns
  // CKKS relin: d enters at limb wd, bit bd (s1 = 32 wd + bd); the output starts at limb ws, bit bs of the total
  // (s1 + p = 32 ws + bs); roundings rbit1 at limb rb1 (divide by P; full form only), rbit2 at limb rb2 (rescale);
  // the result has Lr limbs, the top one masked with tm; lend = last limb of the total the stream must see
  uint32_t wd, bd, ws, bs, rb1, rbit1, rb2, rbit2, Lr, tm, tmq, lend;
  // 2^8, 2^16, 2^24 as run-time values: with literal powers of two ptxas splits every mad.wide of the column sums into
  // IMAD.SHL + IMAD.HI + carry adds (seven multiplier-pipe instructions per limb instead of one IMAD.WIDE per column)
  uint32_t m8, m16, m24;
  PostParams pp;
};

template <int MODE, bool TOP, bool RESC>
struct CrtEpi {
  static constexpr int LOAD_WORDS = 64, MAX_REGS = 96;     // 17 warps are allocated as 20: 20 x 32 x 96 <= 64 K
  static constexpr uint32_t GROUPS = 2, LOAD_WARPS = 8;
  static constexpr bool LOAD_ALT = false;
  static constexpr bool LOAD_TMA = true;                   // residues staged through shared memory by one tensor copy per tile
  static constexpr bool TILE_ALT = true;                   // two whole epilogues on alternate tiles: the epilogue bounds S5
  static constexpr bool CHUNK_ALT = false;
  static constexpr bool RELIN = MODE == POST_CKKS_RELIN || MODE == POST_BGV_RELIN;
  static_assert(!TOP || MODE == POST_CKKS_RELIN, "the top form exists for the CKKS relin target only");
  static_assert(!RESC || MODE == POST_CKKS_RELIN, "the fused rescale is CKKS-only");
  using Params = CrtParams;
  const Params& p;
  const uint32_t N, etid, inner;
  const uint32_t* negm;  // [nl + 2] in shared memory, zero beyond Lraw
  uint32_t* xs;          // [Lx][TC]   (BGV)
  uint32_t* adds;        // [L][TC]    (relin modes)
  uint32_t* scratch;     // [scratch_limbs][TC]  (BGV relin)
  uint32_t* out = nullptr;
  uint32_t* optr = nullptr;
  uint32_t alpha = 0, yprev = 0;
  uint64_t carry = 0;
  uint32_t flag_word = 0;   // word of the flag bitmap this warp's 32 coefficients own: bit = lane
  bool d_ready = false;

  __device__ CrtEpi(const Params& p_, const pipe::PipeArgs&a, uint8_t* sm, uint32_t etid_, uint32_t, uint32_t bar)
      : p(p_), N(a.N), etid(etid_), inner(a.inner), negm(reinterpret_cast<const uint32_t*>(sm)),
        xs(reinterpret_cast<uint32_t*>(sm) + p_.xs_off), adds(reinterpret_cast<uint32_t*>(sm) + p_.adds_off),
        scratch(reinterpret_cast<uint32_t*>(sm) + p_.scratch_off) {
    uint32_t* w = reinterpret_cast<uint32_t*>(sm);
    for (uint32_t k = etid; k < p.ntab; k += TC) w[k] = k < p.Lraw ? __ldg(p.negM + k) : 0u;
    pipe::epi_sync(bar, TC);
  }

  __device__ __forceinline__ void begin_tile(uint32_t o, uint32_t i, uint32_t n0) {
    out = p.out + (size_t)o * p.out_outer + (size_t)i * p.out_inner + n0 + etid;
    optr = out;
    carry = 0; yprev = 0;
    if constexpr (TOP) flag_word = (o * inner + i) * (N >> 5) + ((n0 + etid) >> 5);
    if constexpr (RELIN) {
      const uint32_t* src = p.add + (size_t)o * p.add_outer + (size_t)i * p.add_inner + n0 + etid;
      const uint32_t dst = umma::smem_u32(adds + etid);
      for (uint32_t k = 0; k < p.pp.L; ++k)
        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst + k * TC * 4), "l"(src + (size_t)k * N) : "memory");
      asm volatile("cp.async.commit_group;" ::: "memory");
      d_ready = false;
    }
  }

  // Top-form relin target, first 32 columns of a tile: P[2..8) are the six limbs of S_t = sum_i y_i Wt_i + alpha Nt, the
  // low part of V cut down to its top TOP_BITS bits.  The carry into the high part is round(S_t / 2^96); the cut-off
  // bits can add less than 2^-58 to S_t / 2^96, so the rounding is certain unless the amb_bits fractional bits below the
  // rounding position are all ones -- then the coefficient's bit is set in the bitmap crt_exact_kernel works off.
  __device__ __forceinline__ void top_carry(const uint64_t* P) {
    uint32_t sl[TOP_LIMBS];
    uint64_t cr = 0;
#pragma unroll
    for (int g = 0; g < (int)TOP_LIMBS; ++g) {
      const uint64_t v = cr + P[g + 2];
      sl[g] = (uint32_t)v;
      cr = v >> 32;
    }
    const uint64_t r2 = (uint64_t)sl[2] + 0x80000000u;             // + 2^95
    const uint64_t r3 = (uint64_t)sl[3] + (r2 >> 32);
    const uint64_t r4 = (uint64_t)sl[4] + (r3 >> 32);
    carry = (r3 & 0xFFFFFFFFu) | (r4 << 32);                      // bits 96.. of S_t + 2^95 (S_t < 2^134)
    const uint64_t frac = ((uint64_t)(uint32_t)r2 << 32) | sl[1];  // fractional bits 32..95
    // One bit per coefficient, [polynomial][N / 32] words: the 32 lanes of a warp own consecutive coefficients, i.e. one
    // word, which the warp writes whole (zero or not) -- no atomics, nothing to clear, no coefficient can be dropped.
    const bool amb = (frac >> (64 - p.amb_bits)) == (~0ull >> (64 - p.amb_bits));
    const uint32_t m = __ballot_sync(0xFFFFFFFFu, amb);
    if ((etid & 31) == 0) p.flags[flag_word] = m;
  }

  // bits of (d << s1) that fall into limb lg of the total (any lg): the generic, bounds-checked form
  __device__ __forceinline__ uint32_t d_limb(uint32_t lg) const {
    const uint32_t j = lg - p.wd;                                  // wraps for lg < wd: both tests below then fail
    const uint32_t hi = j < p.pp.L ? adds[j * TC + etid] : 0u;
    if (p.bd == 0) return hi;
    const uint32_t lo = j - 1 < p.pp.L ? adds[(j - 1) * TC + etid] : 0u;
    return __funnelshift_l(lo, hi, p.bd);
  }
  // One limb of the CKKS relin stream with every boundary checked: P = column sum of limb lg of the total.
  __device__ __forceinline__ void relin_step(uint32_t lg, uint64_t P) {
    P += d_limb(lg);
    if (!TOP && lg == p.rb1) P += p.rbit1;
    if (RESC && lg == p.rb2) P += p.rbit2;
    const uint64_t v = carry + P;
    carry = v >> 32;
    const uint32_t y = (uint32_t)v;
    if (lg > p.ws) {
      const uint32_t m = lg - 1 - p.ws;
      if (m < p.pp.L) {
        uint32_t o = __funnelshift_r(yprev, y, p.bs);
        if (m == p.Lr - 1) o &= p.tm;
        if (m >= p.Lr) o = 0;
        *optr = o; optr += N;
      }
    }
    yprev = y;
  }

  __device__ __forceinline__ void consume(uint32_t col0, const uint32_t* t) {
    int g0 = 0;
    if (col0 == 0) {
      uint64_t asum = madw(t[3], p.m24, madw(t[2], p.m16, madw(t[1], p.m8, (uint64_t)t[0])));
      asum += ((uint64_t)t[4] << 32) + ((uint64_t)t[5] << 40);
      alpha = (uint32_t)((asum + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
      g0 = CRT_ALPHA_COLS / 4;
    }
    const uint32_t tb = col0 / 4 - CRT_ALPHA_COLS / 4;             // table / limb index of group element 0 (wraps for col0 = 0; elements 0, 1 unused)
    uint64_t P[8];                                                 // the limb's column sum + alpha * negM: independent of the carry
#pragma unroll
    for (int g = 0; g < 8; ++g) {
      if (g < g0) { P[g] = 0; continue; }
      P[g] = madw(alpha, negm[tb + g], madw(t[4 * g + 3], p.m24, madw(t[4 * g + 2], p.m16, madw(t[4 * g + 1], p.m8, (uint64_t)t[4 * g]))));
    }
    uint32_t l0 = tb;
    if constexpr (TOP) {
      if (col0 == 0) { top_carry(P); return; }
      l0 -= TOP_LIMBS;                                             // from here on l0 counts limbs of the high part
    }
    const uint32_t L = p.pp.L;
    if constexpr (MODE == POST_CKKS_MASK) {
      if (g0 == 0 && l0 + 8 < L) {
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          const uint64_t v = carry + P[g];
          carry = v >> 32;
          *optr = (uint32_t)v; optr += N;
        }
      } else {
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          if (g < g0) continue;
          const uint64_t v = carry + P[g];
          carry = v >> 32;
          const uint32_t lg = l0 + g;
          if (lg < L) { *optr = lg == L - 1 ? ((uint32_t)v & p.tmq) : (uint32_t)v; optr += N; }
        }
      }
    } else if constexpr (MODE == POST_CKKS_RELIN) {
      if (!d_ready && l0 + 8 > p.wd) {                             // the add column is read from here on
        asm volatile("cp.async.wait_group 0;" ::: "memory");
        d_ready = true;
      }
      if (g0 == 0 && l0 > p.ws && l0 + 7 - p.wd < L && l0 + 7 - p.ws < p.Lr) {
        // interior group: d_{j-1}, d_j exist for all eight limbs, no rounding limb (rb1 <= wd, rb2 <= ws < l0), every
        // output limb below the masked top limb
        const uint32_t* ap = adds + (l0 - p.wd) * TC + etid;
        if (p.bd == 0) {
#pragma unroll
          for (int g = 0; g < 8; ++g) P[g] += ap[g * TC];
        } else {
          uint32_t dlo = ap[-TC];
#pragma unroll
          for (int g = 0; g < 8; ++g) {
            const uint32_t dhi = ap[g * TC];
            P[g] += __funnelshift_l(dlo, dhi, p.bd);
            dlo = dhi;
          }
        }
        uint32_t y[9];
        y[0] = yprev;
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          const uint64_t v = carry + P[g];
          carry = v >> 32;
          y[g + 1] = (uint32_t)v;
        }
        yprev = y[8];
#pragma unroll
        for (int g = 0; g < 8; ++g) { *optr = __funnelshift_r(y[g], y[g + 1], p.bs); optr += N; }
      } else if (l0 + 8 <= p.wd && l0 + 8 <= p.ws && (TOP || l0 + 8 <= p.rb1) && (!RESC || l0 + 8 <= p.rb2)) {
        // far below everything: only the carry matters
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          if (g < g0) continue;
          const uint64_t v = carry + P[g];
          carry = v >> 32;
          yprev = (uint32_t)v;
        }
      } else {
#pragma unroll
        for (int g = 0; g < 8; ++g) {
          if (g < g0) continue;
          relin_step(l0 + g, P[g]);
        }
      }
    } else {                                                       // BGV: the column in shared memory
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        if (g < g0) continue;
        const uint64_t v = carry + P[g];
        carry = v >> 32;
        const uint32_t lg = l0 + g;
        if (lg < p.Lx) xs[lg * TC + etid] = (uint32_t)v;
      }
    }
  }

  __device__ void end_tile() {
    if constexpr (MODE == POST_CKKS_MASK) return;                  // the chunks cover all L limbs
    if constexpr (RELIN) {
      if (!d_ready) { asm volatile("cp.async.wait_group 0;" ::: "memory"); d_ready = true; }
    }
    if constexpr (MODE == POST_CKKS_RELIN) {
      for (uint32_t lg = p.nl; lg <= p.lend; ++lg) relin_step(lg, 0);   // limbs past the last chunk: carry and d only
      return;
    }
    if constexpr (MODE == POST_BGV_MODQ || MODE == POST_BGV_RELIN) {
      for (uint32_t lg = p.nl; lg < p.Lx; ++lg) { xs[lg * TC + etid] = (uint32_t)carry; carry = 0; }
      post();
    }
  }
  __device__ void post();
};

template <int MODE, bool TOP, bool RESC>
__device__ void CrtEpi<MODE, TOP, RESC>::post() {
  const PostParams& pp = p.pp;
  const uint32_t Lx = p.Lx;
  Col x{xs + etid};
  Col ad{adds + etid};
  const uint32_t L = pp.L;
  if constexpr (MODE == POST_BGV_MODQ) {
    if (pp.fold_modq) col_fold_mod(x, Lx, pp.logQ, pp.eQ);
    else col_barrett1(x, Lx, pp.d_Q, L, pp.bitsQ, pp.mu1_Q);
    _Pragma("unroll 4")
    for (uint32_t k = 0; k < L; ++k) out[(size_t)k * N] = x.get(k);
    return;
  }
  // POST_BGV_RELIN: V -> xc = V mod PQ -> (q3, rem) = divmod(xc, P) -> centred r, kk -> (hi - kk + d) mod Q
  if constexpr (MODE == POST_BGV_RELIN) {
    const uint32_t LP = pp.L_P, LPQ = pp.L_PQ, g = pp.g_limbs;   // g = LPQ - LP
    if (!pp.fold_full) col_barrett1(x, Lx, pp.d_PQ, LPQ, pp.bitsPQ, pp.mu1_PQ);     // x[0..LPQ) = xc = V mod PQ
    const uint32_t NXX = pp.fold_full ? Lx : LPQ;              // fold_full: the division runs on V itself (see PostParams)
    Col sc{scratch + etid};
    Col q3{sc.p};                                    // the quotient's limbs (nq of them)
    uint32_t nq, qinc = 0;
    if (pp.fold_div) {
      // P = 2^kP + eP: xc = A 2^kP + B = A P + z, z = B - A eP (signed, |z| < 2^(bitsQ + 1 + bits(eP))).  When z < 0, y = -z =
      // j 2^kP + yl = j P + w, w = yl - j eP with j < 2^60 and j eP < 2^92 < 2^kP (ctx.cu: fold_div), so
      //   w > 0:  xc = (A - j - 1) P + (P - w);     w <= 0:  xc = (A - j) P + (-w)
      // -- quotient and remainder in O(L) word operations instead of the two multi-limb products of a Barrett division.
      const uint32_t kP = pp.logP, wq = kP >> 5, bq = kP & 31, eP = pp.eP;      // LP == wq + 1
      const uint32_t nA = NXX - wq;                                              // limbs of A = xc >> kP
      // one pass: limb l of A (a funnel shift of limbs wq + l, wq + l + 1, which this pass has not overwritten yet) goes to the
      // scratch column and, times eP, off limb l of B = xc mod 2^kP
      const uint32_t nz = (LP > nA + 1 ? LP : nA + 1) + 1;                      // limbs of z = B - A eP (signed)
      const uint32_t bmask = bq ? (1u << bq) - 1u : 0u;
      uint32_t borrow = 0, mc = 0;
      _Pragma("unroll 4")
      for (uint32_t l = 0; l < nz; ++l) {
        uint32_t al = 0;
        if (l < nA) {
          const uint32_t lo = x.get(wq + l), hi = wq + l + 1 < NXX ? x.get(wq + l + 1) : 0u;
          al = bq ? (lo >> bq) | (hi << (32 - bq)) : lo;
        }
        if (l <= nA) sc.set(l, al);
        const uint64_t pr = (uint64_t)al * eP + mc;
        const uint32_t sub = (uint32_t)pr, v = l < wq ? x.get(l) : l == wq ? x.get(l) & bmask : 0u, d = v - sub, d2 = d - borrow;
        mc = (uint32_t)(pr >> 32);
        borrow = (v < sub) | (d < borrow);
        x.set(l, d2);
      }
      uint32_t hd[4] = {0u, 0u, 0u, 0u};                                         // what comes off A: j or j + 1, j < 2^95
      if (borrow) {
        uint32_t c1 = 1;                                                         // y = -z
        _Pragma("unroll 4")
        for (uint32_t l = 0; l < nz; ++l) { const uint64_t sm = (uint64_t)(~x.get(l)) + c1; x.set(l, (uint32_t)sm); c1 = (uint32_t)(sm >> 32); }
        uint32_t jw[3];                                                          // j = y >> kP
        for (uint32_t i = 0; i < 3; ++i) {
          const uint32_t lo = wq + i < nz ? x.get(wq + i) : 0u, hi = wq + i + 1 < nz ? x.get(wq + i + 1) : 0u;
          jw[i] = bq ? (lo >> bq) | (hi << (32 - bq)) : lo;
        }
        x.set(wq, bq ? x.get(wq) & ((1u << bq) - 1u) : 0u);                     // yl
        for (uint32_t l = LP; l < nz; ++l) x.set(l, 0u);
        const uint64_t p0 = (uint64_t)jw[0] * eP, p1 = (uint64_t)jw[1] * eP + (p0 >> 32), p2 = (uint64_t)jw[2] * eP + (p1 >> 32);
        const uint32_t je[4] = {(uint32_t)p0, (uint32_t)p1, (uint32_t)p2, (uint32_t)(p2 >> 32)};
        uint32_t bw = 0, any = 0;
        _Pragma("unroll 4")
        for (uint32_t l = 0; l <= LP; ++l) {                                     // w = yl - j eP
          const uint32_t sub = l == 0 ? je[0] : l == 1 ? je[1] : l == 2 ? je[2] : l == 3 ? je[3] : 0u, v = x.get(l), d = v - sub, d2 = d - bw;
          bw = (v < sub) | (d < bw);
          x.set(l, d2); any |= d2;
        }
        uint32_t inc;
        if (!bw && any) {                                                        // w > 0: one more multiple, remainder P - w
          inc = 1;
          uint32_t b2 = 0;
          _Pragma("unroll 4")
          for (uint32_t l = 0; l <= LP; ++l) {
            const uint32_t pl = (l == 0 ? eP : 0u) + (l == wq ? 1u << bq : 0u), v = x.get(l), d = pl - v, d2 = d - b2;
            b2 = (pl < v) | (d < b2);
            x.set(l, d2);
          }
        } else {                                                                 // w <= 0: remainder -w
          inc = 0;
          uint32_t c2 = 1;
          _Pragma("unroll 4")
          for (uint32_t l = 0; l <= LP; ++l) { const uint64_t sm = (uint64_t)(~x.get(l)) + c2; x.set(l, (uint32_t)sm); c2 = (uint32_t)(sm >> 32); }
        }
        uint32_t cy = inc;
        for (uint32_t i = 0; i < 3; ++i) { const uint64_t sm = (uint64_t)jw[i] + cy; hd[i] = (uint32_t)sm; cy = (uint32_t)(sm >> 32); }
        hd[3] = cy;
      }
      nq = nA + 1;
      uint32_t bw = 0;                                                           // quotient = A - hdec (>= 0)
      _Pragma("unroll 4")
      for (uint32_t l = 0; l < nq; ++l) {
        const uint32_t sub = l == 0 ? hd[0] : l == 1 ? hd[1] : l == 2 ? hd[2] : l == 3 ? hd[3] : 0u, v = sc.get(l), d = v - sub, d2 = d - bw;
        bw = (v < sub) | (d < bw);
        sc.set(l, d2);
      }
      if (pp.fold_full) {                                                        // floor(V / P) -> mod Q (it is below 2^(logQ + 42))
        col_fold_mod(sc, nq, pp.logQ, pp.eQ);
        nq = L;
      }
    } else {
    // Barrett quotient estimate (HAC 14.42 generalised): q1 = xc >> 32(LP-1)  (g+1 limbs),
    // q3 = (q1 * mu) >> 32(g+1), mu = floor(2^(32 LPQ) / P)  (muP_limbs limbs); true quotient - q3 in {0,1,2}.
    const uint32_t n1 = g + 1, nmu = pp.muP_limbs;
    {
      uint64_t acc_lo = 0; uint32_t acc_hi = 0;
      for (uint32_t r = 0; r < n1 + nmu; ++r) {
        uint32_t i_lo = (r >= nmu) ? (r - nmu + 1) : 0u;
        uint32_t i_hi = r < n1 ? r : (n1 - 1);
        for (uint32_t i = i_lo; i <= i_hi && i < n1; ++i) {
          uint64_t pr = (uint64_t)x.get(LP - 1 + i) * __ldg(pp.d_muP + (r - i));
          uint64_t s = acc_lo + pr; acc_hi += (s < acc_lo); acc_lo = s;
        }
        sc.set(r, (uint32_t)acc_lo);
        acc_lo = (acc_lo >> 32) | ((uint64_t)acc_hi << 32); acc_hi = 0;
      }
    }
    // q3 = sc[g+1 .. g+1+n1]; rem = xc - q3 * P over LP+1 limbs
    q3 = Col{sc.p + (size_t)(g + 1) * TC};
    nq = n1;                                         // limbs of q3 kept (q3 <= Q < 2^(32 (g+1)))
    {
      uint64_t acc_lo = 0; uint32_t acc_hi = 0; uint32_t borrow = 0;
      for (uint32_t r = 0; r <= LP; ++r) {
        for (uint32_t i = 0; i <= r && i < nq; ++i) {
          uint32_t pj = r - i;
          if (pj < LP) {
            uint64_t pr = (uint64_t)q3.get(i) * __ldg(pp.d_P + pj);
            uint64_t s = acc_lo + pr; acc_hi += (s < acc_lo); acc_lo = s;
          }
        }
        uint32_t pl = (uint32_t)acc_lo;
        acc_lo = (acc_lo >> 32) | ((uint64_t)acc_hi << 32); acc_hi = 0;
        uint32_t av = x.get(r);
        uint32_t d = av - pl, d2 = d - borrow;
        borrow = (av < pl) | (d < borrow);
        x.set(r, d2);
      }
    }
    // corrections: rem in [0, 3P)
    for (int it = 0; it < 2; ++it) {
      if (x.get(LP) != 0 || col_ge(x, pp.d_P, LP)) { col_sub(x, pp.d_P, LP + 1); ++qinc; }
    }
    }
    // centre: rem > (P-1)/2  <=>  2 rem > P - 1  <=> 2 rem >= P + 1 <=> 2 rem > P (P odd)
    bool neg;
    {
      // compare 2*rem with P from the top limb down (2*rem has LP+1 limbs)
      int cmp = 0;
      for (uint32_t k = LP + 1; k-- > 0 && cmp == 0;) {
        uint32_t hi = k < LP ? x.get(k) : 0u, lo = k >= 1 ? x.get(k - 1) : 0u;
        uint32_t two = (hi << 1) | (lo >> 31);
        uint32_t pv = k < LP ? __ldg(pp.d_P + k) : 0u;
        if (two != pv) cmp = two > pv ? 1 : -1;
      }
      neg = cmp > 0;
    }
    if (neg) ++qinc;                                 // hi = q + 1, r = rem - P
    // r mod t
    uint64_t rt = 0;
    if (pp.mu_t) {                                   // word-sized Barrett steps from the top limb down
      uint32_t acc = 0;
      for (uint32_t k = LP; k-- > 0;) acc = horner_mod(acc, x.get(k), pp.t, pp.mu_t);
      rt = acc;
    } else {
      _Pragma("unroll 4")
      for (uint32_t k = 0; k < LP; ++k) rt = (rt + (uint64_t)x.get(k) * __ldg(pp.d_pow32_t + k)) % pp.t;
    }
    if (neg) { uint64_t Pt = __ldg(pp.d_pow32_t + LP); rt = (rt + pp.t - Pt) % pp.t; }   // d_pow32_t[LP] holds P mod t
    uint64_t kk = ((pp.t - rt) % pp.t) * pp.Pinv_t % pp.t;     // (-r P^-1) mod t in [0, t)
    const bool kneg = kk > pp.t / 2;                            // centred: kk - t
    const uint32_t kmag = kneg ? (uint32_t)(pp.t - kk) : (uint32_t)kk;
    // res = q3 + qinc - kk_centred + d as an (L+1)-limb value in x[0 .. L] (between -t/2 and 2 Q + t), then mod Q: one addition of
    // Q or at most two subtractions -- the same residue as reducing before and after the addition of d
    {
      int64_t cc = (int64_t)qinc + (kneg ? (int64_t)kmag : -(int64_t)kmag);
      _Pragma("unroll 4")
      for (uint32_t k = 0; k <= L; ++k) {
        const int64_t v = (int64_t)(k < nq ? q3.get(k) : 0u) + (int64_t)(k < L ? ad.get(k) : 0u) + cc;
        x.set(k, (uint32_t)v);
        cc = v >> 32;
      }
      if (cc < 0) {
        col_add(x, pp.d_Q, L + 1);
      } else {
        for (int it = 0; it < 2; ++it)
          if (x.get(L) != 0 || col_ge(x, pp.d_Q, L)) col_sub(x, pp.d_Q, L + 1);
      }
      _Pragma("unroll 4")
      for (uint32_t k = 0; k < L; ++k) out[(size_t)k * N] = x.get(k);
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// The exact path of the top-form relin target: one thread per flagged coefficient recomputes the whole output
// coefficient from the full constants -- V = sum_i y_i W_i + alpha negM mod 2^(logP+logQ) limb by limb, divide by P with
// rounding, add d, optional rescale (the formulas of DESIGN.md 3, A3/A4) -- and overwrites what the pipeline stored.
// The flagged coefficients are the set bits of a bitmap [polynomial][N / 32] that the pipeline writes in full on every
// launch (kernels_crt.cu, top_carry), so no coefficient can be dropped and nothing needs clearing.  Expected work: 2^-58 of
// the coefficients; the launch costs a few microseconds when no bit is set.
// ------------------------------------------------------------------------------------------------------------------
constexpr uint32_t EXACT_MAX_LIMBS = 168;
struct ExactArgs {
  uint32_t* flags;
  const uint32_t* res; size_t res_outer, res_inner;
  const uint32_t* add; size_t add_outer, add_inner;
  uint32_t* out; size_t out_outer, out_inner;
  const uint32_t* W; const uint32_t* negM; const uint32_t* q;
  uint32_t N, K, Lfull, L, logP, logQ, rescale_bits, inner, nwords;
};

// x[0..n) += 2^bit
__device__ inline void big_add_pow2(uint32_t* x, uint32_t n, uint32_t bit) {
  uint32_t l = bit >> 5, add = 1u << (bit & 31);
  while (l < n && add) { const uint32_t v = x[l]; x[l] = v + add; add = (v + add) < v ? 1u : 0u; ++l; }
}
// x[0..n) = (x >> sh) over n + extra limbs of input, then reduced mod 2^bits
__device__ inline void big_shr_mask(uint32_t* x, uint32_t nin, uint32_t sh, uint32_t bits, uint32_t nout) {
  const uint32_t w = sh >> 5, b = sh & 31;
  for (uint32_t l = 0; l < nout; ++l) {
    const uint32_t lo = l + w < nin ? x[l + w] : 0u, hi = l + w + 1 < nin ? x[l + w + 1] : 0u;
    uint32_t v = b ? (lo >> b) | (hi << (32 - b)) : lo;
    if (32 * l >= bits) v = 0; else if (bits - 32 * l < 32) v &= (1u << (bits - 32 * l)) - 1u;
    x[l] = v;
  }
}

__global__ void __launch_bounds__(64)
crt_exact_kernel(ExactArgs a) {
  pdl_sync();
  uint32_t V[EXACT_MAX_LIMBS + 2];
  const uint32_t wpp = a.N >> 5;                                   // bitmap words per polynomial
  for (uint32_t w = blockIdx.x * blockDim.x + threadIdx.x; w < a.nwords; w += gridDim.x * blockDim.x) {
    uint32_t bits = a.flags[w];
    const uint32_t poly = w / wpp, o = poly / a.inner, i = poly % a.inner;
    while (bits) {
      const uint32_t b = __ffs(bits) - 1;
      bits &= bits - 1;
      const uint32_t n = (w % wpp) * 32 + b;
      const uint32_t* y = a.res + (size_t)o * a.res_outer + (size_t)i * a.res_inner + n;
      const uint32_t nl = a.Lfull + 2;
      for (uint32_t l = 0; l < nl; ++l) V[l] = 0;
      uint64_t asum = 0;
      for (uint32_t j = 0; j < a.K; ++j) {
        const uint32_t yj = y[(size_t)j * a.N];
        asum += (uint64_t)yj * ((1ull << ALPHA_SHIFT) / a.q[j]);
        uint64_t cr = 0;
        const uint32_t* wj = a.W + (size_t)j * a.Lfull;
        for (uint32_t l = 0; l < a.Lfull; ++l) {
          const uint64_t t = (uint64_t)yj * wj[l] + V[l] + cr;
          V[l] = (uint32_t)t; cr = t >> 32;
        }
        for (uint32_t l = a.Lfull; l < nl && cr; ++l) { const uint64_t t = (uint64_t)V[l] + cr; V[l] = (uint32_t)t; cr = t >> 32; }
      }
      const uint32_t alpha = (uint32_t)((asum + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
      {
        uint64_t cr = 0;
        for (uint32_t l = 0; l < a.Lfull; ++l) {
          const uint64_t t = (uint64_t)alpha * a.negM[l] + V[l] + cr;
          V[l] = (uint32_t)t; cr = t >> 32;
        }
      }
      // x = V mod 2^(logP+logQ); k = ((x + 2^(logP-1)) >> logP) mod 2^logQ
      big_shr_mask(V, a.Lfull, 0, a.logP + a.logQ, a.Lfull);
      V[a.Lfull] = V[a.Lfull + 1] = 0;
      big_add_pow2(V, a.Lfull + 1, a.logP - 1);
      big_shr_mask(V, a.Lfull + 1, a.logP, a.logQ, a.L);
      // z = (d + k) mod 2^logQ
      const uint32_t* d = a.add + (size_t)o * a.add_outer + (size_t)i * a.add_inner + n;
      uint32_t cy = 0;
      for (uint32_t l = 0; l < a.L; ++l) {
        const uint64_t t = (uint64_t)V[l] + d[(size_t)l * a.N] + cy;
        V[l] = (uint32_t)t; cy = (uint32_t)(t >> 32);
      }
      V[a.L] = 0;                                                  // the carry out of 2^(32 L) is dropped by the mask below
      big_shr_mask(V, a.L, 0, a.logQ, a.L);
      if (a.rescale_bits) {
        V[a.L] = 0;
        big_add_pow2(V, a.L + 1, a.rescale_bits - 1);
        big_shr_mask(V, a.L + 1, a.rescale_bits, a.logQ - a.rescale_bits, a.L);
      }
      uint32_t* dst = a.out + (size_t)o * a.out_outer + (size_t)i * a.out_inner + n;
      for (uint32_t l = 0; l < a.L; ++l) dst[(size_t)l * a.N] = V[l];
    }
  }
}

// scratch layout of CrtEpi (words): negM table [nl + 2] | xs [Lx][TC] (BGV) | adds [L][TC] (relin modes) |
// BGV divide-by-P scratch [scratch_limbs][TC]
static void crt_scratch_layout(const CrtTarget& tg, const PostParams& pp, CrtParams& ep, size_t& bytes) {
  const bool relin = pp.mode == POST_CKKS_RELIN || pp.mode == POST_BGV_RELIN;
  const bool bgv = pp.mode == POST_BGV_MODQ || pp.mode == POST_BGV_RELIN;
  ep.ntab = tg.nchunks * (pipe::NC / 4);
  ep.nl = ep.ntab - CRT_ALPHA_COLS / 4 - (tg.top ? TOP_LIMBS : 0);
  ep.xs_off = (ep.ntab + 31) / 32 * 32;
  ep.adds_off = ep.xs_off + (bgv ? tg.Lx * TC : 0);
  ep.scratch_off = ep.adds_off + (relin ? pp.L * TC : 0);
  bytes = ((size_t)ep.scratch_off + (pp.mode == POST_BGV_RELIN ? pp.scratch_limbs * TC : 0)) * 4;
}

using CrtEpiAny = CrtEpi<POST_CKKS_MASK, false, false>;   // the pipeline shape (warps, groups, tile alternation) is the same for all

bool crt_target_fits(const CrtTarget& tg, const PostParams& pp) {
  CrtParams ep; size_t bytes;
  crt_scratch_layout(tg, pp, ep, bytes);
  return pipe::make_plan(tg.KB, tg.nchunks, bytes, true, CrtEpiAny::TILE_ALT).ok;
}

cudaError_t launch_crt(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_outer, size_t out_inner,
                       const uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_add, size_t add_outer,
                       size_t add_inner, uint32_t nouter, uint32_t ninner, cudaStream_t s, uint32_t* d_flags) {
  if (nouter * ninner == 0) return cudaSuccess;
  if (tg.top && !d_flags) return cudaErrorInvalidValue;
  if (small_crt_ok(c, tg, pp))                                     // small shapes: one thread per coefficient (kernels_small.cu)
    return launch_crt_small(c, tg, pp, d_out, out_outer, out_inner, d_res, res_outer, res_inner, nouter, ninner, s);
  CrtParams ep;
  size_t epi_bytes;
  crt_scratch_layout(tg, pp, ep, epi_bytes);
  pipe::Plan plan = pipe::make_plan(tg.KB, tg.nchunks, epi_bytes, true, CrtEpiAny::TILE_ALT);
  if (!plan.ok) return cudaErrorInvalidConfiguration;
  const bool relin = pp.mode == POST_CKKS_RELIN || pp.mode == POST_BGV_RELIN;
  if (relin && !d_add) return cudaErrorInvalidValue;
  // TMA staging of the residues: the source as a matrix [rows][N], polynomial (o, i) starting at row (o outer + i inner) / N
  CUtensorMap tmap;
  bool use_tma = false;
  if (res_outer % c->N == 0 && res_inner % c->N == 0 && tg.K <= 256 && c->force_pipe != 2) {
    pipe::add_ring(plan, tg.K);
    const uint64_t rows = (uint64_t)(nouter - 1) * (res_outer / c->N) + (uint64_t)(ninner - 1) * (res_inner / c->N) + tg.K;
    use_tma = plan.ring_slots > 0 && pipe::make_tensor_map(&tmap, d_res, rows, c->N, tg.K);
  }
  pipe::PipeArgs a;
  a.src = d_res; a.src_outer = res_outer; a.src_inner = res_inner;
  a.inner = ninner; a.npoly = nouter * ninner; a.N = c->N; a.nwords = tg.K; a.mask_bits = 0;
  a.B = tg.d_B; a.b_cols = tg.nchunks * pipe::NC;
  pipe::fill_args(a, plan);
  a.row_outer = (uint32_t)(res_outer / c->N); a.row_inner = (uint32_t)(res_inner / c->N);
  const CUtensorMap* tm = use_tma ? &tmap : nullptr;
  ep.out = d_out; ep.out_outer = out_outer; ep.out_inner = out_inner;
  ep.add = relin ? d_add : nullptr; ep.add_outer = add_outer; ep.add_inner = add_inner;
  ep.negM = tg.d_negM; ep.Lraw = tg.Lraw; ep.Lx = tg.Lx; ep.pp = pp;
  ep.tmq = top_mask(pp.logQ);
  // CKKS relin stream (CrtEpi): total = V + 2^(logP-1) + (d << s1) + 2^(s1+p-1), output = bits [s1 + p, ...) of it
  const uint32_t s1 = tg.top ? 0 : pp.logP;                      // the top form hands the epilogue V >> logP directly
  const uint32_t pb = pp.mode == POST_CKKS_RELIN ? pp.rescale_bits : 0, sh = s1 + pb;
  ep.wd = s1 >> 5; ep.bd = s1 & 31;
  ep.ws = sh >> 5; ep.bs = sh & 31;
  ep.rb1 = s1 ? (s1 - 1) >> 5 : 0; ep.rbit1 = s1 ? 1u << ((s1 - 1) & 31) : 0;
  ep.rb2 = pb ? (sh - 1) >> 5 : 0; ep.rbit2 = pb ? 1u << ((sh - 1) & 31) : 0;
  const uint32_t nb = pp.logQ - pb;
  ep.Lr = (nb + 31) / 32; ep.tm = top_mask(nb);
  ep.lend = ep.ws + pp.L;                                        // output limb m needs limbs ws + m and ws + m + 1 of the total
  ep.amb_bits = pp.amb_bits ? pp.amb_bits : TOP_AMB; ep.flags = d_flags;
  ep.m8 = 1u << 8; ep.m16 = 1u << 16; ep.m24 = 1u << 24;
  cudaError_t e;
  {
    LaunchTimer lt(c, KC_CRT, s);
    switch (pp.mode) {
      case POST_CKKS_MASK: e = pipe::launch_pipe<CrtEpi<POST_CKKS_MASK, false, false>>(a, ep, plan.smem, c->n_sm, s, tm); break;
      case POST_BGV_MODQ: e = pipe::launch_pipe<CrtEpi<POST_BGV_MODQ, false, false>>(a, ep, plan.smem, c->n_sm, s, tm); break;
      case POST_BGV_RELIN: e = pipe::launch_pipe<CrtEpi<POST_BGV_RELIN, false, false>>(a, ep, plan.smem, c->n_sm, s, tm); break;
      case POST_CKKS_RELIN:
        if (tg.top) e = pb ? pipe::launch_pipe<CrtEpi<POST_CKKS_RELIN, true, true>>(a, ep, plan.smem, c->n_sm, s, tm)
                           : pipe::launch_pipe<CrtEpi<POST_CKKS_RELIN, true, false>>(a, ep, plan.smem, c->n_sm, s, tm);
        else e = pb ? pipe::launch_pipe<CrtEpi<POST_CKKS_RELIN, false, true>>(a, ep, plan.smem, c->n_sm, s, tm)
                    : pipe::launch_pipe<CrtEpi<POST_CKKS_RELIN, false, false>>(a, ep, plan.smem, c->n_sm, s, tm);
        break;
      default: e = cudaErrorInvalidValue;
    }
  }
  if (e != cudaSuccess || !tg.top) return e;
  LaunchTimer lt(c, KC_CRT, s);
  ExactArgs x;
  x.flags = d_flags; x.res = d_res; x.res_outer = res_outer; x.res_inner = res_inner;
  x.add = d_add; x.add_outer = add_outer; x.add_inner = add_inner;
  x.out = d_out; x.out_outer = out_outer; x.out_inner = out_inner;
  x.W = tg.d_Wfull; x.negM = tg.d_negMfull; x.q = c->d_q;
  x.N = c->N; x.K = tg.K; x.Lfull = tg.Lfull; x.L = pp.L; x.logP = pp.logP; x.logQ = pp.logQ; x.rescale_bits = pp.rescale_bits;
  x.inner = ninner; x.nwords = nouter * ninner * (c->N >> 5);
  const uint32_t blocks = std::min<uint32_t>((x.nwords + 63) / 64, 4u * (uint32_t)c->n_sm);
  e = launch_pdl(crt_exact_kernel, blocks, 64, 0, s, x);
  return e != cudaSuccess ? e : cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// S7: standalone rescale, c' = ((c + 2^(p-1)) >> p) mod 2^(logQ - p).  HBM-bound:
// one thread per coefficient, limb-major so every limb access is a coalesced 128-byte line per warp.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
rescale_kernel(uint32_t* __restrict__ out, const uint32_t* __restrict__ in, uint32_t N, uint32_t L, uint32_t logQ,
               uint32_t p) {
  const uint32_t bpp = N / 256;
  const uint32_t poly = blockIdx.x / bpp;
  const uint32_t n = (blockIdx.x % bpp) * 256 + threadIdx.x;
  const uint32_t* src = in + (size_t)poly * L * N + n;
  uint32_t* dst = out + (size_t)poly * L * N + n;
  const uint32_t ws = p >> 5, bs = p & 31;
  const uint32_t rb = (p - 1) >> 5, rbit = 1u << ((p - 1) & 31);   // limb / bit receiving the rounding 2^(p-1)
  const uint32_t nb = logQ - p, Lr = (nb + 31) / 32, tm2 = top_mask(nb), tmq = top_mask(logQ);
  uint32_t carry = 0;
  // limb w of y = c + 2^(p-1), for w = rb, rb+1, ... in order (limbs below rb never reach the output)
  auto next = [&](uint32_t w) -> uint32_t {
    uint32_t v = 0;
    if (w < L) { v = __ldg(src + (size_t)w * N); if (w == L - 1) v &= tmq; }
    const uint32_t add = (w == rb ? rbit : 0u) + carry;
    const uint32_t s = v + add;
    carry = s < v;
    return s;
  };
  if (rb < ws) (void)next(rb);                    // p multiple of 32: the rounding bit sits one limb below
  uint32_t cur = next(ws);
  for (uint32_t l = 0; l < L; ++l) {
    uint32_t v = 0;
    if (l < Lr) {
      const uint32_t nx = next(ws + l + 1);
      v = bs ? ((cur >> bs) | (nx << (32 - bs))) : cur;
      if (l == Lr - 1) v &= tm2;
      cur = nx;
    }
    dst[(size_t)l * N] = v;
  }
}

cudaError_t launch_rescale(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t npoly, uint32_t p_bits,
                           cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  LaunchTimer lt(c, KC_RESCALE, s);
  rescale_kernel<<<(c->N / 256) * npoly, 256, 0, s>>>(d_out, d_in, c->N, c->L, c->logQ, p_bits);
  return cudaGetLastError();
}

}  // namespace fhe
