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
#include "umma.cuh"

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
__device__ __forceinline__ uint32_t top_mask(uint32_t bits) { return (bits & 31) ? ((1u << (bits & 31)) - 1u) : 0xFFFFFFFFu; }

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

// ------------------------------------------------------------------------------------------------------------------
// CRT kernel.  Block = 128 coefficients of one polynomial (thread = coefficient = TMEM lane).
//   phase 1  the residues y[i][n] are staged as the byte matrix A[n][4 i + b] (umma.cuh) and contracted on the tensor
//            cores with the constant image B: column 8 + e receives S_e = sum_{i,b} y_ib * byte_{e-b}(W_i), columns
//            0..5 the byte sums of sum_i y_i floor(2^48 / q_i) (-> alpha)
//   phase 2  per thread: V = sum_e S_e 2^(8 e) + alpha * negM, carries propagated four columns (one limb) at a time,
//            limbs written to this thread's column in shared memory (which reuses the A image's space)
//   phase 3  post-processing on the limb column (mask / divide-by-P + add [+ rescale] / BGV reductions), store
// ------------------------------------------------------------------------------------------------------------------
struct CrtArgs {
  const uint32_t* res; size_t res_poly_stride;
  uint32_t* out; size_t out_poly_stride;
  const uint32_t* add; size_t add_poly_stride;
  const uint8_t* B; const uint32_t* negM;
  uint32_t N, K, KB, NC, nchunks, Lraw, Lx, region_bytes;
};

__global__ void __launch_bounds__(TC)
crt_kernel(CrtArgs a, PostParams pp) {
  using namespace umma;
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ MmaPipe pipe;
  __shared__ uint32_t tmem_slot;
  uint8_t* sA = smem;                                          // [KB/16][128][16]; later the limb columns xs[Lx][TC]
  uint8_t* sB0 = smem + a.region_bytes;
  uint8_t* sB1 = sB0 + (size_t)a.KB * a.NC;
  uint32_t* xs = reinterpret_cast<uint32_t*>(smem);
  uint32_t* scratch = reinterpret_cast<uint32_t*>(sB0);        // BGV divide-by-P scratch column (B buffers are dead then)
  const uint32_t tid = threadIdx.x, warp = tid >> 5;
  const uint32_t bpp = a.N / TC;
  const uint32_t poly = blockIdx.x / bpp;
  const uint32_t n = (blockIdx.x % bpp) * TC + tid;
  const uint32_t ncols_alloc = pow2_cols(a.nchunks * a.NC);

  // phase 1
  stage_rows(sA, a.res + (size_t)poly * a.res_poly_stride + (n - tid), a.N, a.K, a.KB, 0);
  if (tid == 0) mma_pipe_init(&pipe);
  fence_proxy_async();
  __syncthreads();
  if (warp == 0) tmem_alloc(&tmem_slot, ncols_alloc);           // after staging: a co-resident CTA may still hold TMEM
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = tmem_slot;
  PipeState st = {{0, 0}, {0, 0}, 0};
  if (warp == 0) {   // lane 0 issues; its warp mates park at the convergence barrier instead of polling beside it
    if (tid == 0) mma_phase(&pipe, st, sA, sB0, sB1, a.KB, a.NC, a.B, (size_t)a.KB * a.NC, a.nchunks, tbase);
    __syncwarp();
  }
  mbar_wait(&pipe.done, 0);
  __syncthreads();                                              // nobody overwrites the A image before all MMAs are done
  tc_fence_after();

  // phase 2
  {
    const uint32_t lane_addr = tbase + ((warp * 32u) << 16);
    uint32_t t[32];
    tmem_ld32(lane_addr, t);
    uint64_t asum = 0;
#pragma unroll
    for (int e = 0; e < 6; ++e) asum += (uint64_t)t[e] << (8 * e);
    const uint32_t alpha = (uint32_t)((asum + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
    uint64_t carry = 0;
    uint32_t l = 0;
    // first load: columns 8..31 = limbs 0..5; later loads: eight limbs each
    for (uint32_t col = 0; l < a.Lraw; col += 32) {
      if (col) tmem_ld32(lane_addr + col, t);
#pragma unroll
      for (int g = 0; g < 8; ++g) {
        if ((col == 0 && g < CRT_ALPHA_COLS / 4) || l >= a.Lraw) continue;
        uint64_t v = carry + (uint64_t)alpha * __ldg(a.negM + l);
        v += (uint64_t)t[4 * g] + ((uint64_t)t[4 * g + 1] << 8) + ((uint64_t)t[4 * g + 2] << 16) + ((uint64_t)t[4 * g + 3] << 24);
        xs[l * TC + tid] = (uint32_t)v;
        carry = v >> 32;
        ++l;
      }
    }
    for (; l < a.Lx; ++l) { xs[l * TC + tid] = (uint32_t)carry; carry = 0; }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tbase, ncols_alloc);            // release TMEM before the (long) post-processing
  }

  // phase 3
  Col x{xs + tid};
  uint32_t* out = a.out + (size_t)poly * a.out_poly_stride + n;
  const uint32_t L = pp.L;
  if (pp.mode == POST_CKKS_MASK) {
    const uint32_t tm = top_mask(pp.logQ);
    for (uint32_t l = 0; l < L; ++l) {
      uint32_t v = x.get(l);
      if (l == L - 1) v &= tm;
      out[(size_t)l * a.N] = v;
    }
    return;
  }
  const uint32_t* addp = a.add + (size_t)poly * a.add_poly_stride + n;
  if (pp.mode == POST_CKKS_RELIN) {
    // k = ((X mod 2^logPQ + 2^(logP-1)) >> logP) mod 2^logQ ; bits above logP+logQ never reach k
    col_add_pow2(x, pp.logP - 1, a.Lx);
    uint32_t carry = 0;
    const uint32_t tm = top_mask(pp.logQ);
    for (uint32_t l = 0; l < L; ++l) {               // in place: reads limbs >= l, writes limb l
      uint32_t k = col_bits(x, pp.logP, l, a.Lx);
      uint64_t s = (uint64_t)k + __ldg(addp + (size_t)l * a.N) + carry;
      carry = (uint32_t)(s >> 32);
      uint32_t v = (uint32_t)s;
      if (l == L - 1) v &= tm;
      x.set(l, v);
    }
    if (pp.rescale_bits == 0) {
      for (uint32_t l = 0; l < L; ++l) out[(size_t)l * a.N] = x.get(l);
    } else {
      const uint32_t p = pp.rescale_bits;
      x.set(L, 0);                                   // room for the rounding carry (Lx >= L + 1)
      col_add_pow2(x, p - 1, L + 1);
      const uint32_t nb = pp.logQ - p;               // result bits
      const uint32_t Lr = (nb + 31) / 32;
      const uint32_t tm2 = top_mask(nb);
      for (uint32_t l = 0; l < L; ++l) {
        uint32_t v = 0;
        if (l < Lr) { v = col_bits(x, p, l, L + 1); if (l == Lr - 1) v &= tm2; }
        out[(size_t)l * a.N] = v;
      }
    }
    return;
  }
  if (pp.mode == POST_BGV_MODQ) {
    col_barrett1(x, a.Lx, pp.d_Q, L, pp.bitsQ, pp.mu1_Q);
    for (uint32_t l = 0; l < L; ++l) out[(size_t)l * a.N] = x.get(l);
    return;
  }
  // POST_BGV_RELIN: V -> xc = V mod PQ -> (q3, rem) = divmod(xc, P) -> centred r, kk -> (hi - kk + d) mod Q
  {
    const uint32_t LP = pp.L_P, LPQ = pp.L_PQ, g = pp.g_limbs;   // g = LPQ - LP
    col_barrett1(x, a.Lx, pp.d_PQ, LPQ, pp.bitsPQ, pp.mu1_PQ);   // x[0..LPQ) = xc
    // Barrett quotient estimate (HAC 14.42 generalised): q1 = xc >> 32(LP-1)  (g+1 limbs),
    // q3 = (q1 * mu) >> 32(g+1), mu = floor(2^(32 LPQ) / P)  (muP_limbs limbs); true quotient - q3 in {0,1,2}.
    Col sc{scratch + tid};                           // scratch column: pp.scratch_limbs limbs (B buffers are dead by now)
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
    Col q3{sc.p + (size_t)(g + 1) * TC};
    const uint32_t nq = n1;                          // limbs of q3 kept (q3 <= Q < 2^(32 (g+1)))
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
    uint32_t qinc = 0;
    for (int it = 0; it < 2; ++it) {
      if (x.get(LP) != 0 || col_ge(x, pp.d_P, LP)) { col_sub(x, pp.d_P, LP + 1); ++qinc; }
    }
    // centre: rem > (P-1)/2  <=>  2 rem > P - 1  <=> 2 rem >= P + 1 <=> 2 rem > P (P odd)
    bool neg;
    {
      // compare 2*rem with P from the top limb down (2*rem has LP+1 limbs)
      int cmp = 0;
      for (uint32_t l = LP + 1; l-- > 0 && cmp == 0;) {
        uint32_t hi = l < LP ? x.get(l) : 0u, lo = l >= 1 ? x.get(l - 1) : 0u;
        uint32_t two = (hi << 1) | (lo >> 31);
        uint32_t pv = l < LP ? __ldg(pp.d_P + l) : 0u;
        if (two != pv) cmp = two > pv ? 1 : -1;
      }
      neg = cmp > 0;
    }
    if (neg) ++qinc;                                 // hi = q + 1, r = rem - P
    // r mod t
    uint64_t rt = 0;
    for (uint32_t l = 0; l < LP; ++l) rt = (rt + (uint64_t)x.get(l) * __ldg(pp.d_pow32_t + l)) % pp.t;
    if (neg) { uint64_t Pt = __ldg(pp.d_pow32_t + LP); rt = (rt + pp.t - Pt) % pp.t; }   // d_pow32_t[LP] holds P mod t
    uint64_t kk = ((pp.t - rt) % pp.t) * pp.Pinv_t % pp.t;     // (-r P^-1) mod t in [0, t)
    const bool kneg = kk > pp.t / 2;                            // centred: kk - t
    const uint32_t kmag = kneg ? (uint32_t)(pp.t - kk) : (uint32_t)kk;
    // res = q3 + qinc - kk_centred, as an (L+1)-limb value in x[0..L], then mod Q, then + d mod Q
    {
      // x[l] <- q3[l] for l <= L (q3 has nq = g+1 limbs; zero beyond)
      int64_t adj = (int64_t)qinc + (kneg ? (int64_t)kmag : -(int64_t)kmag);
      // add signed small adj with carry/borrow propagation
      int64_t c = adj;
      for (uint32_t l = 0; l <= L; ++l) {
        int64_t v = (int64_t)(l < nq ? q3.get(l) : 0u) + c;
        x.set(l, (uint32_t)v);
        c = v >> 32;
      }
      // c == -1 here means the value is negative (only possible when q3 + qinc < kk): add Q
      if (c < 0) { col_add(x, pp.d_Q, L + 1); }
      else if (x.get(L) != 0 || col_ge(x, pp.d_Q, L)) col_sub(x, pp.d_Q, L + 1);
      // + d
      uint32_t carry = 0;
      for (uint32_t l = 0; l < L; ++l) {
        uint64_t s = (uint64_t)x.get(l) + __ldg(addp + (size_t)l * a.N) + carry;
        x.set(l, (uint32_t)s);
        carry = (uint32_t)(s >> 32);
      }
      x.set(L, carry);
      if (x.get(L) != 0 || col_ge(x, pp.d_Q, L)) col_sub(x, pp.d_Q, L + 1);
      for (uint32_t l = 0; l < L; ++l) out[(size_t)l * a.N] = x.get(l);
    }
  }
}

cudaError_t launch_crt(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_poly_stride,
                       const uint32_t* d_res, size_t res_poly_stride, const uint32_t* d_add, size_t add_poly_stride,
                       uint32_t npoly, cudaStream_t s) {
  if (!npoly) return cudaSuccess;
  CrtArgs a;
  a.res = d_res; a.res_poly_stride = res_poly_stride;
  a.out = d_out; a.out_poly_stride = out_poly_stride;
  a.add = d_add; a.add_poly_stride = add_poly_stride;
  a.B = tg.d_B; a.negM = tg.d_negM;
  a.N = c->N; a.K = tg.K; a.KB = tg.KB; a.NC = tg.NC; a.nchunks = tg.nchunks; a.Lraw = tg.Lraw; a.Lx = tg.Lx;
  a.region_bytes = std::max(tg.KB * 128u, tg.Lx * 512u);
  size_t tail = 2 * (size_t)tg.KB * tg.NC;
  if (pp.mode == POST_BGV_RELIN && (size_t)pp.scratch_limbs * TC * 4 > tail) tail = (size_t)pp.scratch_limbs * TC * 4;
  const size_t smem = a.region_bytes + tail;
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(crt_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    e = cudaFuncSetAttribute(crt_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  LaunchTimer lt(c, KC_CRT, s);
  crt_kernel<<<(c->N / TC) * npoly, TC, smem, s>>>(a, pp);
  return cudaGetLastError();
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
