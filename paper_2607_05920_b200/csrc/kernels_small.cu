// kernels_small.cu -- the two base conversions on the CUDA cores, for small shapes (S1 limb -> RNS; S5 RNS ->
// limb, Eq. 1 at PAPER.md:77).
//
// The tensor-core pipeline (pipe.cuh) pays about two thousand cycles of barriers, tensor-memory round trips and MMA latency
// per 128-coefficient tile whatever the tile holds.  With two-limb coefficients and five primes (the logQ = 64 cells of the
// polymul sweep) a tile is 3.5 KB of traffic -- 160 cycles at the SM's share of HBM -- and with eight limbs and 18 primes
// (logQ = 256) 13 KB.  Below K <= 32, limbs <= 16, K x limbs <= SMALL_WORK the arithmetic is small enough for the CUDA cores,
// one thread per PAIR of adjacent coefficients (8-byte accesses: twice the bytes in flight per thread):
//   decompose   r_j = sum_l x_l (2^(32 l) mod q_j) mod q_j -- the paper's own formulation -- with the
//               sum kept lazily in 64 bits: one multiply-add per limb above the first and prime, a "fold" (v -> hi32(v) (2^32 mod q)
//               + lo32(v), the same residue below 2^62 + 2^32) after limb 4 and after every three more, one word-sized
//               Barrett step at the end
//   CRT         V = sum_i y_i W_i + alpha negM mod 2^(32 Lraw) limb by limb: 64-bit sums of four products each, added into a
//               96-bit accumulator, alpha as in kernels_crt.cu; CKKS mask mode (the product is reduced mod 2^logQ)
// Both are streaming kernels, limb-major and prime-major accesses coalesced over the coefficient index.
#include "fhe_internal.cuh"

namespace fhe {

constexpr int SMALL_THREADS = 128;   // threads per block, each with two adjacent coefficients: 256 coefficients per chunk
#ifndef FHE_SMALL_CHUNKS
#define FHE_SMALL_CHUNKS 8
#endif
constexpr uint32_t SMALL_CHUNKS = FHE_SMALL_CHUNKS;   // chunks a block walks (a power of two): the constants reach shared memory once per block

// v -> the same residue mod q below 2^62 + 2^32 (c32 = 2^32 mod q < 2^30)
__device__ __forceinline__ uint64_t fold32(uint64_t v, uint32_t c32) { return madw((uint32_t)(v >> 32), c32, (uint64_t)(uint32_t)v); }
// v < 2^60 + 2^32 -> v mod q, q < 2^30: the estimate floor((v >> 29) floor(2^61 / q) / 2^32) is the quotient or up to 2 less,
// so the 32-bit remainder is below 3 q
__device__ __forceinline__ uint32_t barrett60(uint64_t v, uint32_t q, uint32_t mu61) {
  const uint32_t qh = __umulhi((uint32_t)(v >> 29), mu61);
  uint32_t t = (uint32_t)v - qh * q;
  t = min(t, t - 2 * q);
  return min(t, t - q);
}

// LMAX: compile-time bound of the limb count (2, 4, 8, 12, 16): the loops over the limbs are unrolled over registers; limbs
// between Lin and LMAX are zero and cost their multiply-adds.
// Bounds of the lazy sum: a product is below (2^32 - 1)(2^30 - 1) < 2^62 - 2^32, so limb 0 (taken as it is) plus four products
// stay below 2^64, and so does a folded value (< 2^62 + 2^32) plus three products.  Two folds bring any 64-bit value below
// 2^60 + 2^32 (the second one multiplies at most 2^30 by c32 < 2^30), which barrett60 accepts.
template <int LMAX>
__global__ void __launch_bounds__(SMALL_THREADS)
decompose_small_kernel(uint32_t* __restrict__ res, size_t res_outer, size_t res_inner, const uint32_t* __restrict__ limbs,
                       size_t limb_outer, size_t limb_inner, uint32_t inner, uint32_t N, uint32_t Lin, uint32_t K,
                       uint32_t mask_bits, const uint4* __restrict__ qsmall, const uint32_t* __restrict__ pow32q,
                       const uint2* __restrict__ scale, uint32_t cpb) {
  pdl_sync();
  constexpr int LP = LMAX < 4 ? 4 : LMAX;                          // constants of a prime: LP words, read four at a time
  __shared__ uint4 sq[SMALL_DEC_K];
  __shared__ __align__(16) uint32_t sp[SMALL_DEC_K * LP];
  for (uint32_t j = threadIdx.x; j < K; j += SMALL_THREADS) sq[j] = __ldg(qsmall + j);
  for (uint32_t k = threadIdx.x; k < K * LP; k += SMALL_THREADS) sp[k] = (k % LP) < (uint32_t)LMAX ? __ldg(pow32q + (k / LP) * SMALL_LIMBS + k % LP) : 0u;
  __syncthreads();
  const uint32_t bpp = N / (2 * SMALL_THREADS) / cpb;              // blocks per polynomial, each walking cpb chunks (powers of two)
  const uint32_t poly = blockIdx.x / bpp, po = poly / inner, pi = poly % inner;
  for (uint32_t cc = 0; cc < cpb; ++cc) {
  const uint32_t n = ((blockIdx.x % bpp) * cpb + cc) * 2 * SMALL_THREADS + 2 * threadIdx.x;
  const uint32_t* src = limbs + (size_t)po * limb_outer + (size_t)pi * limb_inner + n;
  uint32_t* dst = res + (size_t)po * res_outer + (size_t)pi * res_inner + n;
  uint32_t x0[LMAX], x1[LMAX];                                     // the two coefficients' limbs
#pragma unroll
  for (int l = 0; l < LMAX; ++l) {
    const uint2 v = (uint32_t)l < Lin ? __ldg(reinterpret_cast<const uint2*>(src + (size_t)l * N)) : make_uint2(0u, 0u);
    x0[l] = v.x; x1[l] = v.y;
  }
  // mask_bits != 0 reduces the input mod 2^mask_bits: its top limb is cut (the limbs above are not loaded: Lin says so)
  const uint32_t mask_w = (mask_bits & 31) ? (mask_bits >> 5) : 0xFFFFFFFFu, mask_m = (1u << (mask_bits & 31)) - 1u;
#pragma unroll
  for (int l = 0; l < LMAX; ++l) {
    const uint32_t m = (uint32_t)l == mask_w ? mask_m : 0xFFFFFFFFu;
    x0[l] &= m; x1[l] &= m;
  }
#pragma unroll 2
  for (uint32_t j = 0; j < K; ++j) {
    const uint4 qc = sq[j];                                        // (q, 2^32 mod q, floor(2^61 / q), floor(2^48 / q))
    uint32_t cw[LP];
#pragma unroll
    for (int l = 0; l < LP; l += 4) {
      const uint4 v = *reinterpret_cast<const uint4*>(sp + j * LP + l);
      cw[l] = v.x; cw[l + 1] = v.y; cw[l + 2] = v.z; cw[l + 3] = v.w;
    }
    uint64_t acc0 = x0[0], acc1 = x1[0];                           // limb 0's constant is 2^0 mod q = 1: no multiplication
#pragma unroll
    for (int l = 1; l < LMAX; ++l) {
      acc0 = madw(x0[l], cw[l], acc0);
      acc1 = madw(x1[l], cw[l], acc1);
      if (l >= 4 && (l - 4) % 3 == 0 && l + 1 < LMAX) {           // after limbs 4, 7, 10, 13
        acc0 = fold32(acc0, qc.y);
        acc1 = fold32(acc1, qc.y);
      }
    }
    acc0 = fold32(acc0, qc.y);
    acc1 = fold32(acc1, qc.y);
    if constexpr (LMAX > 2) {                                      // two limbs: x0 + x1 c < 2^62 + 2^32 already, one fold is enough
      acc0 = fold32(acc0, qc.y);
      acc1 = fold32(acc1, qc.y);
    }
    uint32_t r0 = barrett60(acc0, qc.x, qc.z), r1 = barrett60(acc1, qc.x, qc.z);
    if (scale) {                                                   // the product's final constant rides here
      const uint2 sc = __ldg(scale + j);
      r0 = mul_shoup(r0, sc.x, sc.y, qc.x); r1 = mul_shoup(r1, sc.x, sc.y, qc.x);
    }
    *reinterpret_cast<uint2*>(dst + (size_t)j * N) = make_uint2(r0, r1);   // canonical
  }
  }
}

// 96-bit accumulator of 64-bit sums
struct Acc96 {
  uint32_t a0 = 0, a1 = 0, a2 = 0;
  __device__ __forceinline__ void add(uint64_t g) {
    asm("add.cc.u32 %0, %0, %3;\n\taddc.cc.u32 %1, %1, %4;\n\taddc.u32 %2, %2, 0;"
        : "+r"(a0), "+r"(a1), "+r"(a2) : "r"((uint32_t)g), "r"((uint32_t)(g >> 32)));
  }
  __device__ __forceinline__ uint32_t pop() { const uint32_t v = a0; a0 = a1; a1 = a2; a2 = 0; return v; }
};

// KMAX: compile-time bound of K + 1 (8, 16, 24, 32): slot K of the operand vector holds alpha, row K of the constants negM,
// slots and rows beyond are zero.  A product is below 2^62 (y < 2^30, alpha < 2^9, constants < 2^32), so four of them fit a
// 64-bit sum; a limb's column sum is below 32 x 2^62 plus a carry: 96 bits.
template <int KMAX>
__global__ void __launch_bounds__(SMALL_THREADS)
crt_small_kernel(uint32_t* __restrict__ out, size_t out_outer, size_t out_inner, const uint32_t* __restrict__ res,
                 size_t res_outer, size_t res_inner, uint32_t inner, uint32_t N, uint32_t K, uint32_t Lraw, uint32_t L,
                 uint32_t tmq, const uint32_t* __restrict__ Wl, const uint4* __restrict__ qsmall, uint32_t cpb) {
  pdl_sync();
  __shared__ __align__(16) uint32_t sW[SMALL_LIMBS * KMAX];       // [limb][slot]: a limb's constants side by side, four per load
  __shared__ uint32_t sF[KMAX];
  for (uint32_t k = threadIdx.x; k < Lraw * KMAX; k += SMALL_THREADS) {
    const uint32_t l = k / KMAX, i = k % KMAX;
    sW[k] = i <= K ? __ldg(Wl + i * Lraw + l) : 0u;
  }
  for (uint32_t j = threadIdx.x; j < (uint32_t)KMAX; j += SMALL_THREADS) sF[j] = j < K ? __ldg(qsmall + j).w : 0u;
  __syncthreads();
  const uint32_t bpp = N / (2 * SMALL_THREADS) / cpb;              // blocks per polynomial, each walking cpb chunks (powers of two)
  const uint32_t poly = blockIdx.x / bpp, po = poly / inner, pi = poly % inner;
  for (uint32_t cc = 0; cc < cpb; ++cc) {
  const uint32_t n = ((blockIdx.x % bpp) * cpb + cc) * 2 * SMALL_THREADS + 2 * threadIdx.x;
  const uint32_t* src = res + (size_t)po * res_outer + (size_t)pi * res_inner + n;
  uint32_t* dst = out + (size_t)po * out_outer + (size_t)pi * out_inner + n;
  uint32_t y0[KMAX], y1[KMAX];                                     // the two coefficients' operand vectors
  uint64_t asum0 = 0, asum1 = 0;
#pragma unroll
  for (int i = 0; i < KMAX; ++i) {
    const uint2 v = (uint32_t)i < K ? __ldg(reinterpret_cast<const uint2*>(src + (size_t)i * N)) : make_uint2(0u, 0u);
    y0[i] = v.x; y1[i] = v.y;
    asum0 = madw(v.x, sF[i], asum0);                               // y floor(2^48 / q) < 2^49 each
    asum1 = madw(v.y, sF[i], asum1);
  }
  const uint32_t alpha0 = (uint32_t)((asum0 + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
  const uint32_t alpha1 = (uint32_t)((asum1 + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
#pragma unroll
  for (int i = 0; i < KMAX; ++i) {
    y0[i] = (uint32_t)i == K ? alpha0 : y0[i];
    y1[i] = (uint32_t)i == K ? alpha1 : y1[i];
  }
  Acc96 acc0, acc1;
  for (uint32_t l = 0; l < L; ++l) {                               // limbs l >= L of V are not needed (mod 2^logQ)
    const uint32_t* wrow = sW + l * KMAX;
#pragma unroll
    for (int i = 0; i < KMAX; i += 4) {
      const uint4 w = *reinterpret_cast<const uint4*>(wrow + i);
      acc0.add(madw(y0[i], w.x, madw(y0[i + 1], w.y, madw(y0[i + 2], w.z, (uint64_t)y0[i + 3] * w.w))));
      acc1.add(madw(y1[i], w.x, madw(y1[i + 1], w.y, madw(y1[i + 2], w.z, (uint64_t)y1[i + 3] * w.w))));
    }
    const uint32_t v0 = acc0.pop(), v1 = acc1.pop();
    *reinterpret_cast<uint2*>(dst + (size_t)l * N) = l == L - 1 ? make_uint2(v0 & tmq, v1 & tmq) : make_uint2(v0, v1);
  }
  }
}

// chunks per block: up to SMALL_CHUNKS (the constants reach shared memory once per block), but only while the launch still has
// several blocks for every block slot of the device -- a small launch keeps one chunk per block and all the parallelism it has
static uint32_t chunks_per_block(const Context* c, uint32_t npoly) {
  const uint32_t cpp = c->N / (2 * SMALL_THREADS);
  uint32_t cpb = cpp < SMALL_CHUNKS ? cpp : SMALL_CHUNKS;
  while (cpb > 1 && (uint64_t)(cpp / cpb) * npoly < (uint64_t)64 * c->n_sm) cpb >>= 1;
  return cpb;
}

bool small_decompose_ok(const Context* c, uint32_t Lin_eff, uint32_t K) {
  return c->force_pipe != 1 && c->d_pow32q && K <= SMALL_DEC_K && Lin_eff <= SMALL_LIMBS && K * Lin_eff <= SMALL_WORK && c->N >= 2 * SMALL_THREADS;
}
bool small_crt_ok(const Context* c, const CrtTarget& tg, const PostParams& pp) {
  return c->force_pipe != 1 && pp.mode == POST_CKKS_MASK && tg.d_Wlimbs != nullptr && tg.K < SMALL_K && tg.Lraw <= SMALL_LIMBS &&
         tg.K * tg.Lraw <= SMALL_WORK && c->N >= 2 * SMALL_THREADS && pp.L <= tg.Lraw;
}

cudaError_t launch_decompose_small(Context* c, uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_limbs,
                                   size_t limb_outer, size_t limb_inner, uint32_t nouter, uint32_t ninner, uint32_t Lin_eff,
                                   uint32_t K, uint32_t mask_bits, cudaStream_t s, const uint2* d_scale) {
  LaunchTimer lt(c, KC_DECOMPOSE, s);
  const uint32_t cpb = chunks_per_block(c, nouter * ninner), grid = (c->N / (2 * SMALL_THREADS) / cpb) * nouter * ninner;
  cudaError_t e;
#define DEC_SMALL(LM) launch_pdl(decompose_small_kernel<LM>, grid, SMALL_THREADS, 0, s, d_res, res_outer, res_inner, d_limbs, \
                                 limb_outer, limb_inner, ninner, c->N, Lin_eff, K, mask_bits, (const uint4*)c->d_qsmall, (const uint32_t*)c->d_pow32q, d_scale, cpb)
  if (Lin_eff <= 2) e = DEC_SMALL(2);
  else if (Lin_eff <= 4) e = DEC_SMALL(4);
  else if (Lin_eff <= 8) e = DEC_SMALL(8);
  else if (Lin_eff <= 12) e = DEC_SMALL(12);
  else e = DEC_SMALL(16);
#undef DEC_SMALL
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_crt_small(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_outer, size_t out_inner,
                             const uint32_t* d_res, size_t res_outer, size_t res_inner, uint32_t nouter, uint32_t ninner, cudaStream_t s) {
  LaunchTimer lt(c, KC_CRT, s);
  const uint32_t cpb = chunks_per_block(c, nouter * ninner), grid = (c->N / (2 * SMALL_THREADS) / cpb) * nouter * ninner;
  const uint32_t tmq = (pp.logQ & 31) ? ((1u << (pp.logQ & 31)) - 1u) : 0xFFFFFFFFu;
  cudaError_t e;
#define CRT_SMALL(KM) launch_pdl(crt_small_kernel<KM>, grid, SMALL_THREADS, 0, s, d_out, out_outer, out_inner, d_res, res_outer, res_inner, \
                                 ninner, c->N, tg.K, tg.Lraw, pp.L, tmq, (const uint32_t*)tg.d_Wlimbs, (const uint4*)c->d_qsmall, cpb)
  if (tg.K < 8) e = CRT_SMALL(8);                                  // K + 1 slots (alpha rides in slot K)
  else if (tg.K < 16) e = CRT_SMALL(16);
  else if (tg.K < 24) e = CRT_SMALL(24);
  else e = CRT_SMALL(32);
#undef CRT_SMALL
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace fhe
