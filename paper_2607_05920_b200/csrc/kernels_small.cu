// kernels_small.cu -- the two base conversions on the CUDA cores, for small shapes (S1 limb -> RNS; S5 RNS ->
// limb, Eq. 1 at PAPER.md:77).
//
// The tensor-core pipeline (pipe.cuh) pays a few thousand cycles of barriers, tensor-memory round trips and MMA latency per
// 128-coefficient tile whatever the tile holds.  With two-limb coefficients and five primes (the logQ = 64 cells of the
// polymul sweep) a tile is 3.5 KB of traffic -- 160 cycles at the SM's share of HBM -- so those cells ran at a fifth of the
// bandwidth.  Below K <= 32, limbs <= 16, K x limbs <= 48 the arithmetic is small enough for one thread per coefficient
// (measured: at K x limbs = 144 the pipeline is the faster one again):
//   decompose   r_j = X mod q_j by Horner over the limbs, r <- (r 2^32 + x_l) mod q_j, one word-sized Barrett step each
//               (this is the paper's own formulation)
//   CRT         V = sum_i y_i W_i + alpha negM mod 2^(32 Lraw) limb by limb with a 96-bit accumulator, alpha as in
//               kernels_crt.cu; CKKS mask mode (the product is reduced mod 2^logQ)
// Both are streaming kernels, limb-major and prime-major accesses coalesced over the coefficient index.
#include "fhe_internal.cuh"

namespace fhe {

constexpr int SMALL_THREADS = 256;

// (r 2^32 + x) mod q for r < q < 2^30:  v = r c32 + x < 2^60 + 2^32,  c32 = 2^32 mod q;  the estimate
// floor((v >> 29) floor(2^61 / q) / 2^32) is the quotient or up to 2 less, so the remainder is below 3 q
__device__ __forceinline__ uint32_t horner_step(uint32_t r, uint32_t x, const uint4 qc) {
  const uint64_t v = (uint64_t)r * qc.y + x;
  const uint32_t qh = __umulhi((uint32_t)(v >> 29), qc.z);
  uint32_t t = (uint32_t)v - qh * qc.x;
  t = min(t, t - 2 * qc.x);
  return min(t, t - qc.x);
}

// LMAX: compile-time bound of the limb count (2, 4, 8, 16): the loops over the limbs are unrolled over registers, and every
// predicated-off iteration would still cost its issue slots
template <int LMAX>
__global__ void __launch_bounds__(SMALL_THREADS)
decompose_small_kernel(uint32_t* __restrict__ res, size_t res_outer, size_t res_inner, const uint32_t* __restrict__ limbs,
                       size_t limb_outer, size_t limb_inner, uint32_t inner, uint32_t N, uint32_t Lin, uint32_t K,
                       uint32_t mask_bits, const uint4* __restrict__ qsmall, const uint2* __restrict__ scale) {
  pdl_sync();
  __shared__ uint4 sq[SMALL_K * 4];
  for (uint32_t j = threadIdx.x; j < K; j += SMALL_THREADS) sq[j] = __ldg(qsmall + j);
  __syncthreads();
  const uint32_t bpp = N / SMALL_THREADS;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * SMALL_THREADS + threadIdx.x;
  const uint32_t po = poly / inner, pi = poly % inner;
  const uint32_t* src = limbs + (size_t)po * limb_outer + (size_t)pi * limb_inner + n;
  uint32_t* dst = res + (size_t)po * res_outer + (size_t)pi * res_inner + n;
  uint32_t x[LMAX];
#pragma unroll
  for (int l = 0; l < LMAX; ++l) x[l] = (uint32_t)l < Lin ? __ldg(src + (size_t)l * N) : 0u;
  if (mask_bits & 31) {
#pragma unroll
    for (int l = 0; l < LMAX; ++l)
      if ((uint32_t)l == (mask_bits >> 5)) x[l] &= (1u << (mask_bits & 31)) - 1u;
  }
#pragma unroll 2
  for (uint32_t j = 0; j < K; ++j) {
    const uint4 qc = sq[j];
    uint32_t r = 0;                                                // limbs >= Lin are zero: their Horner steps leave r = 0
#pragma unroll
    for (int l = LMAX - 1; l >= 0; --l) r = (LMAX > 2 && (uint32_t)l >= Lin) ? r : horner_step(r, x[l], qc);
    if (scale) { const uint2 sc = __ldg(scale + j); r = mul_shoup(r, sc.x, sc.y, qc.x); }   // the product's final constant rides here
    dst[(size_t)j * N] = r;                                        // canonical
  }
}

// 96-bit accumulator acc += a * b
struct Acc96 {
  uint32_t a0 = 0, a1 = 0, a2 = 0;
  __device__ __forceinline__ void mad(uint32_t a, uint32_t b) {
    asm("mad.lo.cc.u32 %0, %3, %4, %0;\n\tmadc.hi.cc.u32 %1, %3, %4, %1;\n\taddc.u32 %2, %2, 0;"
        : "+r"(a0), "+r"(a1), "+r"(a2) : "r"(a), "r"(b));
  }
  __device__ __forceinline__ uint32_t pop() { const uint32_t v = a0; a0 = a1; a1 = a2; a2 = 0; return v; }
};

// KMAX: compile-time bound of the prime count (8, 16, 32), as LMAX above
template <int KMAX>
__global__ void __launch_bounds__(SMALL_THREADS)
crt_small_kernel(uint32_t* __restrict__ out, size_t out_outer, size_t out_inner, const uint32_t* __restrict__ res,
                 size_t res_outer, size_t res_inner, uint32_t inner, uint32_t N, uint32_t K, uint32_t Lraw, uint32_t L,
                 uint32_t tmq, const uint32_t* __restrict__ Wl, const uint4* __restrict__ qsmall) {
  pdl_sync();
  __shared__ uint32_t sW[(SMALL_K + 1) * SMALL_LIMBS];
  __shared__ uint32_t sF[SMALL_K];
  for (uint32_t k = threadIdx.x; k < (K + 1) * Lraw; k += SMALL_THREADS) sW[k] = __ldg(Wl + k);
  for (uint32_t j = threadIdx.x; j < K; j += SMALL_THREADS) sF[j] = __ldg(qsmall + j).w;
  __syncthreads();
  const uint32_t bpp = N / SMALL_THREADS;
  const uint32_t poly = blockIdx.x / bpp, n = (blockIdx.x % bpp) * SMALL_THREADS + threadIdx.x;
  const uint32_t po = poly / inner, pi = poly % inner;
  const uint32_t* src = res + (size_t)po * res_outer + (size_t)pi * res_inner + n;
  uint32_t* dst = out + (size_t)po * out_outer + (size_t)pi * out_inner + n;
  uint32_t y[KMAX];
  uint64_t asum = 0;
#pragma unroll
  for (int i = 0; i < KMAX; ++i) {
    y[i] = (uint32_t)i < K ? __ldg(src + (size_t)i * N) : 0u;
    if ((uint32_t)i < K) asum += (uint64_t)y[i] * sF[i];
  }
  const uint32_t alpha = (uint32_t)((asum + (1ull << (ALPHA_SHIFT - 1))) >> ALPHA_SHIFT);
  Acc96 acc;
  for (uint32_t l = 0; l < L; ++l) {                               // limbs l >= L of V are not needed (mod 2^logQ)
#pragma unroll
    for (int i = 0; i < KMAX; ++i)
      if (KMAX <= 8 || (uint32_t)i < K) acc.mad(y[i], sW[i * Lraw + l]);   // y[i] = 0 beyond K: the small bound skips the test
    acc.mad(alpha, sW[K * Lraw + l]);
    const uint32_t v = acc.pop();
    dst[(size_t)l * N] = l == L - 1 ? (v & tmq) : v;
  }
}

bool small_decompose_ok(const Context* c, uint32_t Lin_eff, uint32_t K) {
  return c->force_pipe != 1 && K <= 4 * SMALL_K && Lin_eff <= SMALL_LIMBS && K * Lin_eff <= SMALL_WORK && c->N >= SMALL_THREADS;
}
bool small_crt_ok(const Context* c, const CrtTarget& tg, const PostParams& pp) {
  return c->force_pipe != 1 && pp.mode == POST_CKKS_MASK && tg.d_Wlimbs != nullptr && tg.K * tg.Lraw <= SMALL_WORK &&
         c->N >= SMALL_THREADS && pp.L <= tg.Lraw;
}

cudaError_t launch_decompose_small(Context* c, uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_limbs,
                                   size_t limb_outer, size_t limb_inner, uint32_t nouter, uint32_t ninner, uint32_t Lin_eff,
                                   uint32_t K, uint32_t mask_bits, cudaStream_t s, const uint2* d_scale) {
  LaunchTimer lt(c, KC_DECOMPOSE, s);
  const uint32_t grid = (c->N / SMALL_THREADS) * nouter * ninner;
  cudaError_t e;
#define DEC_SMALL(LM) launch_pdl(decompose_small_kernel<LM>, grid, SMALL_THREADS, 0, s, d_res, res_outer, res_inner, d_limbs, \
                                 limb_outer, limb_inner, ninner, c->N, Lin_eff, K, mask_bits, (const uint4*)c->d_qsmall, d_scale)
  if (Lin_eff <= 2) e = DEC_SMALL(2);
  else if (Lin_eff <= 4) e = DEC_SMALL(4);
  else if (Lin_eff <= 8) e = DEC_SMALL(8);
  else e = DEC_SMALL(16);
#undef DEC_SMALL
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_crt_small(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_outer, size_t out_inner,
                             const uint32_t* d_res, size_t res_outer, size_t res_inner, uint32_t nouter, uint32_t ninner, cudaStream_t s) {
  LaunchTimer lt(c, KC_CRT, s);
  const uint32_t grid = (c->N / SMALL_THREADS) * nouter * ninner;
  const uint32_t tmq = (pp.logQ & 31) ? ((1u << (pp.logQ & 31)) - 1u) : 0xFFFFFFFFu;
  cudaError_t e;
#define CRT_SMALL(KM) launch_pdl(crt_small_kernel<KM>, grid, SMALL_THREADS, 0, s, d_out, out_outer, out_inner, d_res, res_outer, res_inner, \
                                 ninner, c->N, tg.K, tg.Lraw, pp.L, tmq, (const uint32_t*)tg.d_Wlimbs, (const uint4*)c->d_qsmall)
  if (tg.K <= 8) e = CRT_SMALL(8);
  else if (tg.K <= 16) e = CRT_SMALL(16);
  else e = CRT_SMALL(32);
#undef CRT_SMALL
  return e != cudaSuccess ? e : cudaGetLastError();
}

}  // namespace fhe
