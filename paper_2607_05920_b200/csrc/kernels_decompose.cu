// kernels_decompose.cu -- S1: limb -> RNS decomposition on the tensor cores.
//
// The paper computes r_j = sum_i limb_i * (2^(32 i) mod q_j) mod q_j one coefficient and one prime at a time.  That
// sum is a dense contraction of the coefficient's bytes with a constant matrix, so it runs as one integer GEMM per
// 128-coefficient tile on the conversion pipeline (pipe.cuh):
//     T[n][4 j + c] = sum_kb byte_kb(X_n) * byte_c(2^(8 kb) mod q_j)        u8 x u8 -> s32, exact
//     r_j(X_n)      = (T[n][4j] + 2^8 T[n][4j+1] + 2^16 T[n][4j+2] + 2^24 T[n][4j+3]) mod q_j
// The CUDA cores only do the epilogue: recombine the four byte sums (< 2^49) and one word-sized Barrett reduction.
#include "fhe_internal.cuh"
#include "pipe.cuh"

namespace fhe {

// Epilogue of the pipeline: a 64-column accumulator chunk holds the byte sums of 16 primes; each of the GROUPS epilogue
// warp groups takes 16 / GROUPS of them.  (q_j, floor(2^53 / q_j)) sit in shared memory, padded to whole chunks.
// Per residue: the low word of v = T0 + 2^8 T1 + 2^16 T2 + 2^24 T3 (< 2^49) exactly, an estimate vh <= v >> 21 that
// is at most 20 short (the shifted-out bits of T1, T2 and T0 >> 21 < 16), and one Barrett step: qh = mulhi(vh, mu) is
// floor(v / q) or one less (20 * 2^21 / q < 0.16 for q > 2^28), so the 32-bit remainder lies in [0, 2q).
struct DecParams {
  uint32_t* res; size_t res_outer, res_inner;   // residues of polynomial (o, i) at res + o * res_outer + i * res_inner, [K][N]
  const uint2* qmu;                             // (q_j, floor(2^53 / q_j))
  uint32_t K;
};
// LAZY: the residues leave in [0, 2q) (no final conditional subtraction) -- what the forward transform's lazy butterflies
// accept (kernels_ntt.cu); the debug entry point asks for canonical ones.
template <bool LAZY>
struct DecEpi {
  // Measured on the role timers (C5, 28 tiles per CTA): with two groups splitting every chunk's columns, the chunks of a span
  // were drained one after the other, the span's columns came back 1800 cycles after the MMAs had finished and the next
  // tile's MMA chain (2100 cycles from first issue to commit) could not start before: 4500 cycles per tile with neither the
  // tensor pipe nor the epilogue busy.  Four groups taking whole chunks side by side hand a span back within a few hundred.
  static constexpr int LOAD_WORDS = 40, MAX_REGS = 72;   // 25 warps are allocated as 28: 28 x 32 x 72 <= 64 K
  static constexpr uint32_t GROUPS = 4, LOAD_WARPS = 8;
  static constexpr bool TILE_ALT = false, CHUNK_ALT = true;
  static constexpr bool LOAD_TMA = false;                // staging the limbs through shared memory by TMA (as the CRT does) measured
                                                         // 0.017 ms slower per step than two tiles of register-landing loads
  static constexpr bool LOAD_ALT = true;                 // the loads of two tiles in flight: with four loader warps (one tile) the
                                                         // MMA thread waited 1400 cycles per tile for its A operand
  static constexpr int PPG = 8;                          // primes per consume call: half a chunk
  using Params = DecParams;
  const Params& p;
  const uint32_t N, etid;
  const uint2* tab;
  uint32_t* out = nullptr;
  __device__ DecEpi(const Params& p_, const pipe::PipeArgs& a, uint8_t* sm, uint32_t etid_, uint32_t grp, uint32_t bar)
      : p(p_), N(a.N), etid(etid_), tab(reinterpret_cast<const uint2*>(sm)) {
    uint2* w = reinterpret_cast<uint2*>(sm);
    for (uint32_t j = grp * 128 + etid; j < a.nchunks * 16; j += 128 * GROUPS) w[j] = j < p.K ? make_uint2(0u - __ldg(p.qmu + j).x, __ldg(p.qmu + j).y) : make_uint2(0u, 0u);
    pipe::epi_sync(bar, 128 * GROUPS);
  }
  __device__ __forceinline__ void begin_tile(uint32_t o, uint32_t i, uint32_t n0) {
    out = p.res + (size_t)o * p.res_outer + (size_t)i * p.res_inner + n0 + etid;
  }
  // qm = (2^32 - q, floor(2^53 / q)): with -q in the table the remainder is one multiply-add, lo + qh * (-q).  (Forming the
  // 48-bit value with three 64-bit multiply-adds and one funnel shift -- 4 instructions for these 6 -- measured 0.025 ms
  // SLOWER per step, and one multiply-add per store address 0.009 ms slower: IMAD.WIDE does not issue at the rate of the
  // shifts and adds it replaces.)
  __device__ __forceinline__ uint32_t reduce(const uint32_t* t, const uint2 qm) const {
    const uint32_t lo = t[0] + (t[1] << 8) + (t[2] << 16) + (t[3] << 24);
    const uint32_t vh = (t[3] << 3) + (t[2] >> 5) + (t[1] >> 13);
    const uint32_t qh = __umulhi(vh, qm.y);
    const uint32_t r = lo + qh * qm.x;
    return LAZY ? r : csub(r, 0u - qm.x);
  }
  // The constants are read (two primes per 16-byte load) and all residues of the call computed before the first store: a
  // store through `out` may alias the table as far as the compiler knows, and interleaved they run one residue at a time
  // (LDS -> chain -> STG: 65 cycles per residue measured) instead of PPG independent chains.
  __device__ __forceinline__ void consume(uint32_t col0, const uint32_t* t) {
    const uint32_t j0 = col0 / 4;
    uint4 qm2[PPG / 2];
#pragma unroll
    for (int e = 0; e < PPG / 2; ++e) qm2[e] = reinterpret_cast<const uint4*>(tab + j0)[e];
    uint32_t r[PPG];
#pragma unroll
    for (int e = 0; e < PPG; e += 2) {
      r[e] = reduce(t + 4 * e, make_uint2(qm2[e / 2].x, qm2[e / 2].y));
      r[e + 1] = reduce(t + 4 * e + 4, make_uint2(qm2[e / 2].z, qm2[e / 2].w));
    }
    uint32_t* o = out + (size_t)j0 * N;
    if (j0 + PPG <= p.K) {
#pragma unroll
      for (int e = 0; e < PPG; ++e) { *o = r[e]; o += N; }
    } else {
#pragma unroll
      for (int e = 0; e < PPG; ++e) {
        if (j0 + e < p.K) *o = r[e];
        o += N;
      }
    }
  }
  __device__ __forceinline__ void end_tile() {}
};

cudaError_t launch_decompose(Context* c, uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_limbs,
                             size_t limb_outer, size_t limb_inner, uint32_t nouter, uint32_t ninner, uint32_t Lin,
                             uint32_t K, uint32_t mask_bits, cudaStream_t s, bool lazy, const CrtTarget* tgt) {
  if (nouter * ninner == 0) return cudaSuccess;
  uint32_t eff = Lin;
  if (mask_bits && (mask_bits + 31) / 32 < eff) eff = (mask_bits + 31) / 32;
  const uint32_t KB = (4 * eff + 31) / 32 * 32;
  if (KB > c->dec_KBimg || K > c->Kmax) return cudaErrorInvalidValue;
  if (small_decompose_ok(c, eff, K))                               // small shapes: one thread per coefficient (kernels_small.cu)
    return launch_decompose_small(c, d_res, res_outer, res_inner, d_limbs, limb_outer, limb_inner, nouter, ninner, eff, K, mask_bits, s,
                                  tgt ? tgt->d_scale : nullptr);
  if (tgt && (!tgt->d_decB_scaled || K != tgt->K)) return cudaErrorInvalidValue;
  const pipe::Plan plan = pipe::make_plan(KB, (K + 15) / 16, (size_t)((K + 15) / 16) * 16 * sizeof(uint2), false);
  if (!plan.ok || plan.nA != 2) return cudaErrorInvalidConfiguration;
  pipe::PipeArgs a;
  a.src = d_limbs; a.src_outer = limb_outer; a.src_inner = limb_inner;
  a.inner = ninner; a.npoly = nouter * ninner; a.N = c->N; a.nwords = eff; a.mask_bits = mask_bits;
  a.B = tgt ? tgt->d_decB_scaled : c->d_decB; a.b_cols = c->dec_cols;
  pipe::fill_args(a, plan);
  DecParams ep;
  ep.res = d_res; ep.res_outer = res_outer; ep.res_inner = res_inner; ep.qmu = c->d_qmu; ep.K = K;
  LaunchTimer lt(c, KC_DECOMPOSE, s);
  return lazy ? pipe::launch_pipe<DecEpi<true>>(a, ep, plan.smem, c->n_sm, s)
              : pipe::launch_pipe<DecEpi<false>>(a, ep, plan.smem, c->n_sm, s);
}

}  // namespace fhe
