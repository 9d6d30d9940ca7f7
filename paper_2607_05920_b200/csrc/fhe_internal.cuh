// fhe_internal.cuh -- context layout, launch declarations and device arithmetic shared by the kernels.
// Product code: nothing here is shared with oracle/ (tests only).
#pragma once
#include <cuda_runtime.h>
#include <cstdint>
#include <string>
#include <vector>

#include "../../include/fhe.h"

namespace fhe {

constexpr int MAX_LIMBS_IN = 104;              // widest decompose input (limbs); 416 bytes of contraction
constexpr int DEC_NC = 64;                     // decompose: columns per constant chunk = 16 primes x 4 constant bytes (= pipe::NC)
constexpr int CRT_ALPHA_COLS = 8;              // CRT: leading columns holding the byte sums of sum_i y_i floor(2^48 / q_i)
constexpr int ALPHA_SHIFT = 48;

// ---- CRT target: turns y_i = x_i * (M/q_i)^-1 mod q_i (i < K) into limbs of V = sum y_i W_i + alpha * negM -------------
// W_i = (M/q_i) mod T, negM = (-M) mod T, T = 2^(32 Lraw) (CKKS; masked later) or the odd modulus.  The sum is one
// u8 x u8 -> s32 tensor-core contraction over the bytes of the y_i (umma.cuh): column 8 + e collects byte position e.
struct CrtTarget {
  uint32_t K = 0;        // primes in the basis (prefix of the context's prime list)
  uint32_t KB = 0;       // contraction bytes: 4 K rounded up to a multiple of 32
  uint32_t nchunks = 0;  // 64-column chunks of the constant image (pipe::NC)
  uint32_t Lraw = 0;     // 32-bit limbs of V produced by the carry pass (4 Lraw value columns)
  uint32_t Lx = 0;       // limbs of the per-coefficient column the post-processing works on (>= Lraw + 1)
  uint8_t* d_B = nullptr;      // [KB/16][64 nchunks][16]: the constant matrix as K-major 16-byte core-matrix rows (pipe.cuh)
  uint32_t* d_negM = nullptr;  // [Lraw]
  uint2* d_scale = nullptr;    // [K]: N^-1 * (M/q_i)^-1 * 2^32 mod q_i and its Shoup companion (folded into the iNTT)
  uint8_t* d_decB_scaled = nullptr;   // decompose image whose constants carry d_scale: 2^(8 kb) s_j mod q_j (polymul / tensor targets)
  uint32_t* d_Wlimbs = nullptr; // small CKKS targets only (K <= SMALL_K, see kernels_small.cu): [K][Lraw] limbs of W_i, then [Lraw] negM
  // "Top" form of the CKKS relin target: the output needs floor((V mod 2^(logP+logQ) + 2^(logP-1)) >> logP)
  // mod 2^logQ only, i.e. the high logQ bits of W_i exactly and ONE carry out of the low logP bits.  That carry is taken
  // from the top TOP_BITS bits of the low parts (columns 8..31 of the image, then 4 L columns of the high parts); the
  // truncation can change it only when the TOP_AMB fractional bits below it are all ones, in which case the coefficient
  // is flagged (one bit per coefficient in a bitmap kept in the caller's workspace, written in full by every launch) and
  // recomputed exactly from the full constants by crt_exact_kernel.
  bool top = false;
  uint32_t Lfull = 0;              // limbs of the full constants: ceil((logP + logQ) / 32)
  uint32_t* d_Wfull = nullptr;     // [K][Lfull]: (M/q_i) mod 2^(logP+logQ)
  uint32_t* d_negMfull = nullptr;  // [Lfull]
};
constexpr uint32_t TOP_BITS = 96, TOP_LIMBS = 6, TOP_AMB = 58;
// Shapes below these bounds convert on the CUDA cores (kernels_small.cu): a 128-coefficient tile of the tensor-core pipeline
// costs a few thousand cycles whatever its size, which two-limb coefficients cannot amortise.
#ifndef FHE_SMALL_WORK
#define FHE_SMALL_WORK 192
#endif
constexpr uint32_t SMALL_K = 32, SMALL_LIMBS = 16, SMALL_WORK = FHE_SMALL_WORK;   // K, limbs, K x limbs
constexpr uint32_t SMALL_DEC_K = 128;          // primes the CUDA-core decompose has constants for

enum PostMode : int {
  POST_CKKS_MASK = 0,    // out = X mod 2^logQ
  POST_CKKS_RELIN = 1,   // out = (d + ((X mod 2^logPQ + P/2) >> logP)) mod 2^logQ  [then optional rescale]
  POST_BGV_MODQ = 2,     // out = V mod Q
  POST_BGV_RELIN = 3     // out = (d + round(V mod PQ / P) - kk) mod Q
};

struct PostParams {
  int mode;
  uint32_t L, L_PQ, logQ, logP, bitsQ, bitsP, bitsPQ;
  uint32_t rescale_bits;       // POST_CKKS_RELIN only; 0 = none
  uint32_t amb_bits;           // top-form relin target: fractional bits that must all be ones to flag a coefficient
  // BGV constants (device pointers, little-endian limbs)
  const uint32_t* d_Q;         // [L+1]
  const uint32_t* d_P;         // [L_P+1]
  const uint32_t* d_PQ;        // [L_PQ+1]
  const uint32_t* d_muP;       // Barrett constant for division by P: floor(2^(32 (L_P + g)) / P), g = quotient limbs
  uint32_t L_P, muP_limbs, g_limbs, scratch_limbs;
  uint64_t mu1_Q, mu1_PQ;      // floor(2^(bits+62) / Q), floor(2^(bitsPQ+62) / PQ): one-word Barrett quotient estimates
  uint32_t t, Pinv_t;          // plaintext modulus and P^-1 mod t
  // P = 2^logP + eP (the least odd integer above 2^logP that is 1 mod t).  fold_div: the divide-by-P of the BGV relinearisation
  // goes through that shape -- xc = A 2^logP + B = A P + (B - A eP), and when that is negative one more fold of the same kind
  // (kernels_crt.cu) -- instead of a general multi-limb Barrett division; set when logP >= 96 and the second fold's quotient
  // fits 60 bits (bits(eP) + bitsQ + 1 <= logP + 60: every shape with logQ <= logP + 38 or so)
  uint32_t eP, fold_div;
  uint32_t fold_full;          // fold_div on V itself, without reducing it mod PQ first (floor(V / P) mod Q and V mod P do not change
                               // with multiples of PQ): set when the second fold's quotient fits 95 bits and the quotient's fold mod Q 63
  uint32_t eQ, fold_modq;      // Q = 2^logQ + eQ; fold_modq: V mod Q as (V mod 2^logQ) - (V >> logQ) eQ (+ Q), set when eQ < 2^22 and logQ >= 64
  uint64_t mu_t;               // floor((2^64 - 1) / t) when t < 2^31 (word-sized Barrett steps mod t), else 0
  const uint32_t* d_pow32_t;   // [L_P+1]: 2^(32 i) mod t
};

struct Context {
  // parameters
  uint32_t N = 0, logN = 0, logQ = 0, logP = 0;
  uint64_t t = 0;
  uint32_t bitsQ = 0, bitsP = 0, bitsPQ = 0, L = 0, L_P = 0, L_PQ = 0;
  uint32_t K_pm = 0, K1 = 0, K2 = 0, Kmax = 0;
  int n_sm = 0;
  int device = 0;                 // the CUDA device the context was created on: every call must run with it current
  std::vector<uint32_t> h_q, h_psi;
  std::vector<uint32_t> h_Q, h_P, h_PQ;   // limbs
  // device tables (all primes 0..Kmax-1)
  uint32_t* d_q = nullptr;        // [Kmax]
  uint32_t* d_qinv_neg = nullptr; // [Kmax] -q^-1 mod 2^32 (Montgomery)
  uint2* d_qmu = nullptr;         // [Kmax] (q, floor(2^53 / q)): one-word Barrett pair of the decompose epilogue
  uint4* d_qsmall = nullptr;      // [Kmax] (q, 2^32 mod q, floor(2^61 / q), floor(2^48 / q)): the CUDA-core conversions
  uint32_t* d_pow32q = nullptr;   // [min(Kmax, SMALL_DEC_K)][SMALL_LIMBS]: 2^(32 l) mod q_j, the CUDA-core decompose
  uint2* d_tw_fwd = nullptr;      // [Kmax][N]: psi^bitrev(k) and Shoup companion; the inverse transforms read it mirrored (bf_inv)
  uint2* d_scale_plain = nullptr; // [Kmax]: N^-1 (debug inverse transform)
  uint8_t* d_decB = nullptr;      // [dec_KBimg/16][dec_cols][16]: byte c of 2^(8 kb) mod q_j at column 4 j + c
  uint32_t dec_cols = 0;          // columns of the decompose image: 64 ceil(Kmax / 16)
  uint32_t dec_KBimg = 0;         // contraction bytes covered by the decompose image (widest input, multiple of 32)
  CrtTarget tgt_pm, tgt_tensor, tgt_relin;
  bool fit_pm = false, fit_tensor = false, fit_relin = false;   // does the conversion pipeline hold the target (pipe.cuh)
  PostParams post_pm, post_tensor, post_relin;
  uint32_t *d_Qlimbs = nullptr, *d_Plimbs = nullptr, *d_PQlimbs = nullptr, *d_muP = nullptr, *d_pow32_t = nullptr;
  int force_pipe = 0;             // fhe_debug_force_pipeline: 0 auto; 1 the large-shape paths everywhere (tensor-core conversions,
                                  // three-pass NTT); 2 the small-shape paths wherever they exist (whole-transform NTT at N = 2^13 too)
  uint32_t amb_bits = TOP_AMB;    // fhe_debug_crt_ambiguity lowers it so that tests reach the exact path
  // evk-hat
  uint32_t* d_evk_hat = nullptr;  // [2][K2][N], forward NTT of the evk residues (plain domain)
  bool have_evk = false;
  // rotation / conjugation keys (NEXT-2): same form as the evk, one per slot, with the Galois element they belong to
  static constexpr int MAX_ROT_KEYS = 16;
  uint32_t* d_rot_hat[MAX_ROT_KEYS] = {};
  uint32_t rot_k[MAX_ROT_KEYS] = {};
  // copy streams and events of the host-buffer entry point (created with the context; the hot path creates nothing)
  static constexpr int HOST_PIECES = 32;
  cudaStream_t s_h2d = nullptr, s_d2h = nullptr;
  cudaEvent_t ev_start = nullptr, ev_in[HOST_PIECES] = {}, ev_done[HOST_PIECES] = {};
  // bookkeeping
  mutable std::string err;
  uint64_t launches = 0;
  std::vector<void*> allocs;
  // optional per-kernel timing (fhe_debug_timing): one CUDA event pair per launch, on the launch stream
  bool timing = false;
  struct Ev { int cls; cudaEvent_t a, b; };
  std::vector<Ev> events;
};

enum KernelClass : int { KC_DECOMPOSE = 0, KC_NTT_FWD = 1, KC_NTT_INV = 2, KC_POINTWISE = 3, KC_CRT = 4, KC_RESCALE = 5, KC_COUNT = 6 };

// brackets one kernel launch with events when timing is on (no-ops otherwise)
struct LaunchTimer {
  Context* c; cudaStream_t s; cudaEvent_t b = nullptr;
  LaunchTimer(Context* c_, int cls, cudaStream_t s_) : c(c_), s(s_) {
    c->launches++;
    if (!c->timing) return;
    Context::Ev e; e.cls = cls;
    if (cudaEventCreate(&e.a) != cudaSuccess || cudaEventCreate(&e.b) != cudaSuccess) return;
    cudaEventRecord(e.a, s);
    b = e.b;
    c->events.push_back(e);
  }
  ~LaunchTimer() { if (b) cudaEventRecord(b, s); }
};

// Programmatic dependent launch: the kernels of a step run back to back on one stream, each reading what the previous one
// wrote.  A kernel launched with launch_pdl may have its blocks scheduled while the last wave of the previous kernel is
// still running; pdl_sync() at its very top waits until that kernel has completed and its writes are visible
// (griddepcontrol.wait), then lets the next kernel's blocks be scheduled behind its own (griddepcontrol.launch_dependents).
// Nothing touches global memory before pdl_sync(); after an ordinary launch both instructions are no-ops.
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_sync() {
  asm volatile("griddepcontrol.wait;" ::: "memory");
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t s, Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = s;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at; cfg.numAttrs = 1;
  return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}
#endif

// ---- launchers (kernels_*.cu) --------------------------------------------------------------------------------------
// Polynomials of a launch are indexed (o, i), o < nouter, i < ninner, and live at base + o * outer + i * inner (words).
// decompose: limbs [Lin][N] -> residues [K][N] per polynomial; mask_bits > 0 reduces the input mod 2^mask_bits first;
// lazy: residues in [0, 2q) instead of [0, q) (what the forward transforms accept)
// tgt: the residues additionally carry that target's final constant (scaled constant image; nullptr: plain residues)
cudaError_t launch_decompose(Context* c, uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_limbs,
                             size_t limb_outer, size_t limb_inner, uint32_t nouter, uint32_t ninner, uint32_t Lin,
                             uint32_t K, uint32_t mask_bits, cudaStream_t s, bool lazy = true, const CrtTarget* tgt = nullptr);
// Transforms live in an item-major residue buffer [nitems][S][K][N] (S slots per item); slots 0..U-1 of every item
// are transformed in place.  Forward output is in bit-reversed order and canonical ([0, q)).
cudaError_t launch_ntt_fwd(Context* c, uint32_t* d_res, uint32_t nitems, uint32_t S, uint32_t U, uint32_t K, cudaStream_t s);
// Plain inverse of slots 0..U-1 (the debug entry point; the products go through launch_ntt_product).
// d_scale: per-prime final constant ([K] uint2, value and Shoup companion).
enum PwMode : int { PW_NONE = 0, PW_POLYMUL = 1, PW_TENSOR = 2, PW_RELIN = 3 };
cudaError_t launch_ntt_inv(Context* c, uint32_t* d_res, uint32_t nitems, uint32_t S, uint32_t U, uint32_t K,
                           const uint2* d_scale, cudaStream_t s);
// The product path: forward column pass over the operand slots, ONE fused row pass (last forward pass, pointwise
// products, first inverse pass, all in registers on the same 256-point row), inverse column pass over the result slots.
// The operands arrive untransformed (decompose output) in an item-major buffer [nitems][S][K][N]:
//   PW_POLYMUL S = 1: data <- INTT(NTT(data) * NTT(aux)), aux = [ceil(nitems / aux_group)][K][N], transformed in place too
//   PW_TENSOR  S = 4: slots (a0, a1, b0, b1) -> slots 0..2 = INTT(a0^ b0^, a0^ b1^ + a1^ b0^, a1^ b1^)
//   PW_RELIN   S = 2: slot 0 = d2 -> slots 0, 1 = INTT(d2^ * aux[0], d2^ * aux[1]), aux = a key already in the NTT domain [2][K][N]
// (Montgomery products: each carries a factor 2^-32 that the folded constant removes.)
// aux_group (PW_POLYMUL): item i multiplies aux polynomial i / aux_group, of which there are ceil(nitems / aux_group).
// The final constant of the inverse (CrtTarget::d_scale) is NOT applied here: it rides on an operand -- the second factor is
// decomposed with the target's scaled constant image (Context::d_decB_pm / d_decB_tensor), a key is multiplied by it when it
// is installed (launch_scale_rows).
cudaError_t launch_ntt_product(Context* c, uint32_t* d_res, uint32_t* d_aux, uint32_t nitems, uint32_t K, int pw_mode,
                               cudaStream_t s, uint32_t aux_group = 1);
cudaError_t launch_scale_rows(Context* c, uint32_t* d_res, uint32_t npoly, uint32_t K, const uint2* d_scale, cudaStream_t s);
// CRT + post: residues [K][N] -> limbs [L][N] per polynomial (o, i); d_add: for the relin modes, the polynomial added
// at the end, else nullptr.  d_flags: top-form targets only, nouter * ninner * N / 32 words of workspace for the bitmap of the
// coefficients the exact path recomputes (written in full by the launch: no initialisation needed)
cudaError_t launch_crt(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_outer, size_t out_inner,
                       const uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_add, size_t add_outer,
                       size_t add_inner, uint32_t nouter, uint32_t ninner, cudaStream_t s, uint32_t* d_flags = nullptr);
// CUDA-core conversions for small shapes (kernels_small.cu): same contracts as launch_decompose / launch_crt (CKKS mask mode)
bool small_decompose_ok(const Context* c, uint32_t Lin_eff, uint32_t K);
cudaError_t launch_decompose_small(Context* c, uint32_t* d_res, size_t res_outer, size_t res_inner, const uint32_t* d_limbs,
                                   size_t limb_outer, size_t limb_inner, uint32_t nouter, uint32_t ninner, uint32_t Lin_eff,
                                   uint32_t K, uint32_t mask_bits, cudaStream_t s, const uint2* d_scale);
bool small_crt_ok(const Context* c, const CrtTarget& tg, const PostParams& pp);
cudaError_t launch_crt_small(Context* c, const CrtTarget& tg, const PostParams& pp, uint32_t* d_out, size_t out_outer, size_t out_inner,
                             const uint32_t* d_res, size_t res_outer, size_t res_inner, uint32_t nouter, uint32_t ninner, cudaStream_t s);
// register-only throughput of the NTT butterfly (mode 0), mad.lo.u32 (1), mul.hi.u32 (2) on this device, per second
cudaError_t measure_int_peak(Context* c, int mode, double* per_s, cudaStream_t s);
bool crt_target_fits(const CrtTarget& tg, const PostParams& pp);   // does the pipeline have the TMEM / shared memory for it
// coefficient-wise ring operations (kernels_elem.cu): op 0 add, 1 sub, 2 negate, 3 reduce mod 2^bits (CKKS); bits = the
// modulus width the result is masked to (CKKS)
cudaError_t launch_elem(Context* c, int op, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly,
                        uint32_t bits, cudaStream_t s);
// Galois automorphism X -> X^k (k odd) of ciphertexts (kernels_elem.cu): in2 [B][2][L][N] -> out3 [B][3][L][N] =
// (sigma(c0), 0, sigma(c1)), the triple the key switch of a rotation consumes
cudaError_t launch_automorphism(Context* c, uint32_t* d_out3, const uint32_t* d_in2, uint32_t k, uint32_t batch, cudaStream_t s);
// out = X^k * in mod (X^N + 1, Q), 0 <= k < 2N, per polynomial (kernels_elem.cu); out must not alias in
cudaError_t launch_monomial(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t k, uint32_t npoly, cudaStream_t s);
cudaError_t launch_add_plain(Context* c, uint32_t* d_out, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                             uint32_t group, cudaStream_t s);
cudaError_t launch_mult_scalar(Context* c, uint32_t* d_out, const uint32_t* d_in, int32_t k, uint32_t npoly, cudaStream_t s);
// BGV modulus switch from Q = 2^logQ + e to Q' = 2^new_logQ + e2 (kernels_elem.cu), per coefficient of npoly polynomials [L][N]
cudaError_t launch_modswitch(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logQ, uint32_t e, uint32_t e2,
                             uint32_t npoly, cudaStream_t s);
// offset of the modulus above its power of two: 0 (t == 0), else the least odd c with 2^log + c = 1 (mod t)   (ctx.cu)
uint64_t modulus_offset(uint32_t log, uint64_t t);
cudaError_t launch_rescale(Context* c, uint32_t* d_out, const uint32_t* d_in, uint32_t npoly, uint32_t p_bits,
                           cudaStream_t s);

// ---- device arithmetic ------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ uint32_t mulhi32(uint32_t a, uint32_t b) { return __umulhi(a, b); }

// x in [0, 2q) -> [0, q)
__device__ __forceinline__ uint32_t csub(uint32_t x, uint32_t q) { return min(x, x - q); }
// a b + c with a 64-bit sum (IMAD.WIDE.U32): one instruction on the FMA pipe
__device__ __forceinline__ uint64_t madw(uint32_t a, uint32_t b, uint64_t c) {
  uint64_t d;
  asm("mad.wide.u32 %0, %1, %2, %3;" : "=l"(d) : "r"(a), "r"(b), "l"(c));
  return d;
}

// Shoup multiplication by a constant w < q with companion w' = floor(w 2^32 / q): result in [0, 2q), any a < 2^32.
__device__ __forceinline__ uint32_t mul_shoup_lazy(uint32_t a, uint32_t w, uint32_t wp, uint32_t q) {
  uint32_t h = mulhi32(a, wp);
  return a * w - h * q;
}
__device__ __forceinline__ uint32_t mul_shoup(uint32_t a, uint32_t w, uint32_t wp, uint32_t q) {
  return csub(mul_shoup_lazy(a, w, wp, q), q);
}
// Montgomery reduction of t < 2^63 (t < 2 q^2 suffices): returns t 2^-32 mod q in [0, q).  qn = -q^-1 mod 2^32.
__device__ __forceinline__ uint32_t mont_redc(uint64_t t, uint32_t q, uint32_t qn) {
  uint32_t m = (uint32_t)t * qn;
  uint64_t u = t + (uint64_t)m * q;   // < 2^64: t < 2^63, m q < 2^63
  return csub((uint32_t)(u >> 32), q);
}
// acc * 2^32 + limb  mod t   (acc < t < 2^31; mu = floor(2^64 / t) or one less)
__device__ __forceinline__ uint32_t horner_mod(uint32_t acc, uint32_t limb, uint32_t t, uint64_t mu) {
  const uint64_t v = ((uint64_t)acc << 32) | limb;
  uint64_t r = v - __umul64hi(v, mu) * t;                           // quotient estimate at most 2 short: r in [0, 3 t)
  if (r >= t) r -= t;
  if (r >= t) r -= t;
  return (uint32_t)r;
}
// v < 2^49 -> v mod q with mu = floor(2^53 / q): the quotient estimate mulhi(v >> 21, mu) is floor(v/q) or one less
// (v >> 21 < 2^28 and mu < 2^24 lose < 2^-4 + 2^-8 of a unit), so the 32-bit remainder lies in [0, 2q).
__device__ __forceinline__ uint32_t barrett49(uint64_t v, uint32_t q, uint32_t mu) {
  const uint32_t qh = __umulhi((uint32_t)(v >> 21), mu);
  return csub((uint32_t)v - qh * q, q);
}
#endif

}  // namespace fhe
