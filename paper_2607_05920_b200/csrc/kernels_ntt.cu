// kernels_ntt.cu -- S2/S4 negacyclic NTT (Eq. 8-9) with S3, the pointwise products (PAPER.md:354-356,
// Eq. 7), formed in registers between the last forward and the first inverse pass (ntt_row_fused_kernel).
//
// Formulation: merged-psi Cooley-Tukey forward / Gentleman-Sande inverse; the psi^j "twist" of
// PAPER.md:346-350 lives in the butterfly twiddles, so there is no separate twist pass.  tw[k] = psi^bitrev(k); the
// inverse needs psi^-bitrev(k) = -tw[3m - 1 - k] (m = the level of k) and reads the same table (bf_inv).  A forward stage with m groups pairs j and j + N/(2m) with twiddle index m + group;
// the forward output is in bit-reversed order, the pointwise products do not care and the inverse undoes it.
//
// Split (the paper's two-pass / four-step idea): N = N1 * 256.  The first log2 N1 stages act on
// "columns" (stride 256) with the N1-point prefix of the table, the last 8 stages on contiguous 256-point "rows" r with
// table indices (N1 + r) m' + i'.  Both are one "local transform with base": twiddle index = base * m' + i' (base = 1
// for columns, N1 + r for row r), so the paper's separate twiddle-multiplication pass and transpose do not exist.
//
// Each pass is register-tiled: a thread owns 16 points, runs four radix-2 stages on them in registers, trades points
// with the other threads of its sub-transform through shared memory once, and runs the remaining (up to four) stages
// in registers again.  Butterflies are Harvey's lazy ones with Shoup twiddles: values stay in [0, 4q) (forward) resp.
// [0, 2q) (inverse), which is why the primes are below 2^30 (PAPER.md:312 allows 30- or 31-bit).  Only the last pass
// of a transform brings values back to [0, q).
#include "fhe_internal.cuh"

namespace fhe {

// ---- butterflies ----------------------------------------------------------------------------------------------------
// forward: X, Y in [0, 4q) -> X + wY, X - wY in [0, 4q)
__device__ __forceinline__ void bf_fwd(uint32_t& X, uint32_t& Y, const uint2 w, const uint32_t q, const uint32_t q2) {
  const uint32_t x = min(X, X - q2);
  const uint32_t t = mul_shoup_lazy(Y, w.x, w.y, q);
  X = x + t;
  Y = x - t + q2;
}
// inverse: X, Y in [0, 2q) -> X + Y, w^-1 (X - Y) in [0, 2q).  There is no inverse table: with k = m + i, 0 <= i < m,
// psi^-bitrev(k) = -psi^bitrev(3m - 1 - k) (psi^N = -1, and the bit reversal of the complement of i is the complement of its
// bit reversal), so the inverse stages read the FORWARD table mirrored inside each level -- w below is tw_fwd[3m - 1 - k] --
// and the sign goes into the difference: w^-1 (X - Y) = w (Y - X).  Same instructions as with a table of its own; half the
// twiddle bytes, and in the fused row pass both directions hit the same L1 lines.
__device__ __forceinline__ void bf_inv(uint32_t& X, uint32_t& Y, const uint2 w, const uint32_t q, const uint32_t q2) {
  const uint32_t s = X + Y;
  const uint32_t d = Y - X + q2;
  X = min(s, s - q2);
  Y = mul_shoup_lazy(d, w.x, w.y, q);
}
// mirror of a base inside its level: a local transform with base b in [m0, 2 m0) uses twiddle indices (b << s) + i at its
// stage s; mirrored, (mir_base(b, m0) << s) + (2^s - 1 - i)
__device__ __forceinline__ uint32_t mir_base(uint32_t base, uint32_t m0) { return 3 * m0 - 1 - base; }

template <int NG>
__device__ __forceinline__ void load_tw(const uint2* __restrict__ p, uint2 (&w)[8]) {
  if constexpr (NG == 1) {
    w[0] = __ldg(p);
  } else {
#pragma unroll
    for (int g = 0; g < NG; g += 2) {
      const uint4 v = __ldg(reinterpret_cast<const uint4*>(p + g));
      w[g] = make_uint2(v.x, v.y);
      w[g + 1] = make_uint2(v.z, v.w);
    }
  }
}

// Stage with S = log2(groups inside the thread's points): H = E >> (S + 1) is the register stride, the thread's
// 1 << S twiddles are consecutive table entries starting at `tw`.
template <int E, int S, bool INV>
__device__ __forceinline__ void reg_stage(uint32_t (&x)[16], const uint2* __restrict__ tw, uint32_t q, uint32_t q2) {
  constexpr int NG = 1 << S, H = E >> (S + 1);
  uint2 w[8];
  load_tw<NG>(tw, w);
#pragma unroll
  for (int g = 0; g < NG; ++g)
#pragma unroll
    for (int k = 0; k < H; ++k) {
      const int i0 = g * 2 * H + k;
      if (!INV) bf_fwd(x[i0], x[i0 + H], w[g], q, q2);
      else bf_inv(x[i0], x[i0 + H], w[NG - 1 - g], q, q2);           // mirrored table: `tw` points at the mirrored block
    }
}

// Phase A of a local transform of 2^LN points, LN > 4: the thread's 16 points differ in the top four index bits; the
// first NS = min(4, LN - 4) stages of the local transform (phase B runs the last four).  The twiddles do not depend on
// the thread: index (base << s) + g.
template <bool INV, int NS>
__device__ __forceinline__ void phase_a(uint32_t (&x)[16], const uint2* __restrict__ tw, uint32_t base, uint32_t q, uint32_t q2) {
  if (!INV) {
    reg_stage<16, 0, false>(x, tw + base, q, q2);
    if constexpr (NS > 1) reg_stage<16, 1, false>(x, tw + 2 * base, q, q2);
    if constexpr (NS > 2) reg_stage<16, 2, false>(x, tw + 4 * base, q, q2);
    if constexpr (NS > 3) reg_stage<16, 3, false>(x, tw + 8 * base, q, q2);
  } else {
    if constexpr (NS > 3) reg_stage<16, 3, true>(x, tw + 8 * base, q, q2);
    if constexpr (NS > 2) reg_stage<16, 2, true>(x, tw + 4 * base, q, q2);
    if constexpr (NS > 1) reg_stage<16, 1, true>(x, tw + 2 * base, q, q2);
    reg_stage<16, 0, true>(x, tw + base, q, q2);
  }
}
// Phase B: the thread's E = min(16, 2^LN) points are contiguous, starting at local index tb * E; local stages
// LN - log2(E) .. LN - 1.  Stage with S in-thread group bits uses twiddles ((base << s) + (tb << S)) + g, s = LN - log2 E + S.
template <int LN, bool INV>
__device__ __forceinline__ void phase_b(uint32_t (&x)[16], const uint2* __restrict__ tw, uint32_t base, uint32_t tb, uint32_t q, uint32_t q2) {
  constexpr int LE = LN < 4 ? LN : 4, E = 1 << LE, S0 = LN - LE;
  if (INV) tb = (1u << S0) - 1 - tb;                               // inverse: `base` is the mirrored base, and the thread's block mirrors too
#define STG(S) reg_stage<E, S, INV>(x, tw + (base << (S0 + S)) + (tb << S), q, q2)
  if (!INV) {
    if constexpr (LE > 0) STG(0);
    if constexpr (LE > 1) STG(1);
    if constexpr (LE > 2) STG(2);
    if constexpr (LE > 3) STG(3);
  } else {
    if constexpr (LE > 3) STG(3);
    if constexpr (LE > 2) STG(2);
    if constexpr (LE > 1) STG(1);
    if constexpr (LE > 0) STG(0);
  }
#undef STG
}

// The same stages on NOPS sequences that share every twiddle (adjacent columns of one prime in the column pass): the
// twiddles are loaded once per stage.
template <int NOPS, int E, int S, bool INV>
__device__ __forceinline__ void reg_stage_multi(uint32_t (&x)[NOPS][16], const uint2* __restrict__ tw, uint32_t q, uint32_t q2) {
  constexpr int NG = 1 << S, H = E >> (S + 1);
  uint2 w[8];
  load_tw<NG>(tw, w);
#pragma unroll
  for (int o = 0; o < NOPS; ++o)
#pragma unroll
    for (int g = 0; g < NG; ++g)
#pragma unroll
      for (int k = 0; k < H; ++k) {
        const int i0 = g * 2 * H + k;
        if (!INV) bf_fwd(x[o][i0], x[o][i0 + H], w[g], q, q2);
        else bf_inv(x[o][i0], x[o][i0 + H], w[NG - 1 - g], q, q2);
      }
}
template <int NOPS, bool INV, int NS>
__device__ __forceinline__ void phase_a_multi(uint32_t (&x)[NOPS][16], const uint2* __restrict__ tw, uint32_t base, uint32_t q, uint32_t q2) {
  if (!INV) {
    reg_stage_multi<NOPS, 16, 0, false>(x, tw + base, q, q2);
    if constexpr (NS > 1) reg_stage_multi<NOPS, 16, 1, false>(x, tw + 2 * base, q, q2);
    if constexpr (NS > 2) reg_stage_multi<NOPS, 16, 2, false>(x, tw + 4 * base, q, q2);
    if constexpr (NS > 3) reg_stage_multi<NOPS, 16, 3, false>(x, tw + 8 * base, q, q2);
  } else {
    if constexpr (NS > 3) reg_stage_multi<NOPS, 16, 3, true>(x, tw + 8 * base, q, q2);
    if constexpr (NS > 2) reg_stage_multi<NOPS, 16, 2, true>(x, tw + 4 * base, q, q2);
    if constexpr (NS > 1) reg_stage_multi<NOPS, 16, 1, true>(x, tw + 2 * base, q, q2);
    reg_stage_multi<NOPS, 16, 0, true>(x, tw + base, q, q2);
  }
}
template <int NOPS, int LN, bool INV>
__device__ __forceinline__ void phase_b_multi(uint32_t (&x)[NOPS][16], const uint2* __restrict__ tw, uint32_t base, uint32_t tb, uint32_t q, uint32_t q2) {
  constexpr int S0 = LN - 4;
  if (INV) tb = (1u << S0) - 1 - tb;
#define STGM(S) reg_stage_multi<NOPS, 16, S, INV>(x, tw + (base << (S0 + S)) + (tb << S), q, q2)
  if (!INV) { STGM(0); STGM(1); STGM(2); STGM(3); }
  else { STGM(3); STGM(2); STGM(1); STGM(0); }
#undef STGM
}

__device__ __forceinline__ uint32_t canon4(uint32_t v, uint32_t q, uint32_t q2) { v = min(v, v - q2); return min(v, v - q); }

// Montgomery product: a b 2^-32 mod q in [0, q) (the inverse transform's final constant carries the 2^32)
__device__ __forceinline__ uint32_t mm(uint32_t a, uint32_t b, uint32_t q, uint32_t qn) {
  return mont_redc((uint64_t)a * b, q, qn);
}

struct NttArgs {
  uint32_t* data;            // transforms: item-major [nitems][S][K][N]; slots 0..U-1 of every item are transformed
  const uint32_t* aux;       // PW_POLYMUL: b [nitems][K][N]; PW_RELIN: evk-hat [2][K][N]
  const uint2* tw;           // [Kmax][N] psi^bitrev(k) with Shoup companions: the one table of both directions (bf_inv)
  const uint32_t* q;         // [Kmax]
  const uint32_t* qn;        // [Kmax] -q^-1 mod 2^32
  const uint2* scale;        // [K] final constant of the inverse (with Shoup companion)
  uint32_t N, K, N1, S, U, units, nitems;
  uint32_t aux_group;        // PW_POLYMUL: item i multiplies aux polynomial i / aux_group (1: pairwise; > 1: shared operand)
  // Traversal order, so that a pass STARTS on what the pass before it wrote LAST (the tail of a 260-350 MB output is still in
  // the L2 when the next kernel begins).  Column pass: 0 = transforms in memory order (item, slot, prime); 1 = prime-major,
  // ascending.  Fused row pass: 1 = units in descending order.
  uint32_t order;
};
#ifndef NTT_L2_ORDER
#define NTT_L2_ORDER 1
#endif

// ------------------------------------------------------------------------------------------------------------------
// Column pass: 2^LN-point transforms over elements e * 256 + c (c = column), in place.  A block owns T adjacent
// columns of one (polynomial, prime); thread (t, cc) works on column cc; the block always has 256 threads and
// 4096 points.  Shared-memory tile [e][cc]: every access of a warp is to 32 (or 16) consecutive words.
// ------------------------------------------------------------------------------------------------------------------
template <int LN, bool INV>
__global__ void __launch_bounds__(256, 6)
ntt_col_kernel(NttArgs a) {
  pdl_sync();
  constexpr int LE = LN < 4 ? LN : 4, E = 1 << LE;   // points per thread
  constexpr int TPC = (1 << LN) / E;                 // threads per column
  constexpr int T = 256 / TPC;                       // columns per block
  __shared__ uint32_t sm[LN > 4 ? 4096 : 1];
  const uint32_t tid = threadIdx.x, cc = tid % T, t = tid / T;
  const uint32_t tiles = 256 / T;
  const uint32_t tr = blockIdx.x / tiles, c0 = (blockIdx.x % tiles) * T;
  const uint32_t item = tr / (a.U * a.K), rem = tr % (a.U * a.K), slot = rem / a.K, j = rem % a.K;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q;
  const uint2* tw = a.tw + (size_t)j * a.N;
  uint32_t* g = a.data + ((size_t)(item * a.S + slot) * a.K + j) * a.N + c0 + cc;
  uint32_t x[16];

  if constexpr (LN > 4) {
    if (!INV) {
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = g[(size_t)(i * TPC + t) * 256];
      phase_a<false, LN - 4>(x, tw, 1, q, q2);
#pragma unroll
      for (int i = 0; i < 16; ++i) sm[(i * TPC + t) * T + cc] = x[i];
      __syncthreads();
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = sm[(t * 16 + i) * T + cc];
      phase_b<LN, false>(x, tw, 1, t, q, q2);
#pragma unroll
      for (int i = 0; i < 16; ++i) g[(size_t)(t * 16 + i) * 256] = x[i];
    } else {
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = g[(size_t)(t * 16 + i) * 256];
      phase_b<LN, true>(x, tw, 1, t, q, q2);
#pragma unroll
      for (int i = 0; i < 16; ++i) sm[(t * 16 + i) * T + cc] = x[i];
      __syncthreads();
#pragma unroll
      for (int i = 0; i < 16; ++i) x[i] = sm[(i * TPC + t) * T + cc];
      phase_a<true, LN - 4>(x, tw, 1, q, q2);
      if (a.scale) {
        const uint2 sc = __ldg(a.scale + j);
#pragma unroll
        for (int i = 0; i < 16; ++i) g[(size_t)(i * TPC + t) * 256] = mul_shoup(x[i], sc.x, sc.y, q);
      } else {                                                     // the constant rides on an operand (fold_scale): canonicalise only
#pragma unroll
        for (int i = 0; i < 16; ++i) g[(size_t)(i * TPC + t) * 256] = csub(x[i], q);
      }
    }
  } else {
#pragma unroll
    for (int i = 0; i < E; ++i) x[i] = g[(size_t)i * 256];
    phase_b<LN, INV>(x, tw, 1, 0, q, q2);
    if (!INV) {
#pragma unroll
      for (int i = 0; i < E; ++i) g[(size_t)i * 256] = x[i];
    } else if (a.scale) {
      const uint2 sc = __ldg(a.scale + j);
#pragma unroll
      for (int i = 0; i < E; ++i) g[(size_t)i * 256] = mul_shoup(x[i], sc.x, sc.y, q);
    } else {
#pragma unroll
      for (int i = 0; i < E; ++i) g[(size_t)i * 256] = csub(x[i], q);
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Column pass, two adjacent columns per thread (LN > 4): the same transforms as ntt_col_kernel, but a thread moves its
// points as 8-byte pairs, so that a warp access is two full 128-byte lines of two rows instead of two half lines, and the
// two columns share the twiddles of every stage.  A block owns 2 T2 adjacent columns of one (polynomial, prime).
// ------------------------------------------------------------------------------------------------------------------
template <int LN, bool INV, bool PM>
__global__ void __launch_bounds__(256, 4)
ntt_col2_kernel(NttArgs a) {
  pdl_sync();
  static_assert(LN > 4 && LN <= 8, "paired column pass: 32..256-point columns");
  constexpr int TPC = (1 << LN) / 16;                // threads per column pair
  constexpr int T2 = 256 / TPC;                      // column pairs per block
  constexpr int W = 2 * T2;                          // columns per block = words per tile row
  __shared__ __align__(8) uint32_t sm[8192];
  const uint32_t tid = threadIdx.x, cp = tid % T2, t = tid / T2;
  constexpr uint32_t tiles = 256 / W;
  const uint32_t tr = blockIdx.x / tiles, c0 = (blockIdx.x % tiles) * W;
  // PM: prime-major traversal (the transforms of a prime side by side, primes ascending) instead of memory order (item, slot, prime)
  const uint32_t d1 = PM ? a.nitems * a.U : a.U * a.K, d2 = PM ? a.U : a.K;
  const uint32_t hi = tr / d1, rem = tr % d1, mid = rem / d2, lo = rem % d2;
  const uint32_t item = PM ? mid : hi, slot = PM ? lo : mid, j = PM ? hi : lo;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q;
  const uint2* tw = a.tw + (size_t)j * a.N;
  uint32_t* g = a.data + ((size_t)(item * a.S + slot) * a.K + j) * a.N + c0 + 2 * cp;
  uint32_t x[2][16];
  auto ld2 = [&](const uint32_t* p, int i) { const uint2 v = *reinterpret_cast<const uint2*>(p); x[0][i] = v.x; x[1][i] = v.y; };
  if (!INV) {
#pragma unroll
    for (int i = 0; i < 16; ++i) ld2(g + (size_t)(i * TPC + t) * 256, i);
    phase_a_multi<2, false, LN - 4>(x, tw, 1, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) *reinterpret_cast<uint2*>(sm + (i * TPC + t) * W + 2 * cp) = make_uint2(x[0][i], x[1][i]);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) ld2(sm + (t * 16 + i) * W + 2 * cp, i);
    phase_b_multi<2, LN, false>(x, tw, 1, t, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) *reinterpret_cast<uint2*>(g + (size_t)(t * 16 + i) * 256) = make_uint2(x[0][i], x[1][i]);
  } else {
#pragma unroll
    for (int i = 0; i < 16; ++i) ld2(g + (size_t)(t * 16 + i) * 256, i);
    phase_b_multi<2, LN, true>(x, tw, 1, t, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) *reinterpret_cast<uint2*>(sm + (t * 16 + i) * W + 2 * cp) = make_uint2(x[0][i], x[1][i]);
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) ld2(sm + (i * TPC + t) * W + 2 * cp, i);
    phase_a_multi<2, true, LN - 4>(x, tw, 1, q, q2);
    if (a.scale) {
      const uint2 sc = __ldg(a.scale + j);
#pragma unroll
      for (int i = 0; i < 16; ++i)
        *reinterpret_cast<uint2*>(g + (size_t)(i * TPC + t) * 256) = make_uint2(mul_shoup(x[0][i], sc.x, sc.y, q), mul_shoup(x[1][i], sc.x, sc.y, q));
    } else {                                                       // the constant rides on an operand (fold_scale): canonicalise only
#pragma unroll
      for (int i = 0; i < 16; ++i)
        *reinterpret_cast<uint2*>(g + (size_t)(i * TPC + t) * 256) = make_uint2(csub(x[0][i], q), csub(x[1][i], q));
    }
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Row pass: 256-point transforms over contiguous rows, in place.  A block owns 16 rows, a half-warp one row.  The
// exchange between the two register phases stays inside the half-warp (padded tile: 20 words per 16 points, 336 per
// row, conflict-free for the scalar phase-A and the 128-bit phase-B accesses).
// Forward: rows are the last pass, results leave canonical.  Inverse: rows are the first pass; PW selects what is
// transformed (PwMode) -- the pointwise products are formed in registers from the forward-domain operands.
// FINAL: there is no column pass (N = 256), so the inverse applies the scale here.
// ------------------------------------------------------------------------------------------------------------------
constexpr int ROW_SM = 336;

__device__ __forceinline__ void row_fwd_core(uint32_t (&x)[16], uint32_t* srow, uint32_t t, const uint2* tw, uint32_t base,
                                             uint32_t q, uint32_t q2) {
  phase_a<false, 4>(x, tw, base, q, q2);
#pragma unroll
  for (int i = 0; i < 16; ++i) srow[i * 20 + t] = x[i];
  __syncwarp();
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint4 v = *reinterpret_cast<const uint4*>(srow + t * 20 + 4 * k);
    x[4 * k] = v.x; x[4 * k + 1] = v.y; x[4 * k + 2] = v.z; x[4 * k + 3] = v.w;
  }
  __syncwarp();
  phase_b<8, false>(x, tw, base, t, q, q2);
}
// in: x = the thread's 16 contiguous points (values in [0, 2q)); out: x[i] = point i * 16 + t.  tw = the FORWARD table,
// base = the row's mirrored base (mir_base)
__device__ __forceinline__ void row_inv_core(uint32_t (&x)[16], uint32_t* srow, uint32_t t, const uint2* tw, uint32_t base,
                                             uint32_t q, uint32_t q2) {
  phase_b<8, true>(x, tw, base, t, q, q2);
#pragma unroll
  for (int k = 0; k < 4; ++k)
    *reinterpret_cast<uint4*>(srow + t * 20 + 4 * k) = make_uint4(x[4 * k], x[4 * k + 1], x[4 * k + 2], x[4 * k + 3]);
  __syncwarp();
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = srow[i * 20 + t];
  __syncwarp();
  phase_a<true, 4>(x, tw, base, q, q2);
}

__device__ __forceinline__ void load16(uint32_t (&x)[16], const uint32_t* __restrict__ p) {
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint4 v = *reinterpret_cast<const uint4*>(p + 4 * k);
    x[4 * k] = v.x; x[4 * k + 1] = v.y; x[4 * k + 2] = v.z; x[4 * k + 3] = v.w;
  }
}

__global__ void __launch_bounds__(256)
ntt_row_fwd_kernel(NttArgs a) {
  pdl_sync();
  __shared__ __align__(16) uint32_t sm[16 * ROW_SM];
  const uint32_t tid = threadIdx.x, t = tid & 15, rl = tid >> 4;
  const uint32_t unit = blockIdx.x * 16 + rl;           // row of a transform: ((item * U + slot) * K + j) * N1 + r
  if (unit >= a.units) return;                          // whole half-warps leave together; no block-wide barrier below
  const uint32_t r = unit % a.N1, tr = unit / a.N1;
  const uint32_t item = tr / (a.U * a.K), rem = tr % (a.U * a.K), slot = rem / a.K, j = rem % a.K;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q;
  const uint2* tw = a.tw + (size_t)j * a.N;
  uint32_t* g = a.data + ((size_t)(item * a.S + slot) * a.K + j) * a.N + (size_t)r * 256;
  uint32_t x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = g[i * 16 + t];
  row_fwd_core(x, sm + rl * ROW_SM, t, tw, a.N1 + r, q, q2);
#pragma unroll
  for (int k = 0; k < 4; ++k)
    *reinterpret_cast<uint4*>(g + t * 16 + 4 * k) = make_uint4(canon4(x[4 * k], q, q2), canon4(x[4 * k + 1], q, q2),
                                                                canon4(x[4 * k + 2], q, q2), canon4(x[4 * k + 3], q, q2));
}

template <bool FINAL>
__global__ void __launch_bounds__(256)
ntt_row_inv_kernel(NttArgs a) {
  pdl_sync();
  __shared__ __align__(16) uint32_t sm[16 * ROW_SM];
  const uint32_t tid = threadIdx.x, t = tid & 15, rl = tid >> 4;
  const uint32_t unit = blockIdx.x * 16 + rl;           // row of a transform, as in the forward row pass
  if (unit >= a.units) return;
  const uint32_t r = unit % a.N1, tr = unit / a.N1;
  const uint32_t item = tr / (a.U * a.K), rem = tr % (a.U * a.K), slot = rem / a.K, j = rem % a.K;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q;
  const uint2* tw = a.tw + (size_t)j * a.N;
  uint32_t* g = a.data + ((size_t)(item * a.S + slot) * a.K + j) * a.N + (size_t)r * 256;
  uint32_t x[16];
  load16(x, g + t * 16);
  row_inv_core(x, sm + rl * ROW_SM, t, tw, mir_base(a.N1 + r, a.N1), q, q2);
  if (FINAL) {
    const uint2 sc = __ldg(a.scale + j);
#pragma unroll
    for (int i = 0; i < 16; ++i) g[i * 16 + t] = mul_shoup(x[i], sc.x, sc.y, q);
  } else {
#pragma unroll
    for (int i = 0; i < 16; ++i) g[i * 16 + t] = x[i];
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Fused row pass: the last forward pass, the pointwise products (S3) and the first inverse pass all act on the same
// contiguous 256-point row of one prime, and the forward row pass leaves every thread with 16 contiguous points --
// exactly what the inverse row pass starts from.  So the operands' rows are transformed forward in registers, the
// products formed in registers, and the product rows transformed back, with no HBM round trip in between.
// Operands after the forward rows: the first factor canonical ([0, q)), the second lazy ([0, 4q)): a b < 4 q^2 < 2^62,
// a0 b1 + a1 b0 < 8 q^2 < 2^63 (q < 2^30), so mont_redc's precondition holds and its result is in [0, 2q) -- what the
// inverse butterflies accept.
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void ldrow(uint32_t (&x)[16], const uint32_t* g, uint32_t t) {
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = g[i * 16 + t];
}

constexpr int FUSED_ROWS = 2;   // units (half-warps) per block: one warp; measured 0.435 / 0.424 / 0.422 / 0.418 ms per C5 step for 16 / 8 / 4 / 2
template <int PW, bool FINAL>
__global__ void __launch_bounds__(16 * FUSED_ROWS, 512 / (16 * FUSED_ROWS))
ntt_row_fused_kernel(NttArgs a) {
  pdl_sync();
  __shared__ __align__(16) uint32_t sm[FUSED_ROWS * ROW_SM];
  const uint32_t tid = threadIdx.x, t = tid & 15, rl = tid >> 4;
  // unit = (j * N1 + r) * nitems + item: the half-warps of a block that share (j, r) share every twiddle of both
  // directions (2 KB per row and direction, twice the row itself), so the tables cross L2 -> SM once per (j, r)
  uint32_t unit = blockIdx.x * FUSED_ROWS + rl;
  if (unit >= a.units) return;
  if (a.order) unit = a.units - 1 - unit;                          // start on the primes the forward column pass wrote last
  const uint32_t item = unit % a.nitems, jr = unit / a.nitems;
  const uint32_t r = jr % a.N1, j = jr / a.N1;
  uint32_t* srow = sm + rl * ROW_SM;
  const size_t KN = (size_t)a.K * a.N;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q, qn = __ldg(a.qn + j);
  const uint2* twf = a.tw + (size_t)j * a.N;                       // both directions read the forward table (bf_inv)
  const uint32_t base = a.N1 + r;
  const size_t poff = (size_t)j * a.N + (size_t)r * 256;

  auto fwd = [&](uint32_t (&x)[16]) { row_fwd_core(x, srow, t, twf, base, q, q2); };
  auto fwd_canon = [&](uint32_t (&x)[16]) {
    row_fwd_core(x, srow, t, twf, base, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = canon4(x[i], q, q2);
  };
  auto finish = [&](uint32_t (&x)[16], uint32_t* g) {
    row_inv_core(x, srow, t, twf, mir_base(base, a.N1), q, q2);
    if (FINAL) {                                                   // N = 256: no column pass; the constant rides on an operand
#pragma unroll
      for (int i = 0; i < 16; ++i) g[i * 16 + t] = csub(x[i], q);
    } else {
#pragma unroll
      for (int i = 0; i < 16; ++i) g[i * 16 + t] = x[i];
    }
  };

  if constexpr (PW == PW_POLYMUL) {
    uint32_t* g = a.data + (size_t)item * KN + poff;
    uint32_t x[16], y[16];
    ldrow(x, g, t);
    ldrow(y, a.aux + (size_t)(item / a.aux_group) * KN + poff, t);
    fwd_canon(x);
    fwd(y);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(x[i], y[i], q, qn);
    finish(x, g);
  } else if constexpr (PW == PW_TENSOR) {
    uint32_t* g = a.data + (size_t)item * 4 * KN + poff;       // slots a0, a1, b0, b1 at g + slot * KN
    uint32_t a0[16], a1[16], b0[16], b1[16], x[16];
    ldrow(a0, g, t);
    ldrow(a1, g + KN, t);
    ldrow(b0, g + 2 * KN, t);
    ldrow(b1, g + 3 * KN, t);
    // The exchange inside the first transform orders every lane's operand loads before the first store below.
    fwd_canon(a0);
    fwd_canon(a1);
    fwd(b0);
    fwd(b1);
    // One copy of the inverse transform's code, looped over the three outputs (uniform branches form the products):
    // fully unrolled the kernel is 55 KB of straight-line code and stalled on instruction fetch more than on anything else.
#pragma unroll 1
    for (int op = 0; op < 3; ++op) {
      if (op == 0) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mm(a0[i], b0[i], q, qn);
      } else if (op == 1) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mont_redc((uint64_t)a0[i] * b1[i] + (uint64_t)a1[i] * b0[i], q, qn);
      } else {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mm(a1[i], b1[i], q, qn);
      }
      finish(x, g + (size_t)op * KN);
    }
  } else {   // PW_RELIN: slot 0 = d2 residues after the forward column pass; aux = evk-hat (fully transformed, canonical)
    static_assert(PW == PW_RELIN, "fused row pass: unknown mode");
    uint32_t* g = a.data + (size_t)item * 2 * KN + poff;
    uint32_t d[16], e0[16], e1[16], x[16];
    ldrow(d, g, t);
    load16(e0, a.aux + poff + t * 16);
    load16(e1, a.aux + KN + poff + t * 16);
    fwd_canon(d);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(d[i], e0[i], q, qn);
    finish(x, g);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(d[i], e1[i], q, qn);
    finish(x, g + KN);
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Whole transform in one kernel, N = 2^12 and 2^13 (north_star: "one fused kernel for N <= 2^13"; the paper's reason for two
// passes is only that one block's shared memory cannot hold the polynomial at n >= 2^16).  One block per
// (item, prime) of N / 16 threads keeps the prime-polynomial on chip: column phase (16- or 32-point transforms at stride
// 256, in registers), transposition through a shared-memory tile, row phase (row_fwd_core), the pointwise products in
// registers, and the same backwards -- forward transforms, S3 and inverse transforms with ONE read of the operands and ONE
// write of the results (three words per point and product instead of nine in the three-pass plan).
// The tile keeps rows at a stride of 336 words, so a row's region doubles as the exchange scratch of its row transform.
// ------------------------------------------------------------------------------------------------------------------
constexpr int WROW = ROW_SM;

// the thread's 16 points of the column phase: g[N] (global) -> registers.  All operands of a block are loaded before the first
// transform starts, so that their latency is paid once.
template <int LN1>
__device__ __forceinline__ void whole_load(uint32_t (&x)[16], const uint32_t* __restrict__ g, uint32_t tid) {
  constexpr int TPC = (1 << LN1) / 16;                             // threads per column
  const uint32_t cc = tid & 255, tc = tid >> 8;
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = g[(i * TPC + tc) * 256 + cc];
}
// registers (whole_load) -> registers: thread (r = tid / 16, t = tid % 16) ends with 16 contiguous points of row r, in [0, 4q)
template <int LN1>
__device__ __forceinline__ void whole_fwd(uint32_t (&x)[16], uint32_t* tile, uint32_t tid, const uint2* __restrict__ tw,
                                          uint32_t q, uint32_t q2) {
  static_assert(LN1 == 4 || LN1 == 5, "whole transform: N = 2^12 or 2^13");
  constexpr int TPC = (1 << LN1) / 16;
  const uint32_t cc = tid & 255, tc = tid >> 8, r = tid >> 4, t = tid & 15;
  if constexpr (LN1 == 4) {
    phase_b<4, false>(x, tw, 1, 0, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) tile[i * WROW + cc] = x[i];
  } else {
    phase_a<false, 1>(x, tw, 1, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) tile[(i * TPC + tc) * WROW + cc] = x[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = tile[(tc * 16 + i) * WROW + cc];
    phase_b<5, false>(x, tw, 1, tc, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) tile[(tc * 16 + i) * WROW + cc] = x[i];   // the positions this thread has just read
  }
  __syncthreads();
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = tile[r * WROW + i * 16 + t];
  __syncwarp();                                                    // the row is in registers before its region turns into scratch
  row_fwd_core(x, tile + r * WROW, t, tw, (1u << LN1) + r, q, q2);
  __syncthreads();                                                 // the tile is free for the next operand
}
// registers (16 contiguous points of row r, [0, 2q)) -> g[N] (global), canonical (the final constant rides on an operand)
template <int LN1>
__device__ __forceinline__ void whole_inv(uint32_t (&x)[16], uint32_t* __restrict__ g, uint32_t* tile, uint32_t tid,
                                          const uint2* __restrict__ tw, uint32_t q, uint32_t q2) {
  constexpr int TPC = (1 << LN1) / 16;
  const uint32_t cc = tid & 255, tc = tid >> 8, r = tid >> 4, t = tid & 15;
  row_inv_core(x, tile + r * WROW, t, tw, mir_base((1u << LN1) + r, 1u << LN1), q, q2);   // x[i] = point i * 16 + t of row r
#pragma unroll
  for (int i = 0; i < 16; ++i) tile[r * WROW + i * 16 + t] = x[i];
  __syncthreads();
  if constexpr (LN1 == 4) {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = tile[i * WROW + cc];
    phase_b<4, true>(x, tw, 1, 0, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) g[i * 256 + cc] = csub(x[i], q);
  } else {
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = tile[(tc * 16 + i) * WROW + cc];
    phase_b<5, true>(x, tw, 1, tc, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) tile[(tc * 16 + i) * WROW + cc] = x[i];
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = tile[(i * TPC + tc) * WROW + cc];
    phase_a<true, 1>(x, tw, 1, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) g[(i * TPC + tc) * 256 + cc] = csub(x[i], q);
  }
  __syncthreads();                                                 // the tile is free for the next result
}

template <int PW, int LN1>
// blocks per SM at N = 2^12: two with four operand arrays in registers; the plain product (two arrays) takes three -- measured
// 3.39 -> 3.30 ms per call at logQ = 1240 with 68 bytes of spills, four blocks (64 registers, 190 bytes of spills) 3.56 ms
#ifndef WHOLE_PM_MINB
#define WHOLE_PM_MINB 3
#endif
__global__ void __launch_bounds__(16 << LN1, LN1 == 4 ? (PW == PW_POLYMUL ? WHOLE_PM_MINB : 2) : 1)
ntt_whole_kernel(NttArgs a) {
  pdl_sync();
  extern __shared__ __align__(16) uint32_t tile[];                 // [N / 256][WROW]
  const uint32_t tid = threadIdx.x;
  const uint32_t item = blockIdx.x % a.nitems, j = blockIdx.x / a.nitems;   // the items of a prime side by side: its tables stay in L2
  const size_t KN = (size_t)a.K * a.N, poff = (size_t)j * a.N;
  const uint32_t q = __ldg(a.q + j), q2 = 2 * q, qn = __ldg(a.qn + j);
  const uint2* twf = a.tw + (size_t)j * a.N;
  const uint2* twi = twf;                                         // both directions read the forward table (bf_inv)
  if constexpr (PW == PW_POLYMUL) {
    uint32_t* g = a.data + (size_t)item * KN + poff;
    uint32_t x[16], y[16];
    whole_load<LN1>(x, g, tid);
    whole_load<LN1>(y, a.aux + (size_t)(item / a.aux_group) * KN + poff, tid);
    whole_fwd<LN1>(x, tile, tid, twf, q, q2);
    whole_fwd<LN1>(y, tile, tid, twf, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(canon4(x[i], q, q2), y[i], q, qn);
    whole_inv<LN1>(x, g, tile, tid, twi, q, q2);
  } else if constexpr (PW == PW_TENSOR) {
    uint32_t* g = a.data + (size_t)item * 4 * KN + poff;           // slots a0, a1, b0, b1 at g + slot * KN
    uint32_t a0[16], a1[16], b0[16], b1[16], x[16];
    whole_load<LN1>(a0, g, tid);
    whole_load<LN1>(a1, g + KN, tid);
    whole_load<LN1>(b0, g + 2 * KN, tid);
    whole_load<LN1>(b1, g + 3 * KN, tid);
    whole_fwd<LN1>(a0, tile, tid, twf, q, q2);
    whole_fwd<LN1>(a1, tile, tid, twf, q, q2);
    whole_fwd<LN1>(b0, tile, tid, twf, q, q2);
    whole_fwd<LN1>(b1, tile, tid, twf, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) { a0[i] = canon4(a0[i], q, q2); a1[i] = canon4(a1[i], q, q2); }
    // every thread of the block has read all four operands (the barrier at the end of the last whole_fwd): slots 0..2 may go
#pragma unroll 1
    for (int op = 0; op < 3; ++op) {
      if (op == 0) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mm(a0[i], b0[i], q, qn);
      } else if (op == 1) {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mont_redc((uint64_t)a0[i] * b1[i] + (uint64_t)a1[i] * b0[i], q, qn);
      } else {
#pragma unroll
        for (int i = 0; i < 16; ++i) x[i] = mm(a1[i], b1[i], q, qn);
      }
      whole_inv<LN1>(x, g + (size_t)op * KN, tile, tid, twi, q, q2);
    }
  } else {   // PW_RELIN: slot 0 = d2 residues; aux = the key, fully transformed and canonical (same point order as whole_fwd leaves)
    static_assert(PW == PW_RELIN, "whole transform: unknown mode");
    uint32_t* g = a.data + (size_t)item * 2 * KN + poff;
    const uint32_t r = tid >> 4, t = tid & 15;
    uint32_t d[16], e0[16], e1[16], x[16];
    whole_load<LN1>(d, g, tid);
    load16(e0, a.aux + poff + (size_t)r * 256 + t * 16);
    load16(e1, a.aux + KN + poff + (size_t)r * 256 + t * 16);
    whole_fwd<LN1>(d, tile, tid, twf, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) d[i] = canon4(d[i], q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(d[i], e0[i], q, qn);
    whole_inv<LN1>(x, g, tile, tid, twi, q, q2);
#pragma unroll
    for (int i = 0; i < 16; ++i) x[i] = mm(d[i], e1[i], q, qn);
    whole_inv<LN1>(x, g + KN, tile, tid, twi, q, q2);
  }
}

// ------------------------------------------------------------------------------------------------------------------
// Calibration of the roofline the NTT kernels are held against ("calibrate the integer peak in the same
// run with a register-only microbenchmark of the actual mix").  MODE 0: the forward butterfly itself (bf_fwd: one
// IMAD.HI, two IMAD, three adds / min) on 16 registers per thread with register-resident twiddles, no memory traffic;
// MODE 1: mad.lo.u32 alone; MODE 2: mul.hi.u32 alone.  Measured on B200: 32-bit multiply-add issues at 64 lanes per
// clock per SM, multiply-high at 32, add / min at 128 on another pipe -- so a butterfly costs 4 + 2 + 2 = 8 cycles of
// the multiplier pipe per warp and the pipe, not the issue slots or HBM, bounds the NTT arithmetic.
// ------------------------------------------------------------------------------------------------------------------
template <int MODE>
__global__ void __launch_bounds__(256)
int_peak_kernel(uint32_t* out, uint32_t q, uint2 w0, uint2 w1, uint32_t rounds) {
  uint32_t x[16];
#pragma unroll
  for (int i = 0; i < 16; ++i) x[i] = (threadIdx.x * 16 + i) * 2654435761u % q;
  const uint32_t q2 = 2 * q;
  for (uint32_t r = 0; r < rounds; ++r) {
    if (MODE == 0) {
#pragma unroll
      for (int h = 8; h >= 1; h >>= 1)
#pragma unroll
        for (int i = 0; i < 16; ++i)
          if (!(i & h)) bf_fwd(x[i], x[i + h], (i & 1) ? w1 : w0, q, q2);
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k)
#pragma unroll
        for (int i = 0; i < 16; ++i) {
          if (MODE == 1) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x[i]) : "r"(w0.x), "r"(w1.x));
          else asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(x[i]) : "r"(w0.y));
        }
    }
  }
  uint32_t acc = 0;
#pragma unroll
  for (int i = 0; i < 16; ++i) acc ^= x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = acc;
}

// ops per second of MODE on the whole device: 8 blocks of 256 threads per SM, `rounds` chosen for a few milliseconds
cudaError_t measure_int_peak(Context* c, int mode, double* per_s, cudaStream_t s) {
  const uint32_t q = c->h_q[0], rounds = 1024;
  const uint32_t w = c->h_psi[0];
  const uint2 w0 = make_uint2(w, (uint32_t)(((uint64_t)w << 32) / q)), w1 = make_uint2(q - w, (uint32_t)(((uint64_t)(q - w) << 32) / q));
  const uint32_t blocks = 8 * (uint32_t)c->n_sm;
  uint32_t* d = nullptr;
  cudaError_t e = cudaMalloc(&d, (size_t)blocks * 256 * 4);
  if (e != cudaSuccess) return e;
  cudaEvent_t e0, e1;
  cudaEventCreate(&e0); cudaEventCreate(&e1);
  float best = 1e30f;
  for (int rep = 0; rep < 4; ++rep) {                              // first repetition is the warm-up
    cudaEventRecord(e0, s);
    if (mode == 0) int_peak_kernel<0><<<blocks, 256, 0, s>>>(d, q, w0, w1, rounds);
    else if (mode == 1) int_peak_kernel<1><<<blocks, 256, 0, s>>>(d, q, w0, w1, rounds);
    else int_peak_kernel<2><<<blocks, 256, 0, s>>>(d, q, w0, w1, rounds);
    cudaEventRecord(e1, s);
    e = cudaEventSynchronize(e1);
    if (e != cudaSuccess) break;
    float ms = 0;
    cudaEventElapsedTime(&ms, e0, e1);
    if (rep > 0 && ms < best) best = ms;
  }
  cudaEventDestroy(e0); cudaEventDestroy(e1);
  cudaFree(d);
  if (e != cudaSuccess) return e;
  const double per_thread = mode == 0 ? 32.0 : 64.0;               // butterflies resp. instructions per thread and round
  *per_s = per_thread * rounds * 256.0 * blocks / (best * 1e-3);
  return cudaSuccess;
}

// ------------------------------------------------------------------------------------------------------------------
// The inverse transform of a product ends with a per-prime constant (N^-1 (M/q_j)^-1 2^32: the transform's own scale, the
// CRT's y_i, the Montgomery factor of the pointwise product).  It is folded into an OPERAND instead (the transforms are
// linear): the decompose of the second factor uses a constant image that carries it (ctx.cu), and a key (evk-hat, rotation
// keys) is multiplied by it once, here, when it is installed.  The inverse column pass then only canonicalises.
// ------------------------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256)
scale_rows_kernel(uint32_t* __restrict__ data, const uint2* __restrict__ scale, const uint32_t* __restrict__ qtab, uint32_t N, uint32_t K) {
  const size_t idx = (size_t)blockIdx.x * 256 + threadIdx.x;      // over [npoly][K][N]
  const uint32_t j = (uint32_t)((idx / N) % K);
  const uint2 sc = __ldg(scale + j);
  data[idx] = mul_shoup(data[idx], sc.x, sc.y, __ldg(qtab + j));
}
cudaError_t launch_scale_rows(Context* c, uint32_t* d_res, uint32_t npoly, uint32_t K, const uint2* d_scale, cudaStream_t s) {
  LaunchTimer lt(c, KC_NTT_FWD, s);
  scale_rows_kernel<<<(uint32_t)((size_t)npoly * K * c->N / 256), 256, 0, s>>>(d_res, d_scale, c->d_q, c->N, K);
  return cudaGetLastError();
}

// ---- launchers ------------------------------------------------------------------------------------------------------
template <bool INV>
static cudaError_t launch_col(Context* c, const NttArgs& a, uint32_t ntr, cudaStream_t s) {
  const uint32_t ln1 = c->logN - 8;
  LaunchTimer lt(c, INV ? KC_NTT_INV : KC_NTT_FWD, s);
  cudaError_t e = cudaSuccess;
#define COL_CASE(LN)                                                                           \
  case LN: {                                                                                   \
    constexpr int TPC = (1 << LN) / ((LN) < 4 ? (1 << (LN)) : 16);                             \
    e = launch_pdl(ntt_col_kernel<LN, INV>, ntr * TPC, 256, 0, s, a);                          \
    break;                                                                                     \
  }
#define COL2_CASE(LN)                                                                          \
  case LN: {                                                                                   \
    constexpr int TPC = (1 << LN) / 16;                                                        \
    e = a.order ? launch_pdl(ntt_col2_kernel<LN, INV, true>, ntr * (256 / (2 * (256 / TPC))), 256, 0, s, a)    \
                : launch_pdl(ntt_col2_kernel<LN, INV, false>, ntr * (256 / (2 * (256 / TPC))), 256, 0, s, a);  \
    break;                                                                                     \
  }
  switch (ln1) {   // blocks per transform = 256 / T = TPC (single columns) or TPC / 2 (column pairs)
    COL_CASE(1) COL_CASE(2) COL_CASE(3) COL_CASE(4) COL2_CASE(5) COL2_CASE(6) COL2_CASE(7) COL2_CASE(8)
    default: return cudaErrorInvalidValue;
  }
#undef COL_CASE
#undef COL2_CASE
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_ntt_fwd(Context* c, uint32_t* d_res, uint32_t nitems, uint32_t S, uint32_t U, uint32_t K, cudaStream_t s) {
  if (!nitems || !U) return cudaSuccess;
  NttArgs a;
  a.data = d_res; a.aux = nullptr; a.tw = c->d_tw_fwd; a.q = c->d_q; a.qn = c->d_qinv_neg; a.scale = nullptr;
  a.N = c->N; a.K = K; a.N1 = c->N / 256; a.S = S; a.U = U; a.nitems = nitems; a.aux_group = 1; a.order = 0;
  const uint32_t ntr = nitems * U * K;
  a.units = ntr * a.N1;
  if (c->logN > 8) {
    cudaError_t e = launch_col<false>(c, a, ntr, s);
    if (e != cudaSuccess) return e;
  }
  LaunchTimer lt(c, KC_NTT_FWD, s);
  const cudaError_t e = launch_pdl(ntt_row_fwd_kernel, (a.units + 15) / 16, 256, 0, s, a);
  return e != cudaSuccess ? e : cudaGetLastError();
}

cudaError_t launch_ntt_inv(Context* c, uint32_t* d_res, uint32_t nitems, uint32_t S, uint32_t U, uint32_t K,
                           const uint2* d_scale, cudaStream_t s) {
  if (!nitems || !U) return cudaSuccess;
  NttArgs a;
  a.data = d_res; a.aux = nullptr; a.tw = c->d_tw_fwd; a.q = c->d_q; a.qn = c->d_qinv_neg; a.scale = d_scale;
  a.N = c->N; a.K = K; a.N1 = c->N / 256; a.S = S; a.U = U; a.nitems = nitems; a.aux_group = 1; a.order = 0;
  const bool fin = c->logN == 8;
  a.units = nitems * U * K * a.N1;
  const uint32_t blocks = (a.units + 15) / 16;
  {
    LaunchTimer lt(c, KC_NTT_INV, s);
    cudaError_t e;
    if (fin) e = launch_pdl(ntt_row_inv_kernel<true>, blocks, 256, 0, s, a);
    else e = launch_pdl(ntt_row_inv_kernel<false>, blocks, 256, 0, s, a);
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (!fin) return launch_col<true>(c, a, nitems * U * K, s);
  return cudaSuccess;
}

// S2 + S3 + S4 of a product in three launches (four for PW_POLYMUL): forward column pass over the operand slots, the
// fused row pass, inverse column pass over the result slots.
cudaError_t launch_ntt_product(Context* c, uint32_t* d_res, uint32_t* d_aux, uint32_t nitems, uint32_t K, int pw_mode,
                               cudaStream_t s, uint32_t aux_group) {
  if (!nitems) return cudaSuccess;
  uint32_t S, Uin, Uout;
  switch (pw_mode) {
    case PW_POLYMUL: S = 1; Uin = 1; Uout = 1; break;
    case PW_TENSOR: S = 4; Uin = 4; Uout = 3; break;
    case PW_RELIN: S = 2; Uin = 1; Uout = 2; break;
    default: return cudaErrorInvalidValue;
  }
  NttArgs a;
  a.data = d_res; a.aux = nullptr; a.tw = c->d_tw_fwd; a.q = c->d_q; a.qn = c->d_qinv_neg; a.scale = nullptr;
  a.N = c->N; a.K = K; a.N1 = c->N / 256; a.S = S; a.U = Uin; a.units = 0; a.nitems = nitems; a.aux_group = aux_group ? aux_group : 1;
  // product path: forward columns prime-major ascending, fused rows descending, inverse columns prime-major ascending (the
  // fused rows then finish on prime 0) -- each pass starts on the tail of the previous one's output
  const uint32_t l2o = NTT_L2_ORDER;
  a.order = l2o ? 1 : 0;
  const bool fin = c->logN == 8;
  cudaError_t e;
  // the whole product in one launch (ntt_whole_kernel): measured 5-9 % faster than the three passes at N = 2^12, 8-13 % slower
  // at N = 2^13 (512-thread blocks, one or two per SM: the block-wide barriers of the transpositions are not hidden), so
  // N = 2^13 takes it only on request (fhe_debug_force_pipeline(ctx, 2))
  if ((c->logN == 12 && c->force_pipe != 1) || (c->logN == 13 && c->force_pipe == 2)) {
    a.aux = d_aux; a.scale = nullptr; a.U = Uout;
    a.units = nitems * K;
    const uint32_t threads = c->N / 16;
    const size_t smem = (size_t)(c->N / 256) * WROW * sizeof(uint32_t);
    LaunchTimer lt(c, KC_POINTWISE, s);
#define WHOLE_CASE(PW)                                                                                      \
  case PW:                                                                                                  \
    e = c->logN == 12 ? launch_pdl(ntt_whole_kernel<PW, 4>, a.units, threads, smem, s, a)                   \
                      : launch_pdl(ntt_whole_kernel<PW, 5>, a.units, threads, smem, s, a);                  \
    break;
    switch (pw_mode) { WHOLE_CASE(PW_POLYMUL) WHOLE_CASE(PW_TENSOR) WHOLE_CASE(PW_RELIN) default: e = cudaErrorInvalidValue; }
#undef WHOLE_CASE
    return e != cudaSuccess ? e : cudaGetLastError();
  }
  if (!fin) {
    if ((e = launch_col<false>(c, a, nitems * Uin * K, s)) != cudaSuccess) return e;
    if (pw_mode == PW_POLYMUL) {
      a.data = d_aux; a.nitems = (nitems + a.aux_group - 1) / a.aux_group;   // the shared operands: their own item count
      if ((e = launch_col<false>(c, a, a.nitems * K, s)) != cudaSuccess) return e;
      a.data = d_res; a.nitems = nitems;
    }
  }
  a.aux = d_aux; a.scale = nullptr; a.U = Uout;
  a.units = nitems * K * a.N1;
  const uint32_t blocks = (a.units + FUSED_ROWS - 1) / FUSED_ROWS;
  {
    LaunchTimer lt(c, KC_POINTWISE, s);
#define FUSED_CASE(PW)                                                                 \
  case PW:                                                                             \
    if (fin) e = launch_pdl(ntt_row_fused_kernel<PW, true>, blocks, 16 * FUSED_ROWS, 0, s, a);     \
    else e = launch_pdl(ntt_row_fused_kernel<PW, false>, blocks, 16 * FUSED_ROWS, 0, s, a);        \
    break;
    switch (pw_mode) { FUSED_CASE(PW_POLYMUL) FUSED_CASE(PW_TENSOR) FUSED_CASE(PW_RELIN) default: e = cudaErrorInvalidValue; }
#undef FUSED_CASE
    if (e == cudaSuccess) e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  if (!fin) return launch_col<true>(c, a, nitems * Uout * K, s);
  return cudaSuccess;
}

}  // namespace fhe
