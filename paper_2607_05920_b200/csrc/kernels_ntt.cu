// kernels_ntt.cu -- S2/S4 negacyclic NTT passes, S3 pointwise products.
//
// NTT formulation (Eq. 8-9): merged-psi Cooley-Tukey forward / Gentleman-Sande inverse
// (PAPER.md:352, 358); the psi^j "twist" of PAPER.md:346-350 is folded into the butterfly twiddles, so no separate
// twist pass exists.  tw_fwd[k] = psi^bitrev_logN(k), tw_inv[k] = psi^-bitrev_logN(k).  Forward stage with m
// groups (m = 1, 2, .., N/2) pairs j and j + t, t = N/(2m), twiddle index m + (j >> log2(2t)).  Output of the
// forward transform is in bit-reversed order; the pointwise products do not care, the inverse undoes it.
//
// Two-pass split for N = N1 * N2 (the paper's "column NTT, twiddle, row NTT"): with the merged
// twiddles the first log2 N1 stages act on columns (stride N2) with the N1-point table prefix, the last log2 N2
// stages act on contiguous rows r with table indices (N1 + r) m' + i'.  Both are one "local transform with base":
// twiddle index = base * m' + i' (base = 1 for columns / whole transforms, N1 + r for row r), so there is no separate
// twiddle-multiplication pass and no transpose.
#include "fhe_internal.cuh"

namespace fhe {

// ------------------------------------------------------------------------------------------------------------------
// S2 / S4: local transform of n = 2^ln points with twiddle index base * m' + i', T transforms per block, radix-2
// stages in shared memory (first correct version; the register-tiled version replaces it where it matters).
// Layout of the tile in shared memory = flat load order f:
//   column tile (COL): f = e * T + tt  <->  global  e * N2 + col0 + tt
//   row tile    (ROW): f = tt * n + e  <->  global (row0 + tt) * n + e         (also the whole-transform case, T = 1)
// ------------------------------------------------------------------------------------------------------------------
template <bool INV, bool COL>
__global__ void __launch_bounds__(256)
ntt_tile_kernel(uint32_t* __restrict__ data, const uint2* __restrict__ tw_all, const uint32_t* __restrict__ qarr,
                const uint2* __restrict__ scale, uint32_t N, uint32_t K, uint32_t ln, uint32_t lT, uint32_t N1,
                uint32_t tiles_per_tr, bool apply_scale) {
  extern __shared__ uint32_t sm[];
  const uint32_t n = 1u << ln, T = 1u << lT;
  const uint32_t tile = blockIdx.x % tiles_per_tr;
  const uint32_t pp = blockIdx.x / tiles_per_tr;          // poly * K + prime
  const uint32_t j = pp % K;
  const uint32_t q = __ldg(qarr + j);
  const uint2* tw = tw_all + (size_t)j * N;
  uint32_t* g = data + (size_t)pp * N;
  const uint32_t total = n * T;
  const uint32_t N2 = COL ? (N / n) : n;

  for (uint32_t f = threadIdx.x; f < total; f += blockDim.x) {
    size_t off = COL ? ((size_t)(f >> lT) * N2 + tile * T + (f & (T - 1))) : ((size_t)tile * total + f);
    sm[f] = g[off];
  }
  __syncthreads();

  const uint32_t half = total >> 1;   // butterflies per stage in the tile
  for (uint32_t st = 0; st < ln; ++st) {
    const uint32_t sp = INV ? (ln - 1 - st) : st;     // stage parameter: m' = 2^sp
    const uint32_t ltl = ln - 1 - sp;                 // log2 of the local butterfly stride
    const uint32_t tl = 1u << ltl;
    for (uint32_t x = threadIdx.x; x < half; x += blockDim.x) {
      uint32_t tt, b;
      if (COL) { tt = x & (T - 1); b = x >> lT; }
      else     { b = x & ((n >> 1) - 1); tt = x >> (ln - 1); }
      const uint32_t ip = b >> ltl, jj = b & (tl - 1);
      const uint32_t e0 = (ip << (ltl + 1)) + jj, e1 = e0 + tl;
      const uint32_t base = COL ? 1u : (N1 + tile * T + tt);   // N1 == 0 and tile == 0 for whole transforms -> +1 below
      const uint32_t widx = (COL || N1) ? ((base << sp) + ip) : ((1u << sp) + ip);
      const uint2 w = __ldg(tw + widx);
      const uint32_t i0 = COL ? (e0 * T + tt) : (tt * n + e0);
      const uint32_t i1 = COL ? (e1 * T + tt) : (tt * n + e1);
      const uint32_t U = sm[i0], V = sm[i1];
      if (!INV) {
        const uint32_t Vw = mul_shoup(V, w.x, w.y, q);
        sm[i0] = csub(U + Vw, q);
        const uint32_t d = U - Vw;
        sm[i1] = min(d, d + q);
      } else {
        sm[i0] = csub(U + V, q);
        const uint32_t d = U - V;
        sm[i1] = mul_shoup(min(d, d + q), w.x, w.y, q);
      }
    }
    __syncthreads();
  }
  uint2 sc = make_uint2(0, 0);
  if (apply_scale) sc = __ldg(scale + j);
  for (uint32_t f = threadIdx.x; f < total; f += blockDim.x) {
    size_t off = COL ? ((size_t)(f >> lT) * N2 + tile * T + (f & (T - 1))) : ((size_t)tile * total + f);
    uint32_t v = sm[f];
    if (apply_scale) v = mul_shoup(v, sc.x, sc.y, q);
    g[off] = v;
  }
}

cudaError_t launch_ntt(Context* c, uint32_t* d_res, uint32_t npoly, uint32_t K, bool inverse, const uint2* d_scale,
                       cudaStream_t s) {
  if (npoly == 0) return cudaSuccess;
  const uint32_t N = c->N, logN = c->logN;
  const uint32_t ntr = npoly * K;
  if (logN <= 13) {   // one kernel: the whole transform in shared memory
    size_t smem = (size_t)N * 4;
    LaunchTimer lt(c, inverse ? KC_NTT_INV : KC_NTT_FWD, s);
    if (!inverse)
      ntt_tile_kernel<false, false><<<ntr, 256, smem, s>>>(d_res, c->d_tw_fwd, c->d_q, d_scale, N, K, logN, 0, 0, 1, false);
    else
      ntt_tile_kernel<true, false><<<ntr, 256, smem, s>>>(d_res, c->d_tw_inv, c->d_q, d_scale, N, K, logN, 0, 0, 1, true);
    return cudaGetLastError();
  }
  const uint32_t ln2 = 8, ln1 = logN - ln2, N1 = 1u << ln1, N2 = 1u << ln2;
  const uint32_t lTc = 5, lTr = 4;                       // 32 columns / 16 rows per block
  const uint32_t col_tiles = N2 >> lTc, row_tiles = N1 >> lTr;
  const size_t smem_col = (size_t)N1 * (1u << lTc) * 4, smem_row = (size_t)N2 * (1u << lTr) * 4;
  if (!inverse) {
    { LaunchTimer lt(c, KC_NTT_FWD, s);
    ntt_tile_kernel<false, true><<<ntr * col_tiles, 256, smem_col, s>>>(d_res, c->d_tw_fwd, c->d_q, d_scale, N, K, ln1, lTc, N1, col_tiles, false); }
    { LaunchTimer lt(c, KC_NTT_FWD, s);
    ntt_tile_kernel<false, false><<<ntr * row_tiles, 256, smem_row, s>>>(d_res, c->d_tw_fwd, c->d_q, d_scale, N, K, ln2, lTr, N1, row_tiles, false); }
  } else {
    { LaunchTimer lt(c, KC_NTT_INV, s);
    ntt_tile_kernel<true, false><<<ntr * row_tiles, 256, smem_row, s>>>(d_res, c->d_tw_inv, c->d_q, d_scale, N, K, ln2, lTr, N1, row_tiles, false); }
    LaunchTimer lt(c, KC_NTT_INV, s);
    ntt_tile_kernel<true, true><<<ntr * col_tiles, 256, smem_col, s>>>(d_res, c->d_tw_inv, c->d_q, d_scale, N, K, ln1, lTc, N1, col_tiles, true);
  }
  return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------------------------
// S3: pointwise products in the NTT domain (Eq. 7), Montgomery form: each product carries 2^-32,
// removed by the inverse transform's final constant.
// ------------------------------------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t mm(uint32_t a, uint32_t b, uint32_t q, uint32_t qn) {
  return mont_redc((uint64_t)a * b, q, qn);
}

__global__ void __launch_bounds__(256)
pw_polymul_kernel(uint32_t* __restrict__ a, const uint32_t* __restrict__ b, uint32_t N4, uint32_t K,
                  const uint32_t* __restrict__ qarr, const uint32_t* __restrict__ qnarr, uint32_t gx) {
  const uint32_t pp = blockIdx.x / gx, j = pp % K, cx = blockIdx.x % gx;
  const uint32_t q = __ldg(qarr + j), qn = __ldg(qnarr + j);
  uint4* pa = reinterpret_cast<uint4*>(a) + (size_t)pp * N4;
  const uint4* pb = reinterpret_cast<const uint4*>(b) + (size_t)pp * N4;
  for (uint32_t i = cx * blockDim.x + threadIdx.x; i < N4; i += gx * blockDim.x) {
    uint4 x = pa[i], y = pb[i];
    x.x = mm(x.x, y.x, q, qn); x.y = mm(x.y, y.y, q, qn); x.z = mm(x.z, y.z, q, qn); x.w = mm(x.w, y.w, q, qn);
    pa[i] = x;
  }
}

// r: [batch][4][K][N] = (a0, a1, b0, b1) -> slots 0..2 = (a0 b0, a0 b1 + a1 b0, a1 b1)
__global__ void __launch_bounds__(256)
pw_tensor_kernel(uint32_t* __restrict__ r, uint32_t N4, uint32_t K, const uint32_t* __restrict__ qarr,
                 const uint32_t* __restrict__ qnarr, uint32_t gx) {
  const uint32_t pp = blockIdx.x / gx, cx = blockIdx.x % gx, j = pp % K, bi = pp / K;
  const uint32_t q = __ldg(qarr + j), qn = __ldg(qnarr + j);
  const size_t ps = (size_t)K * N4;   // poly stride in uint4
  uint4* base = reinterpret_cast<uint4*>(r) + (size_t)bi * 4 * ps + (size_t)j * N4;
  for (uint32_t i = cx * blockDim.x + threadIdx.x; i < N4; i += gx * blockDim.x) {
    const uint4 a0 = base[i], a1 = base[ps + i], b0 = base[2 * ps + i], b1 = base[3 * ps + i];
    uint4 d0, d1, d2;
#define TP(c)                                                                     \
  d0.c = mm(a0.c, b0.c, q, qn);                                                   \
  d1.c = mont_redc((uint64_t)a0.c * b1.c + (uint64_t)a1.c * b0.c, q, qn);         \
  d2.c = mm(a1.c, b1.c, q, qn);
    TP(x) TP(y) TP(z) TP(w)
#undef TP
    base[i] = d0; base[ps + i] = d1; base[2 * ps + i] = d2;
  }
}

// r: [batch][2][K][N], slot 0 = d2^ -> slot 0 = d2^ * evk_b^, slot 1 = d2^ * evk_a^
__global__ void __launch_bounds__(256)
pw_relin_kernel(uint32_t* __restrict__ r, const uint32_t* __restrict__ evk, uint32_t N4, uint32_t K,
                const uint32_t* __restrict__ qarr, const uint32_t* __restrict__ qnarr, uint32_t gx) {
  const uint32_t pp = blockIdx.x / gx, cx = blockIdx.x % gx, j = pp % K, bi = pp / K;
  const uint32_t q = __ldg(qarr + j), qn = __ldg(qnarr + j);
  const size_t ps = (size_t)K * N4;
  uint4* base = reinterpret_cast<uint4*>(r) + (size_t)bi * 2 * ps + (size_t)j * N4;
  const uint4* eb = reinterpret_cast<const uint4*>(evk) + (size_t)j * N4;
  const uint4* ea = eb + ps;
  for (uint32_t i = cx * blockDim.x + threadIdx.x; i < N4; i += gx * blockDim.x) {
    const uint4 d = base[i], b = eb[i], a = ea[i];
    uint4 xb, xa;
    xb.x = mm(d.x, b.x, q, qn); xb.y = mm(d.y, b.y, q, qn); xb.z = mm(d.z, b.z, q, qn); xb.w = mm(d.w, b.w, q, qn);
    xa.x = mm(d.x, a.x, q, qn); xa.y = mm(d.y, a.y, q, qn); xa.z = mm(d.z, a.z, q, qn); xa.w = mm(d.w, a.w, q, qn);
    base[i] = xb; base[ps + i] = xa;
  }
}

static inline uint32_t pw_grid_x(uint32_t N4) { return (N4 + 255) / 256 > 16 ? 16 : (N4 + 255) / 256; }

cudaError_t launch_pw_polymul(Context* c, uint32_t* d_a, const uint32_t* d_b, uint32_t batch, uint32_t K,
                              cudaStream_t s) {
  if (!batch) return cudaSuccess;
  const uint32_t N4 = c->N / 4;
  LaunchTimer lt(c, KC_POINTWISE, s);
  pw_polymul_kernel<<<pw_grid_x(N4) * batch * K, 256, 0, s>>>(d_a, d_b, N4, K, c->d_q, c->d_qinv_neg, pw_grid_x(N4));
  return cudaGetLastError();
}
cudaError_t launch_pw_tensor(Context* c, uint32_t* d_r, uint32_t batch, uint32_t K, cudaStream_t s) {
  if (!batch) return cudaSuccess;
  const uint32_t N4 = c->N / 4;
  LaunchTimer lt(c, KC_POINTWISE, s);
  pw_tensor_kernel<<<pw_grid_x(N4) * batch * K, 256, 0, s>>>(d_r, N4, K, c->d_q, c->d_qinv_neg, pw_grid_x(N4));
  return cudaGetLastError();
}
cudaError_t launch_pw_relin(Context* c, uint32_t* d_r, const uint32_t* d_evk_hat, uint32_t batch, uint32_t K,
                            cudaStream_t s) {
  if (!batch) return cudaSuccess;
  const uint32_t N4 = c->N / 4;
  LaunchTimer lt(c, KC_POINTWISE, s);
  pw_relin_kernel<<<pw_grid_x(N4) * batch * K, 256, 0, s>>>(d_r, d_evk_hat, N4, K, c->d_q, c->d_qinv_neg, pw_grid_x(N4));
  return cudaGetLastError();
}

}  // namespace fhe
