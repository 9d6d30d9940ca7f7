// kernels_decompose.cu -- S1: limb -> RNS decomposition on the tensor cores.
//
// The paper computes r_j = sum_i limb_i * (2^(32 i) mod q_j) mod q_j one coefficient and one prime at a time.  That
// sum is a dense contraction of the coefficient's bytes with a constant matrix, so it runs as one integer GEMM per
// 128-coefficient tile (umma.cuh):
//     T[n][4 j + c] = sum_kb byte_kb(X_n) * byte_c(2^(8 kb) mod q_j)        u8 x u8 -> s32, exact
//     r_j(X_n)      = (T[n][4j] + 2^8 T[n][4j+1] + 2^16 T[n][4j+2] + 2^24 T[n][4j+3]) mod q_j
// The CUDA cores only do the epilogue: recombine the four byte sums (< 2^49) and one word-sized Barrett reduction.
#include "fhe_internal.cuh"
#include "umma.cuh"

namespace fhe {

using namespace umma;

struct DecArgs {
  uint32_t* res; size_t res_poly_stride;
  const uint32_t* limbs; size_t limb_poly_stride;
  const uint8_t* B; size_t chunk_stride;
  const uint2* qmu;
  uint32_t N, Lin, K, KB, mask_bits, nchunks;
};

constexpr uint32_t DEC_GROUP_COLS = DEC_NC * DEC_GROUP_CHUNKS;   // TMEM columns per CTA

__global__ void __launch_bounds__(TILE_M)
decompose_mma_kernel(DecArgs a) {
  extern __shared__ __align__(1024) uint8_t smem[];
  __shared__ MmaPipe pipe;
  __shared__ uint32_t tmem_slot;
  uint8_t* sA = smem;
  uint8_t* sB0 = sA + (size_t)a.KB * TILE_M;
  uint8_t* sB1 = sB0 + (size_t)a.KB * DEC_NC;
  const uint32_t tid = threadIdx.x, warp = tid >> 5;
  const uint32_t tiles = a.N / TILE_M;
  const uint32_t poly = blockIdx.x / tiles;
  const uint32_t n0 = (blockIdx.x % tiles) * TILE_M;

  stage_rows(sA, a.limbs + (size_t)poly * a.limb_poly_stride + n0, a.N, a.Lin, a.KB, a.mask_bits);
  if (tid == 0) mma_pipe_init(&pipe);
  if (warp == 0) tmem_alloc(&tmem_slot, DEC_GROUP_COLS);
  fence_proxy_async();
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = tmem_slot;
  const uint32_t lane_addr = tbase + ((warp * 32u) << 16);
  uint32_t* out = a.res + (size_t)poly * a.res_poly_stride + n0 + tid;

  PipeState st = {{0, 0}, {0, 0}, 0};
  for (uint32_t c0 = 0; c0 < a.nchunks; c0 += DEC_GROUP_CHUNKS) {
    const uint32_t nch = min((uint32_t)DEC_GROUP_CHUNKS, a.nchunks - c0);
    if (warp == 0) {   // lane 0 issues; its warp mates park at the convergence barrier instead of polling beside it
      if (tid == 0) mma_phase(&pipe, st, sA, sB0, sB1, a.KB, DEC_NC, a.B + (size_t)c0 * a.chunk_stride, a.chunk_stride, nch, tbase);
      __syncwarp();
    }
    mbar_wait(&pipe.done, st.done_par);
    st.done_par ^= 1;
    __syncwarp();
    tc_fence_after();
    for (uint32_t cc = 0; cc < nch * DEC_NC; cc += 32) {
      const uint32_t j0 = (c0 * DEC_NC + cc) / 4;
      if (j0 >= a.K) break;
      uint32_t t[32];
      tmem_ld32(lane_addr + cc, t);
#pragma unroll
      for (int e = 0; e < 8; ++e) {
        const uint32_t j = j0 + e;
        if (j < a.K) {
          const uint2 qm = __ldg(a.qmu + j);
          const uint64_t lo = (uint64_t)t[4 * e + 1] * 256u + t[4 * e];
          const uint64_t hi = (uint64_t)t[4 * e + 3] * 256u + t[4 * e + 2];
          out[(size_t)j * a.N] = barrett49(lo + (hi << 16), qm.x, qm.y);
        }
      }
    }
    tc_fence_before();
    __syncthreads();   // every warp has drained its lanes before the next group's MMAs overwrite them
    tc_fence_after();
  }
  if (warp == 0) tmem_dealloc(tbase, DEC_GROUP_COLS);
}

cudaError_t launch_decompose(Context* c, uint32_t* d_res, size_t res_poly_stride, const uint32_t* d_limbs,
                             size_t limb_poly_stride, uint32_t npoly, uint32_t Lin, uint32_t K, uint32_t mask_bits,
                             cudaStream_t s) {
  if (npoly == 0) return cudaSuccess;
  uint32_t eff = Lin;
  if (mask_bits && (mask_bits + 31) / 32 < eff) eff = (mask_bits + 31) / 32;
  DecArgs a;
  a.res = d_res; a.res_poly_stride = res_poly_stride;
  a.limbs = d_limbs; a.limb_poly_stride = limb_poly_stride;
  a.B = c->d_decB; a.chunk_stride = (size_t)c->dec_KBimg * DEC_NC;
  a.qmu = c->d_qmu;
  a.N = c->N; a.Lin = eff; a.K = K; a.mask_bits = mask_bits;
  a.KB = (4 * eff + 31) / 32 * 32;
  a.nchunks = (K + 15) / 16;
  if (a.KB > c->dec_KBimg || K > c->Kmax) return cudaErrorInvalidValue;
  const size_t smem = smem_for_tmem_residency((size_t)a.KB * (TILE_M + 2 * DEC_NC), DEC_GROUP_COLS);
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(decompose_mma_kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    // several CTAs per SM are the latency hiding here: ask for the full shared-memory carveout, not the driver's guess
    e = cudaFuncSetAttribute(decompose_mma_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  LaunchTimer lt(c, KC_DECOMPOSE, s);
  decompose_mma_kernel<<<(c->N / TILE_M) * npoly, TILE_M, smem, s>>>(a);
  return cudaGetLastError();
}

}  // namespace fhe
