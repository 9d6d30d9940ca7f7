// umma.cuh -- sm_100a tensor-core plumbing for the two base conversions of the path (S1 limb -> RNS, S5 RNS -> limb).
//
// Both conversions are dense integer contractions over the bytes of a word-major array:
//     D[n][c] = sum_kb  byte_kb(row n)  *  Bconst[kb][c]            (u8 x u8 -> s32, exact)
// with n = coefficient index (M = 128 rows per CTA), kb = byte index of the input words (limbs resp. residues),
// c = output column (bytes of the per-prime constants resp. byte positions of the reconstructed integer).
// They run on the 5th-generation tensor cores: tcgen05.mma kind::i8, the A operand in tensor memory (written there with
// tcgen05.st), the constant B operand in shared memory in the no-swizzle K-major canonical layout (8 x 16-byte core
// matrices), accumulators in TMEM, read back with tcgen05.ld.  The pipeline built from these pieces is pipe.cuh.
// Everything here is inline PTX; there is no library dependency.
#pragma once
#include <cuda.h>   // CUtensorMap (the type only; the encoder is fetched through the runtime, no libcuda link)
#include <cuda_runtime.h>
#include <cstdint>

namespace fhe {
namespace umma {

constexpr int TILE_M = 128;          // rows (coefficients) per CTA = TMEM lanes = threads
constexpr int KSTEP = 32;            // bytes of the contraction dimension one kind::i8 instruction consumes

// 2-D tensor map over a word matrix [rows][cols] of uint32 (row-major, dense), box [box_rows][box_cols]: the driver's
// encoder, fetched through the runtime (no link against libcuda).  false: no encoder / bad arguments -- callers fall back
// to loads that land in registers.
inline bool make_tensor_map(CUtensorMap* tm, const uint32_t* base, uint64_t rows, uint32_t cols, uint32_t box_rows,
                            uint32_t box_cols = TILE_M) {
  typedef CUresult (*Encode)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                             const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                             CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
  static Encode enc = nullptr;
  static bool tried = false;
  if (!tried) {
    tried = true;
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) == cudaSuccess && qr == cudaDriverEntryPointSuccess)
      enc = (Encode)fn;
    else
      cudaGetLastError();
  }
  if (!enc || box_rows == 0 || box_rows > 256 || box_cols == 0 || box_cols > 256 || rows == 0) return false;
  const cuuint64_t gdim[2] = {cols, rows}, gstride[1] = {(cuuint64_t)cols * 4};
  const cuuint32_t box[2] = {box_cols, box_rows}, estr[2] = {1, 1};
  return enc(tm, CU_TENSOR_MAP_DATA_TYPE_UINT32, 2, (void*)base, gdim, gstride, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
             CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier -------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Blocks until the phase with the given parity has completed.  A wait that does not complete can only mean a programming
// error in this file; it traps (launch failure) instead of hanging the device -- but by wall clock, not by poll count:
// under compute-sanitizer, an ncu replay or time-slicing a correct kernel can poll millions of times.  The timer is read
// once per 2^10 unsuccessful polls (each try_wait suspends the thread until the phase completes or the hint runs out).
constexpr uint64_t MBAR_TIMEOUT_NS = 60ull * 1000 * 1000 * 1000;
// upper bound of one hardware suspension of try_wait: a waiting warp sleeps instead of spending issue slots on polling
constexpr uint32_t MBAR_SUSPEND_HINT_NS = 10u * 1000 * 1000;
__device__ __forceinline__ uint64_t global_ns() {
  uint64_t t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  uint32_t polls = 0;
  uint64_t t0 = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity), "r"(MBAR_SUSPEND_HINT_NS)
        : "memory");
    if (done) break;
    if ((++polls & 0x3FFu) == 0) {
      const uint64_t now = global_ns();
      if (t0 == 0) t0 = now;
      else if (now - t0 > MBAR_TIMEOUT_NS) __trap();
    }
  }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// one 2-D tensor copy global -> shared (TMA): the map's box at (column c0, row c1) of the tensor map, bytes counted on bar
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* tmap, uint32_t c0, uint32_t c1, uint64_t* bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(tmap), "r"(c0), "r"(c1), "r"(smem_u32(bar))
               : "memory");
}
// orders this thread's earlier generic-proxy accesses to shared memory before later async-proxy (TMA) ones
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// ---- bulk copy global -> shared (1-D TMA), completion counted in bytes on an mbarrier -------------------------------------
__device__ __forceinline__ void bulk_g2s(void* smem_dst, const void* gmem_src, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                   smem_u32(smem_dst)),
               "l"(gmem_src), "r"(bytes), "r"(smem_u32(bar))
               : "memory");
}

// ---- TMEM -------------------------------------------------------------------------------------------------------------
// one full warp; ncols a power of two in [32, 512]; the base address lands in *slot (shared memory)
__device__ __forceinline__ void tmem_alloc(uint32_t* slot, uint32_t ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(slot)), "r"(ncols)
               : "memory");
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t base, uint32_t ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(base), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// ---- descriptors --------------------------------------------------------------------------------------------------------
// Shared-memory matrix descriptor, K-major, no swizzle ("interleave"): element (row r, byte kb) of the operand sits at
//   start + (r / 8) * sbo + (kb / 16) * lbo + (r % 8) * 16 + kb % 16.
// Both images used here keep rows dense (sbo = 128), so a row costs 16 bytes per K chunk: [kb/16][row][16].
__device__ __forceinline__ uint64_t smem_desc(uint32_t saddr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
  uint64_t d = 0;
  d |= (uint64_t)((saddr >> 4) & 0x3FFFu);
  d |= (uint64_t)((lbo_bytes >> 4) & 0x3FFFu) << 16;
  d |= (uint64_t)((sbo_bytes >> 4) & 0x3FFFu) << 32;
  d |= (uint64_t)1 << 46;   // descriptor version of sm_100
  return d;                  // base offset 0, layout type 0 (no swizzle)
}
// Instruction descriptor for kind::i8: D = s32, A = B = unsigned 8-bit, both K-major, M = 128, N = ncols (multiple of 16).
__device__ __forceinline__ uint32_t idesc_u8(uint32_t ncols) {
  return (2u << 4) | ((ncols >> 3) << 17) | ((uint32_t)(TILE_M >> 4) << 24);
}
// arrive on `bar` once every MMA issued so far by this thread has finished (also orders them before the arrive)
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

}  // namespace umma
}  // namespace fhe
