// umma.cuh -- sm_100a tensor-core plumbing for the two base conversions of the path (S1 limb -> RNS, S5 RNS -> limb).
//
// Both conversions are dense integer contractions over the bytes of a word-major array:
//     D[n][c] = sum_kb  byte_kb(row n)  *  Bconst[kb][c]            (u8 x u8 -> s32, exact)
// with n = coefficient index (M = 128 rows per CTA), kb = byte index of the input words (limbs resp. residues),
// c = output column (bytes of the per-prime constants resp. byte positions of the reconstructed integer).
// They run on the 5th-generation tensor cores: tcgen05.mma kind::i8, operands in shared memory in the no-swizzle
// K-major canonical layout (8 x 16-byte core matrices), accumulators in TMEM, read back with tcgen05.ld.
// Everything here is inline PTX; there is no library dependency.
#pragma once
#include <cuda_runtime.h>
#include <cstdint>

namespace fhe {
namespace umma {

constexpr int TILE_M = 128;          // rows (coefficients) per CTA = TMEM lanes = threads
constexpr int KSTEP = 32;            // bytes of the contraction dimension one kind::i8 instruction consumes
constexpr int ROWBLK = TILE_M * 16;  // bytes between consecutive 16-byte K chunks of the A image ("leading byte offset")

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

// ---- mbarrier -------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
// Blocks until the phase with the given parity has completed.  A wait that does not complete within ~2^26 polls can
// only mean a programming error in this file: trap (launch failure) instead of hanging the device.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  uint32_t done = 0;
  uint32_t polls = 0;
  while (true) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}\n"
        : "=r"(done)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    if (done) break;
    if (++polls > (1u << 26)) __trap();
  }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
// make generic-proxy shared-memory writes (st.shared) visible to the async proxy (tensor core, bulk copy)
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
__device__ __forceinline__ uint32_t pow2_cols(uint32_t c) {
  uint32_t p = 32;
  while (p < c) p <<= 1;
  return p;
}

// 32 consecutive columns of this thread's TMEM lane (lane = 32 * (warp % 4) + lane id) -> registers
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&r)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}

// Dynamic shared memory to request so that no more CTAs become resident on an SM than can hold `tmem_cols` TMEM
// columns each (512 per SM): a CTA that blocks inside tcgen05.alloc holds up the SM's other tcgen05 traffic.
inline size_t smem_for_tmem_residency(size_t smem_needed, uint32_t tmem_cols) {
  const size_t per_sm = 227 * 1024;
  const uint32_t max_ctas = 512 / tmem_cols;                 // 1, 2, 4, 8, 16
  const size_t floor_bytes = per_sm / (max_ctas + 1) + 1024; // one more CTA would not fit (1 KB: per-CTA reserved + static)
  return smem_needed > floor_bytes ? smem_needed : floor_bytes;
}

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
__device__ __forceinline__ void mma_i8(uint32_t tmem_d, uint64_t adesc, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t}\n" ::"r"(tmem_d),
      "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// arrive on `bar` once every MMA issued so far by this thread has finished (also orders them before the arrive)
__device__ __forceinline__ void mma_commit(uint64_t* bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar)) : "memory");
}

// ---- the MMA phase shared by both kernels ---------------------------------------------------------------------------------
// One thread streams `nchunks` column chunks of the constant matrix from global memory (each chunk is stored as its
// shared-memory image [KBimg/16][NC][16 bytes], of which the first KB/16 blocks are used) through a two-deep buffer
// and issues, per chunk, KB/32 MMAs into TMEM columns [chunk * NC, chunk * NC + NC).  Returns after committing
// everything to `done`; callers wait on `done` (parity `done_parity`) before touching TMEM or reusing sA.
struct MmaPipe {
  uint64_t full[2];   // bulk copy of buffer b landed
  uint64_t freed[2];  // MMAs reading buffer b finished
  uint64_t done;      // all MMAs of a phase finished
};

__device__ __forceinline__ void mma_pipe_init(MmaPipe* p) {
  mbar_init(&p->full[0], 1); mbar_init(&p->full[1], 1);
  mbar_init(&p->freed[0], 1); mbar_init(&p->freed[1], 1);
  mbar_init(&p->done, 1);
  fence_barrier_init();
}

struct PipeState { uint32_t full_par[2], freed_par[2], done_par; };

__device__ __forceinline__ void mma_phase(MmaPipe* p, PipeState& st, const uint8_t* sA, uint8_t* sB0, uint8_t* sB1,
                                          uint32_t KB, uint32_t NC, const uint8_t* gB, size_t chunk_stride,
                                          uint32_t nchunks, uint32_t tmem_base) {
  const uint32_t bytes = KB * NC;            // used prefix of a chunk image
  const uint32_t idesc = idesc_u8(NC);
  const uint32_t lboB = NC * 16;
  uint8_t* sB[2] = {sB0, sB1};
  const uint32_t pre = nchunks < 2 ? nchunks : 2;
  for (uint32_t c = 0; c < pre; ++c) {
    mbar_expect_tx(&p->full[c], bytes);
    bulk_g2s(sB[c], gB + (size_t)c * chunk_stride, bytes, &p->full[c]);
  }
  for (uint32_t c = 0; c < nchunks; ++c) {
    const uint32_t b = c & 1;
    mbar_wait(&p->full[b], st.full_par[b]); st.full_par[b] ^= 1;
    tc_fence_after();
    const uint32_t aaddr = smem_u32(sA), baddr = smem_u32(sB[b]);
    for (uint32_t k = 0; k < KB / KSTEP; ++k) {
      const uint64_t da = smem_desc(aaddr + k * 2 * ROWBLK, ROWBLK, 128);
      const uint64_t db = smem_desc(baddr + k * 2 * lboB, lboB, 128);
      mma_i8(tmem_base + c * NC, da, db, idesc, k > 0);
    }
    mma_commit(&p->freed[b]);
    if (c + 2 < nchunks) {
      mbar_wait(&p->freed[b], st.freed_par[b]); st.freed_par[b] ^= 1;
      mbar_expect_tx(&p->full[b], bytes);
      bulk_g2s(sB[b], gB + (size_t)(c + 2) * chunk_stride, bytes, &p->full[b]);
    } else {
      st.freed_par[b] ^= 1;   // phase completes without being waited on; keep the parity bookkeeping in step
    }
  }
  mma_commit(&p->done);
}

// Stage 128 rows of a word-major array into the A image: word w of row r comes from src[w * wstride + r].
// Words >= nwords read as zero; if mask_bits != 0 the row's value is first reduced mod 2^mask_bits (callers pass
// nwords <= ceil(mask_bits / 32)).  Thread t owns row t: 32 independent coalesced loads are in flight per thread
// before the first dependent instruction (the loads are the only long-latency step of the kernels built on this),
// then eight conflict-free 16-byte stores.
__device__ __forceinline__ void stage_rows(uint8_t* sA, const uint32_t* __restrict__ src, size_t wstride, uint32_t nwords,
                                           uint32_t KB, uint32_t mask_bits) {
  const uint32_t t = threadIdx.x;
  const uint32_t nch = KB / 16;
  const uint32_t* p = src + t;
  for (uint32_t kc0 = 0; kc0 < nch; kc0 += 8) {
    uint32_t w[32];
#pragma unroll
    for (int i = 0; i < 32; ++i) {
      const uint32_t wi = kc0 * 4 + i;
      w[i] = __ldg(p + (size_t)min(wi, nwords - 1) * wstride);     // clamped: always a valid address, no branch
    }
#pragma unroll
    for (int i = 0; i < 32; ++i)
      if (kc0 * 4 + i >= nwords) w[i] = 0;
#pragma unroll
    for (int c = 0; c < 8; ++c)
      if (kc0 + c < nch)
        *reinterpret_cast<uint4*>(sA + (size_t)(kc0 + c) * ROWBLK + t * 16) = make_uint4(w[4 * c], w[4 * c + 1], w[4 * c + 2], w[4 * c + 3]);
  }
  if (mask_bits & 31) {   // partial top word: each thread patches its own row (same thread wrote it)
    const uint32_t wi = mask_bits >> 5;
    if (wi < nwords) {
      uint32_t* q = reinterpret_cast<uint32_t*>(sA + (size_t)(wi / 4) * ROWBLK + t * 16) + (wi % 4);
      *q &= (1u << (mask_bits & 31)) - 1u;
    }
  }
}

}  // namespace umma
}  // namespace fhe
