// pipe.cuh -- the persistent, warp-specialised conversion pipeline both base conversions run on (S1 limb -> RNS,
// S5 RNS -> limb; PAPER.md:337-344, 360-366 -- the steps the paper calls its primary bottleneck).
//
// Both conversions are the contraction  D[n][c] = sum_kb byte_kb(row n) * Bconst[kb][c]  (u8 x u8 -> s32, exact) over a
// word-major array src[w][n] (umma.cuh).  One CTA per SM walks the 128-coefficient tiles of every polynomial of the
// launch; inside it three roles run concurrently, tied together by mbarriers only:
//
//   loader warps       global -> registers -> TMEM: thread (quarter, lane) owns tile row 32 quarter + lane, which is
//                      TMEM lane 32 quarter + lane.  Word w of its coefficient is column w of the A operand: the i8
//                      MMA reads an A operand held in TMEM as four K-bytes per 32-bit cell, little-endian -- exactly
//                      the word-major data, so no transposition through shared memory exists.  Up to 64 coalesced
//                      loads are in flight per thread; the A operand is double-buffered.
//   MMA thread (1)     per tile and per 64-column chunk of the constant matrix (resident in shared memory, loaded once
//                      per CTA with cp.async.bulk; streamed through a ring when it does not fit): KB/32
//                      tcgen05.mma kind::i8 into one buffer of a ring of accumulator chunks in TMEM.
//   epilogue warps     (4 or 8) tcgen05.ld of a finished accumulator chunk, then the conversion's own arithmetic (an Epi
//                      functor: Barrett reduction and store for S1; carry pass, mod-Q / divide-by-P post-processing and
//                      store for S5).
//
// TMEM budget: nA * KB/4 columns of A + nD * 64 columns of accumulators <= 512.
#pragma once
#include "umma.cuh"

namespace fhe {
namespace pipe {

using namespace umma;

constexpr uint32_t NC = 64;                                   // accumulator columns per chunk
constexpr uint32_t MAX_SLOTS = 16, MAX_D = 4, MAX_A = 2;
constexpr uint32_t CTRL_BYTES = 1024;
constexpr size_t SMEM_LIMIT = 227 * 1024;

struct Ctrl {
  uint64_t a_full[MAX_A], a_free[MAX_A];      // A operand buffer written (256 loader arrivals) / consumed (MMA commit)
  uint64_t d_full[MAX_D], d_free[MAX_D];      // accumulator chunk finished (MMA commit) / drained (128 epilogue arrivals)
  uint64_t b_full[MAX_SLOTS], b_free[MAX_SLOTS];
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= CTRL_BYTES, "control block");

struct PipeArgs {
  // A source: polynomial p = (o, i) = (p / inner, p % inner) lives at src + o * src_outer + i * src_inner; word w of
  // coefficient n at [w * N + n].  Words >= nwords read as zero; mask_bits != 0 reduces the row mod 2^mask_bits.
  const uint32_t* src; size_t src_outer, src_inner;
  uint32_t inner, npoly, N, nwords, mask_bits;
  // contraction
  const uint8_t* B; size_t chunk_stride;      // chunk c of the constant image at B + c * chunk_stride; KB * NC bytes used
  uint32_t KB, nchunks, nslots, nA, nD, tmem_cols;
  uint32_t epi_off, b_off;                    // byte offsets of the epilogue scratch and the B slots in dynamic smem
};

// ---- host-side plan -----------------------------------------------------------------------------------------------------
struct Plan {
  uint32_t KB = 0, nchunks = 0, nslots = 0, nA = 0, nD = 0, tmem_cols = 0, epi_off = 0, b_off = 0;
  size_t smem = 0;
  bool ok = false;
};
inline Plan make_plan(uint32_t KB, uint32_t nchunks, size_t epi_bytes) {
  Plan p;
  p.KB = KB; p.nchunks = nchunks;
  const uint32_t a_cols = KB / 4;
  p.nD = (2 * a_cols + 4 * NC <= 512) ? 4 : 2;
  p.nA = (2 * a_cols + p.nD * NC <= 512) ? 2 : 1;
  const uint32_t cols = p.nA * a_cols + p.nD * NC;
  if (cols > 512 || nchunks == 0) return p;
  p.tmem_cols = 32;
  while (p.tmem_cols < cols) p.tmem_cols <<= 1;
  p.epi_off = CTRL_BYTES;
  p.b_off = (uint32_t)((CTRL_BYTES + epi_bytes + 127) & ~(size_t)127);
  const size_t chunk_bytes = (size_t)KB * NC;
  if (p.b_off + 2 * chunk_bytes > SMEM_LIMIT) return p;
  size_t fit = (SMEM_LIMIT - p.b_off) / chunk_bytes;
  if (fit > MAX_SLOTS) fit = MAX_SLOTS;
  p.nslots = nchunks <= fit ? nchunks : (uint32_t)fit;
  if (p.nslots < nchunks && p.nslots < 2) return p;
  p.smem = p.b_off + (size_t)p.nslots * chunk_bytes;
  p.ok = true;
  return p;
}
inline void fill_args(PipeArgs& a, const Plan& p) {
  a.KB = p.KB; a.nchunks = p.nchunks; a.nslots = p.nslots; a.nA = p.nA; a.nD = p.nD; a.tmem_cols = p.tmem_cols;
  a.epi_off = p.epi_off; a.b_off = p.b_off;
}

#ifdef __CUDACC__
// ---- device helpers -------------------------------------------------------------------------------------------------------
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
// D[tmem] (+)= A[tmem] * B[smem]: A operand in tensor memory (lane = row, 32-bit cell = four K bytes)
__device__ __forceinline__ void mma_i8_ts(uint32_t tmem_d, uint32_t tmem_a, uint64_t bdesc, uint32_t idesc, uint32_t accumulate) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t}\n" ::"r"(tmem_d),
      "r"(tmem_a), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
__device__ __forceinline__ void tmem_st8(uint32_t taddr, const uint32_t* r) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]),
               "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7])
               : "memory");
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// 32 columns, no wait (callers batch two of these before tmem_ld_wait)
__device__ __forceinline__ void tmem_ld32_nowait(uint32_t taddr, uint32_t* r) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
      "{%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
        "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
        "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
        "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
      : "r"(taddr)
      : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// One batch of 32 words (A columns [32 b, 32 b + 32)) of this thread's row: issue the loads.
__device__ __forceinline__ void load_batch(uint32_t (&w)[32], const uint32_t* __restrict__ p, size_t N, uint32_t b,
                                           uint32_t nwords) {
#pragma unroll
  for (int i = 0; i < 32; ++i) {
    const uint32_t wi = b * 32 + i;
    w[i] = wi < nwords ? __ldg(p + (size_t)wi * N) : 0u;        // warp-uniform predicate
  }
}
// ... then zero the padding, mask the top word and write the batch to TMEM columns [32 b, min(32 b + 32, a_cols)).
__device__ __forceinline__ void store_batch(uint32_t (&w)[32], uint32_t taddr_a, uint32_t b, uint32_t nwords, uint32_t a_cols,
                                            uint32_t mask_bits) {
#pragma unroll
  for (int i = 0; i < 32; ++i)
    if ((mask_bits & 31) && b * 32 + i == (mask_bits >> 5)) w[i] &= (1u << (mask_bits & 31)) - 1u;
  (void)nwords;
#pragma unroll
  for (int c = 0; c < 4; ++c)
    if (b * 32 + c * 8 < a_cols) tmem_st8(taddr_a + b * 32 + c * 8, &w[c * 8]);
}

// ---- the kernel -------------------------------------------------------------------------------------------------------------
// Epi: struct with
//   static constexpr uint32_t LOAD_WARPS;                             4 or 8 loader warps (one or two per TMEM lane quarter)
//   static constexpr uint32_t GROUPS;                                 1: every epilogue warp takes the 64 columns of a chunk
//                                                                     2: warp group g takes columns [32 g, 32 g + 32) of it
//   struct Params;                                                    by-value kernel argument
//   __device__ Epi(const Params&, const PipeArgs&, uint8_t* scratch, uint32_t etid, uint32_t grp);
//   __device__ void begin_tile(uint32_t o, uint32_t i, uint32_t n0);  polynomial (o, i), first coefficient of the tile
//   __device__ void consume(uint32_t col0, const uint32_t* t);        32 accumulator columns [col0, col0 + 32) of row etid
//   __device__ void end_tile();
// Warp roles: [0, 4 GROUPS) epilogue, then LOAD_WARPS loaders, then the MMA issuer.
constexpr uint32_t nthreads(uint32_t groups, uint32_t load_warps) { return (4 * groups + load_warps + 1) * 32; }

// barrier among the epilogue threads only (id 1; id 0 is __syncthreads)
__device__ __forceinline__ void epi_sync(uint32_t nthr) { asm volatile("bar.sync 1, %0;" ::"r"(nthr) : "memory"); }

template <class Epi>
__global__ void __launch_bounds__(nthreads(Epi::GROUPS, Epi::LOAD_WARPS), 1)
pipe_kernel(const __grid_constant__ PipeArgs a, const __grid_constant__ typename Epi::Params ep) {
  constexpr uint32_t EPIW = 4 * Epi::GROUPS, LOAD_WARPS = Epi::LOAD_WARPS, HALVES = LOAD_WARPS / 4, MMAW = EPIW + LOAD_WARPS;
  extern __shared__ __align__(1024) uint8_t smem[];
  Ctrl* ctl = reinterpret_cast<Ctrl*>(smem);
  uint8_t* sB = smem + a.b_off;
  const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t tpp = a.N / TILE_M;                               // tiles per polynomial
  const uint32_t ntiles = a.npoly * tpp;
  const uint32_t mine = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const uint32_t a_cols = a.KB / 4;
  const uint32_t chunk_bytes = a.KB * NC;
  const bool resident = a.nslots >= a.nchunks;
  const uint32_t dmask = a.nD - 1, dshift = a.nD == 4 ? 2 : 1;     // nD in {2, 4}
  const uint32_t amask = a.nA - 1, ashift = a.nA - 1;              // nA in {1, 2}

  if (tid == 0) {
    for (uint32_t i = 0; i < MAX_A; ++i) { mbar_init(&ctl->a_full[i], LOAD_WARPS * 32); mbar_init(&ctl->a_free[i], 1); }
    for (uint32_t i = 0; i < MAX_D; ++i) { mbar_init(&ctl->d_full[i], 1); mbar_init(&ctl->d_free[i], EPIW * 32); }
    for (uint32_t i = 0; i < MAX_SLOTS; ++i) { mbar_init(&ctl->b_full[i], 1); mbar_init(&ctl->b_free[i], 1); }
    fence_barrier_init();
  }
  if (warp == MMAW) tmem_alloc(&ctl->tmem_base, a.tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_a = ctl->tmem_base;                          // A buffers: columns [0, nA * a_cols)
  const uint32_t tmem_d = tmem_a + a.nA * a_cols;                  // accumulator ring: nD chunks of NC columns

  if (warp == MMAW) {
    // ===== MMA issuer (one thread) =====
    if (lane == 0 && mine) {
      const uint32_t total = mine * a.nchunks;
      uint32_t ld_slot = 0, ld_chunk = 0, ld_count = 0;            // next chunk to fetch: ring slot, chunk of the image
      auto load_next = [&]() {
        mbar_expect_tx(&ctl->b_full[ld_slot], chunk_bytes);
        bulk_g2s(sB + (size_t)ld_slot * chunk_bytes, a.B + (size_t)ld_chunk * a.chunk_stride, chunk_bytes, &ctl->b_full[ld_slot]);
        if (++ld_slot == a.nslots) ld_slot = 0;
        if (++ld_chunk == a.nchunks) ld_chunk = 0;
        ++ld_count;
      };
      const uint32_t pre = total < a.nslots ? total : a.nslots;
      while (ld_count < pre) load_next();
      const uint32_t idesc = idesc_u8(NC);
      const uint32_t lboB = NC * 16;
      uint32_t g = 0, slot = 0, slot_par = 0;                      // running chunk index, its ring slot and the slot's use parity
      uint32_t pslot = 0, pslot_par = 0;                           // the same for the previous chunk
      for (uint32_t k = 0; k < mine; ++k) {
        const uint32_t abuf = k & amask;
        mbar_wait(&ctl->a_full[abuf], (k >> ashift) & 1);
        tc_fence_after();
        for (uint32_t c = 0; c < a.nchunks; ++c, ++g) {
          if (!resident || k == 0) mbar_wait(&ctl->b_full[slot], slot_par);
          const uint32_t dbuf = g & dmask;
          mbar_wait(&ctl->d_free[dbuf], ((g >> dshift) & 1) ^ 1);
          tc_fence_after();
          const uint32_t baddr = smem_u32(sB + (size_t)slot * chunk_bytes);
          for (uint32_t ks = 0; ks < a.KB / KSTEP; ++ks) {
            const uint64_t db = smem_desc(baddr + ks * 2 * lboB, lboB, 128);
            mma_i8_ts(tmem_d + dbuf * NC, tmem_a + abuf * a_cols + ks * (KSTEP / 4), db, idesc, ks > 0);
          }
          mma_commit(&ctl->d_full[dbuf]);
          if (!resident) {
            mma_commit(&ctl->b_free[slot]);
            if (g >= 1 && ld_count < total) {                      // the slot of the previous chunk is the next to refill
              mbar_wait(&ctl->b_free[pslot], pslot_par);
              load_next();
            }
          }
          pslot = slot; pslot_par = slot_par;
          if (++slot == a.nslots) { slot = 0; slot_par ^= 1; }
        }
        mma_commit(&ctl->a_free[abuf]);
      }
    }
    __syncwarp();
  } else if (warp >= EPIW) {
    // ===== loaders =====
    const uint32_t lw = warp - EPIW, quarter = lw & 3, half = lw >> 2;
    const uint32_t row = quarter * 32 + lane;
    const uint32_t nbatch = (a_cols + 31) / 32;
    uint32_t tile = blockIdx.x;
    uint32_t poly = tile / tpp, tin = tile % tpp;                  // advanced incrementally below
    const uint32_t dpoly = gridDim.x / tpp, dtin = gridDim.x % tpp;
    uint32_t po = poly / a.inner, pi = poly % a.inner;
    for (uint32_t k = 0; k < mine; ++k) {
      const uint32_t* p = a.src + (size_t)po * a.src_outer + (size_t)pi * a.src_inner + tin * TILE_M + row;
      const uint32_t abuf = k & amask;
      const uint32_t taddr = tmem_a + abuf * a_cols + ((quarter * 32u) << 16);
      bool waited = false;
      for (uint32_t b = half; b < nbatch; b += 2 * HALVES) {       // this warp's batches, two at a time
        uint32_t w0[32], w1[32];
        const bool two = b + HALVES < nbatch;
        load_batch(w0, p, a.N, b, a.nwords);
        if (two) load_batch(w1, p, a.N, b + HALVES, a.nwords);
        if (!waited) {                                             // loads are in flight while the buffer is still being read
          mbar_wait(&ctl->a_free[abuf], ((k >> ashift) & 1) ^ 1);
          tc_fence_after();
          waited = true;
        }
        store_batch(w0, taddr, b, a.nwords, a_cols, a.mask_bits);
        if (two) store_batch(w1, taddr, b + HALVES, a.nwords, a_cols, a.mask_bits);
      }
      if (!waited) mbar_wait(&ctl->a_free[abuf], ((k >> ashift) & 1) ^ 1);   // a warp without batches still keeps in step
      tmem_st_wait();
      tc_fence_before();
      mbar_arrive(&ctl->a_full[abuf]);
      tin += dtin; poly += dpoly;
      if (tin >= tpp) { tin -= tpp; ++poly; }
      po = poly / a.inner; pi = poly % a.inner;
    }
  } else {
    // ===== epilogue =====
    const uint32_t grp = warp >> 2;
    const uint32_t etid = (warp & 3) * 32 + lane;                  // 0..127 = tile row = TMEM lane
    const uint32_t lane_off = ((warp & 3) * 32u) << 16;
    Epi epi(ep, a, smem + a.epi_off, etid, grp);
    uint32_t g = 0;
    for (uint32_t k = 0; k < mine; ++k) {
      const uint32_t tile = blockIdx.x + k * gridDim.x;
      const uint32_t poly = tile / tpp, n0 = (tile % tpp) * TILE_M;
      epi.begin_tile(poly / a.inner, poly % a.inner, n0);
      for (uint32_t c = 0; c < a.nchunks; ++c, ++g) {
        const uint32_t dbuf = g & dmask;
        mbar_wait(&ctl->d_full[dbuf], (g >> dshift) & 1);
        tc_fence_after();
        if constexpr (Epi::GROUPS == 1) {
          uint32_t t[64];
          tmem_ld32_nowait(tmem_d + dbuf * NC + lane_off, t);
          tmem_ld32_nowait(tmem_d + dbuf * NC + 32 + lane_off, t + 32);
          tmem_ld_wait();
          tc_fence_before();
          mbar_arrive(&ctl->d_free[dbuf]);                         // the accumulator chunk is in registers: hand it back
          epi.consume(c * NC, t);
          epi.consume(c * NC + 32, t + 32);
        } else {
          uint32_t t[32];
          tmem_ld32_nowait(tmem_d + dbuf * NC + grp * 32 + lane_off, t);
          tmem_ld_wait();
          tc_fence_before();
          mbar_arrive(&ctl->d_free[dbuf]);
          epi.consume(c * NC + grp * 32, t);
        }
      }
      epi.end_tile();
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == MMAW) tmem_dealloc(tmem_a, a.tmem_cols);
}

template <class Epi>
inline cudaError_t launch_pipe(const PipeArgs& a, const typename Epi::Params& ep, size_t smem, int n_sm, cudaStream_t s) {
  static size_t configured = 0;
  if (smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(pipe_kernel<Epi>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  const uint32_t ntiles = a.npoly * (a.N / TILE_M);
  const uint32_t grid = ntiles < (uint32_t)n_sm ? ntiles : (uint32_t)n_sm;
  pipe_kernel<Epi><<<grid, nthreads(Epi::GROUPS, Epi::LOAD_WARPS), smem, s>>>(a, ep);
  return cudaGetLastError();
}
#endif  // __CUDACC__

}  // namespace pipe
}  // namespace fhe
