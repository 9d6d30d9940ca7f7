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
//                      the word-major data, so no transposition through shared memory exists.  The A operand is
//                      double-buffered when tensor memory has the room.
//   MMA thread (1)     per tile: KB/32 tcgen05.mma kind::i8 per SPAN of up to 256 accumulator columns.  A
//                      tcgen05.mma costs ~100 cycles whatever its N, plus ~350 when it starts a new accumulator
//                      (measured on B200), so the instruction is made as wide as the ISA allows (N = 256) and the K
//                      loop as long as the operand: narrow 64-column MMAs left the tensor pipe as the bottleneck.
//   epilogue warps     tcgen05.ld of 64 finished accumulator columns (a "chunk"), then the conversion's own arithmetic
//                      (an Epi functor: Barrett reduction and store for S1; carry pass, mod-Q / divide-by-P
//                      post-processing and store for S5).  A chunk's columns are handed back to the MMA thread as soon
//                      as they are in registers, so the next tile's MMAs overlap this tile's arithmetic.
//
// Tensor memory holds the A buffers and ONE set of accumulator columns for all chunks of a pass:
//   nA * KB/4 + 64 * chunks_per_pass <= 512 columns.
// When the constant matrix has more columns than that (or than shared memory holds), the launch runs several passes over
// its tiles, pass p with columns [p * cpp * 64, ...) of B resident in shared memory (loaded once per pass per CTA).
#pragma once
#include <cstring>
#include "umma.cuh"

namespace fhe {
namespace pipe {

using namespace umma;

constexpr uint32_t NC = 64;                                   // accumulator columns per chunk (the epilogue's unit)
constexpr uint32_t SPAN = 4;                                  // chunks per MMA span: N = 256
constexpr uint32_t MAX_CHUNKS = 8, MAX_SPANS = 2, MAX_A = 2;  // per pass (512 TMEM columns)
constexpr uint32_t CTRL_BYTES = 1024;
constexpr size_t SMEM_LIMIT = 227 * 1024;

struct Ctrl {
  uint64_t a_full[MAX_A], a_free[MAX_A];      // A buffer written (one arrival per loader warp) / consumed (MMA commit)
  uint64_t d_full[2][MAX_SPANS];              // [accumulator set] the span's accumulators finished (MMA commit)
  uint64_t d_free[2][MAX_CHUNKS];                // the chunk's accumulators are in registers (one arrival per epilogue warp)
  uint64_t g_full[MAX_SPANS][4];              // CHUNK_ALT: the span finished, barrier [wi mod 4] for work item wi
  uint64_t r_full[2], r_free[2];              // TMA staging ring of the A source: slot landed (tx bytes) / read out by every loader warp
  uint64_t b_full, mma_done;                  // B of the pass landed (bulk copies) / every MMA of the pass finished
  uint32_t tmem_base;
};
static_assert(sizeof(Ctrl) <= CTRL_BYTES, "control block");

struct PipeArgs {
  // A source: polynomial p = (o, i) = (p / inner, p % inner) lives at src + o * src_outer + i * src_inner; word w of
  // coefficient n at [w * N + n].  Words >= nwords read as zero; mask_bits != 0 reduces the row mod 2^mask_bits.
  const uint32_t* src; size_t src_outer, src_inner;
  uint32_t inner, npoly, N, nwords, mask_bits;
  // contraction: the constant image is [kb / 16][b_cols][16 bytes] (K-major core matrices, no swizzle), KB bytes of
  // contraction and nchunks * 64 columns of it are used
  const uint8_t* B; uint32_t b_cols;
  uint32_t KB, nchunks;
  uint32_t npass, cpp;                        // passes over the tiles, chunks per pass (the last pass may have fewer)
  uint32_t nA, nsets, tmem_cols;              // nsets: accumulator column sets (2: tiles alternate between them, TILE_ALT)
  uint32_t epi_stride;                        // TILE_ALT: bytes between the scratch regions of the two epilogue groups
  uint32_t epi_off, b_off;                    // byte offsets of the epilogue scratch and of B in dynamic smem
  // TMA staging of the A source (Epi::LOAD_TMA): ring_slots tiles of [nwords][128] words at ring_off, filled by one 2-D
  // tensor copy each from the matrix view [rows][N] of the source (row of word w of polynomial (o, i) = row_outer o + row_inner i + w)
  uint32_t ring_slots, ring_off, row_outer, row_inner;
};

// ---- host-side plan -----------------------------------------------------------------------------------------------------
struct Plan {
  uint32_t KB = 0, nchunks = 0, npass = 0, cpp = 0, nA = 0, nsets = 1, tmem_cols = 0, epi_off = 0, b_off = 0, epi_stride = 0;
  uint32_t ring_slots = 0, ring_off = 0;      // TMA staging ring (add_ring)
  size_t smem = 0;
  bool ok = false;
};
// single_pass: the epilogue carries state across the chunks of a tile (S5), so all columns must fit at once
// tile_alt: two epilogue groups on alternate tiles, each with its own accumulator set and scratch region; taken when two
// sets of all chunks fit beside ONE A buffer (single pass), else the plan falls back to one set served by group 0 alone.
inline Plan make_plan(uint32_t KB, uint32_t nchunks, size_t epi_bytes, bool single_pass, bool tile_alt = false) {
  Plan p;
  p.KB = KB; p.nchunks = nchunks;
  const uint32_t a_cols = KB / 4;
  if (nchunks == 0 || a_cols + NC > 512) return p;
  p.epi_off = CTRL_BYTES;
  p.epi_stride = (uint32_t)((epi_bytes + 127) & ~(size_t)127);
  p.b_off = CTRL_BYTES + (tile_alt ? 2 : 1) * p.epi_stride;
  if (p.b_off + (size_t)KB * NC > SMEM_LIMIT) return p;
  const uint32_t smem_chunks = (uint32_t)((SMEM_LIMIT - p.b_off) / ((size_t)KB * NC));
  if (tile_alt && a_cols + 2 * nchunks * NC <= 512 && nchunks <= MAX_CHUNKS &&
      p.b_off + (size_t)nchunks * KB * NC <= SMEM_LIMIT) {
    p.nA = 1; p.nsets = 2; p.npass = 1; p.cpp = nchunks;
  }
  for (uint32_t nA = 2; nA >= 1 && !p.npass; --nA) {
    if (nA * a_cols + NC > 512) continue;
    uint32_t cap = (512 - nA * a_cols) / NC;                // chunks tensor memory holds beside the A buffers
    if (cap > MAX_CHUNKS) cap = MAX_CHUNKS;
    if (cap > smem_chunks) cap = smem_chunks;
    if (cap == 0) continue;
    const uint32_t npass = (nchunks + cap - 1) / cap;
    if (single_pass && npass > 1) continue;                 // try nA = 1, which leaves more columns
    p.nA = nA; p.npass = npass; p.cpp = (nchunks + npass - 1) / npass;
  }
  if (!p.npass) return p;
  const uint32_t cols = p.nA * a_cols + p.nsets * p.cpp * NC;
  p.tmem_cols = 32;
  while (p.tmem_cols < cols) p.tmem_cols <<= 1;
  p.smem = p.b_off + (size_t)p.cpp * KB * NC;
  p.ok = true;
  return p;
}
// Room behind B for TWO staged tiles of `nwords` source words ([nwords][128] uint32 each), or no ring at all.  The ring is
// only taken while the CTA stays within RING_SMEM_CAP: the launches overlap their neighbours' tails (PDL), and a CTA that
// fills the SM's shared memory cannot become resident beside the last CTAs of the transform before it -- measured at the
// bench shape, a 204 KB relin CRT lost 0.075 ms of the step to that while its own time fell by 0.008 ms; one slot alone was
// slower than register-landing loads.
constexpr size_t RING_SMEM_CAP = 160 * 1024;
inline void add_ring(Plan& p, uint32_t nwords) {
  if (!p.ok) return;
  const size_t off = (p.smem + 127) & ~(size_t)127, slot = (size_t)nwords * TILE_M * 4;
  if (off + 2 * slot > RING_SMEM_CAP) return;
  p.ring_slots = 2; p.ring_off = (uint32_t)off; p.smem = off + 2 * slot;
}
inline void fill_args(PipeArgs& a, const Plan& p) {
  a.KB = p.KB; a.nchunks = p.nchunks; a.npass = p.npass; a.cpp = p.cpp; a.nA = p.nA; a.nsets = p.nsets; a.tmem_cols = p.tmem_cols;
  a.epi_stride = p.epi_stride;
  a.epi_off = p.epi_off; a.b_off = p.b_off;
  a.ring_slots = p.ring_slots; a.ring_off = p.ring_off; a.row_outer = a.row_inner = 0;
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

// streaming load: read once, no L1 line allocated for it
__device__ __forceinline__ uint32_t ld_stream(const uint32_t* p) {
  uint32_t v;
  asm volatile("ld.global.nc.L1::no_allocate.u32 %0, [%1];" : "=r"(v) : "l"(p));
  return v;
}
// One batch of LR words (A columns [w0, w0 + LR)) of this thread's row, word w at q + w * N.  The common case -- every
// word of the batch exists -- is one load and one pointer step per word; only the last batch of a row pays for the
// per-word bound (words past `nvalid` read as zero: the padding of the contraction dimension).
template <int LR>
__device__ __forceinline__ void load_full(uint32_t (&w)[LR], const uint32_t* __restrict__ q, size_t N) {
#pragma unroll
  for (int i = 0; i < LR; ++i) { w[i] = ld_stream(q); q += N; }
}
template <int LR>
__device__ __forceinline__ void load_tail(uint32_t (&w)[LR], const uint32_t* __restrict__ q, size_t N, uint32_t nvalid) {
#pragma unroll
  for (int i = 0; i < LR; ++i) { w[i] = (uint32_t)i < nvalid ? ld_stream(q) : 0u; q += N; }   // warp-uniform predicate
}
// ... then write the batch to TMEM columns [w0, min(w0 + LR, a_cols)), eight at a time.
template <int LR>
__device__ __forceinline__ void store_batch(uint32_t (&w)[LR], uint32_t taddr_a, uint32_t w0, uint32_t a_cols) {
#pragma unroll
  for (int c = 0; c < LR / 8; ++c)
    if (w0 + c * 8 < a_cols) tmem_st8(taddr_a + w0 + c * 8, &w[c * 8]);
}

// ---- the kernel -------------------------------------------------------------------------------------------------------------
// Epi: struct with
//   static constexpr uint32_t LOAD_WARPS;                             4 or 8 loader warps (one or two per TMEM lane quarter)
//   static constexpr bool LOAD_ALT;                                   8 loader warps only.  false: the two warps of a lane quarter
//                                                                     split the words of every tile; true: they take alternate
//                                                                     tiles whole (two tiles' loads in flight; needs nA = 2)
//   static constexpr bool LOAD_TMA;                                   the A source may be staged through shared memory by TMA
//                                                                     (PipeArgs::ring_slots > 0; the loader warps of a lane quarter then
//                                                                     split the words of every tile, whatever LOAD_ALT says)
//   static constexpr int LOAD_WORDS, MAX_REGS;                        words of its row a loader thread has in flight
//                                                                     (multiple of 8); register cap of the kernel
//   static constexpr uint32_t GROUPS;                                 1, 2 or 4 epilogue warp groups: group g takes columns
//                                                                     [g 64/GROUPS, (g + 1) 64/GROUPS) of every chunk
//   struct Params;                                                    by-value kernel argument
//   static constexpr bool TILE_ALT;                                   GROUPS = 2 only: the groups are two whole epilogues on
//                                                                     alternate tiles (own accumulator set, scratch, Epi object)
//   static constexpr bool CHUNK_ALT;                                  the groups take WHOLE chunks in rotation (chunk c of work item
//                                                                     wi goes to group (c + wi) mod GROUPS), so the chunks of a span
//                                                                     are drained side by side and handed back within one chunk time:
//                                                                     the next tile's MMAs overlap this tile's arithmetic.  For
//                                                                     epilogues without state across chunks (S1)
//   __device__ Epi(const Params&, const PipeArgs&, uint8_t* scratch, uint32_t etid, uint32_t grp, uint32_t bar);
//                                                                     bar: named barrier of the threads sharing this scratch (epi_sync)
//   __device__ void begin_tile(uint32_t o, uint32_t i, uint32_t n0);  polynomial (o, i), first coefficient of the tile
//   __device__ void consume(uint32_t col0, const uint32_t* t);        64/GROUPS accumulator columns from col0 on, of row etid
//                                                                     (GROUPS = 1: called twice per chunk, 32 columns each)
//   __device__ void end_tile();
// Warp roles: [0, 4 GROUPS) epilogue, then LOAD_WARPS loaders, then the MMA issuer.
constexpr uint32_t nthreads(uint32_t groups, uint32_t load_warps) { return (4 * groups + load_warps + 1) * 32; }

// barrier among the epilogue threads that share a scratch region (id >= 1; id 0 is __syncthreads)
__device__ __forceinline__ void epi_sync(uint32_t bar, uint32_t nthr) { asm volatile("bar.sync %0, %1;" ::"r"(bar), "r"(nthr) : "memory"); }


template <int NCOL>
__device__ __forceinline__ void tmem_ld_cols(uint32_t taddr, uint32_t* r) {
  static_assert(NCOL == 16 || NCOL == 32, "epilogue slice");
  if constexpr (NCOL == 32) {
    tmem_ld32_nowait(taddr, r);
  } else {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
                   "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
                 : "r"(taddr)
                 : "memory");
  }
}

template <class Epi>
__global__ void __maxnreg__(Epi::MAX_REGS)   // 64 K registers / (warps rounded up to a multiple of 4) / 32
pipe_kernel(const __grid_constant__ PipeArgs a, const __grid_constant__ typename Epi::Params ep,
            const __grid_constant__ CUtensorMap tmap) {
  constexpr uint32_t GROUPS = Epi::GROUPS, EPIW = 4 * GROUPS, LOAD_WARPS = Epi::LOAD_WARPS, HALVES = LOAD_WARPS / 4,
                     MMAW = EPIW + LOAD_WARPS, GC = NC / GROUPS;
  constexpr int LR = Epi::LOAD_WORDS;
  constexpr bool ALT = Epi::LOAD_ALT;
  static_assert(!ALT || LOAD_WARPS == 8, "alternating loaders come in pairs");
  static_assert((GROUPS == 1 || GROUPS == 2 || GROUPS == 4) && (LOAD_WARPS == 4 || LOAD_WARPS == 8), "pipeline shape");
  static_assert(((EPIW + LOAD_WARPS + 1 + 3) / 4 * 4) * 32 * Epi::MAX_REGS <= 65536, "one CTA must fit the register file");
  extern __shared__ __align__(1024) uint8_t smem[];
  Ctrl* ctl = reinterpret_cast<Ctrl*>(smem);
  uint8_t* sB = smem + a.b_off;
  const uint32_t tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
  const uint32_t tpp = a.N / TILE_M;                               // tiles per polynomial
  const uint32_t ntiles = a.npoly * tpp;
  const uint32_t mine = blockIdx.x < ntiles ? (ntiles - blockIdx.x + gridDim.x - 1) / gridDim.x : 0;
  const uint32_t a_cols = a.KB / 4;
  const uint32_t amask = a.nA - 1, ashift = a.nA - 1;              // nA in {1, 2}

  if (tid == 0) {
    for (uint32_t i = 0; i < MAX_A; ++i) { mbar_init(&ctl->a_full[i], (ALT && !(Epi::LOAD_TMA && a.ring_slots)) ? 4 : LOAD_WARPS); mbar_init(&ctl->a_free[i], 1); }
    for (uint32_t i = 0; i < MAX_SPANS; ++i) {
      mbar_init(&ctl->d_full[0][i], 1); mbar_init(&ctl->d_full[1][i], 1);
      for (uint32_t g = 0; g < 4; ++g) mbar_init(&ctl->g_full[i][g], 1);
    }
    // one arrival per WARP (its lane 0, after the warp-collective tcgen05.wait): hundreds of per-thread arrivals on one
    // mbarrier serialise in shared memory and were a quarter of the epilogue's time
    for (uint32_t i = 0; i < MAX_CHUNKS; ++i) {
      mbar_init(&ctl->d_free[0][i], (Epi::TILE_ALT || Epi::CHUNK_ALT) ? 4 : EPIW);
      mbar_init(&ctl->d_free[1][i], (Epi::TILE_ALT || Epi::CHUNK_ALT) ? 4 : EPIW);
    }
    for (uint32_t i = 0; i < 2; ++i) { mbar_init(&ctl->r_full[i], 1); mbar_init(&ctl->r_free[i], LOAD_WARPS); }
    mbar_init(&ctl->b_full, 1); mbar_init(&ctl->mma_done, 1);
    fence_barrier_init();
  }
  if (warp == MMAW) tmem_alloc(&ctl->tmem_base, a.tmem_cols);
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  pdl_sync();   // barriers and TMEM are set up while the previous kernel drains; global memory is touched only after this
  const uint32_t tmem_a = ctl->tmem_base;                          // A buffers: columns [0, nA * a_cols)
  const uint32_t tmem_d = tmem_a + a.nA * a_cols;                  // chunk c of the pass: columns [c * NC, c * NC + NC)

  if (warp == MMAW) {
    // ===== MMA issuer (one thread) =====
    if (lane == 0 && mine) {
      const uint32_t nkb = a.KB / 16;                              // 16-byte K blocks of the operands
      uint32_t wi = 0;                                             // work item = (pass, tile) in issue order
      for (uint32_t ps = 0; ps < a.npass; ++ps) {
        const uint32_t c0 = ps * a.cpp;
        const uint32_t nc = a.nchunks - c0 < a.cpp ? a.nchunks - c0 : a.cpp;     // chunks of this pass
        const uint32_t nspan = (nc + SPAN - 1) / SPAN;
        // B of the pass: span s as a dense image [nkb][w_s columns][16] at sB + span_off[s]
        uint32_t span_off[MAX_SPANS], span_w[MAX_SPANS];
        if (ps > 0) {                                              // the previous pass's MMAs still read sB
          mma_commit(&ctl->mma_done);
          mbar_wait(&ctl->mma_done, (ps - 1) & 1);
        }
        {
          uint32_t off = 0;
          mbar_expect_tx(&ctl->b_full, nc * NC * a.KB);
          for (uint32_t sp = 0; sp < nspan; ++sp) {
            const uint32_t w = ((nc - sp * SPAN < SPAN ? nc - sp * SPAN : SPAN)) * NC;
            span_off[sp] = off; span_w[sp] = w;
            const uint8_t* src = a.B + (size_t)(c0 + sp * SPAN) * NC * 16;
            for (uint32_t kb = 0; kb < nkb; ++kb)
              bulk_g2s(sB + off + (size_t)kb * w * 16, src + (size_t)kb * a.b_cols * 16, w * 16, &ctl->b_full);
            off += nkb * w * 16;
          }
          mbar_wait(&ctl->b_full, ps & 1);
        }
        for (uint32_t k = 0; k < mine; ++k, ++wi) {
          const uint32_t abuf = wi & amask;
          mbar_wait(&ctl->a_full[abuf], (wi >> ashift) & 1);
          tc_fence_after();
          for (uint32_t sp = 0; sp < nspan; ++sp) {
            const uint32_t cs = sp * SPAN, ce = cs + SPAN < nc ? cs + SPAN : nc;
            const uint32_t dset = a.nsets == 2 ? (wi & 1) : 0, duse = a.nsets == 2 ? (wi >> 1) : wi;   // the set's use count
            for (uint32_t c = cs; c < ce; ++c) mbar_wait(&ctl->d_free[dset][c], (duse & 1) ^ 1);
            tc_fence_after();
            const uint32_t idesc = idesc_u8(span_w[sp]);
            const uint32_t lbo = span_w[sp] * 16;
            const uint32_t baddr = smem_u32(sB + span_off[sp]);
            for (uint32_t ks = 0; ks < a.KB / KSTEP; ++ks) {
              const uint64_t db = smem_desc(baddr + ks * 2 * lbo, lbo, 128);
              mma_i8_ts(tmem_d + (dset * a.cpp + cs) * NC, tmem_a + abuf * a_cols + ks * (KSTEP / 4), db, idesc, ks > 0);
            }
            if constexpr (Epi::CHUNK_ALT) {
              mma_commit(&ctl->g_full[sp][wi % GROUPS]);
            } else {
              mma_commit(&ctl->d_full[dset][sp]);
            }
          }
          mma_commit(&ctl->a_free[abuf]);
        }
      }
    }
    __syncwarp();
  } else if (warp >= EPIW) {
    // ===== loaders =====
    const uint32_t lw = warp - EPIW, quarter = lw & 3, half = lw >> 2;
    const uint32_t row = quarter * 32 + lane;
    // mask_bits != 0 reduces the row mod 2^mask_bits: its top word is cut (the words above are not loaded at all)
    const uint32_t mask_w = a.mask_bits >> 5, mask_m = (a.mask_bits & 31) ? (1u << (a.mask_bits & 31)) - 1u : 0u;
    uint32_t wi = 0;
    if (Epi::LOAD_TMA && a.ring_slots) {
      // TMA-staged source (the loader warps of a lane quarter split the words of a tile): loader warp 0 keeps up to ring_slots tiles in
      // flight as ONE 2-D tensor copy each into shared memory; every loader warp then moves its words shared -> registers ->
      // TMEM.  The loads of the tiles ahead no longer wait for the registers of the tile being stored (with register-landing
      // loads a tile's loads were issued only after the previous tile's tcgen05.st, and the MMA thread waited for its A
      // operand 800-3300 cycles per tile), and 500 LDG.32 per tile leave the LSU.
      const uint32_t nslots = a.ring_slots, slot_words = a.nwords * TILE_M;
      uint32_t* ring = reinterpret_cast<uint32_t*>(smem + a.ring_off);
      const uint32_t total = a.npass * mine;                       // every pass stages the tiles again
      auto issue = [&](uint32_t it) {                              // lane 0 of loader warp 0
        const uint32_t tile = blockIdx.x + (it % mine) * gridDim.x, poly = tile / tpp, tin = tile % tpp;
        const uint32_t row0 = (poly / a.inner) * a.row_outer + (poly % a.inner) * a.row_inner, slot = it % nslots;
        mbar_expect_tx(&ctl->r_full[slot], slot_words * 4);
        tma_load_2d(ring + (size_t)slot * slot_words, &tmap, tin * TILE_M, row0, &ctl->r_full[slot]);
      };
      if (lw == 0 && lane == 0)
        for (uint32_t it = 0; it < nslots && it < total; ++it) issue(it);
      const uint32_t wph = ((a_cols + HALVES - 1) / HALVES + 7) / 8 * 8;
      const uint32_t w_lo = half * wph, w_hi = w_lo + wph < a_cols ? w_lo + wph : a_cols;
      const uint32_t lim = w_hi < a.nwords ? w_hi : a.nwords;
      for (; wi < total; ++wi) {
        const uint32_t slot = wi % nslots, ph = (wi / nslots) & 1, abuf = wi & amask;
        const uint32_t taddr = tmem_a + abuf * a_cols + ((quarter * 32u) << 16);
        const uint32_t* src = ring + (size_t)slot * slot_words + row;
        mbar_wait(&ctl->r_full[slot], ph);
        bool waited = false;
        for (uint32_t w0 = w_lo; w0 < w_hi; w0 += LR) {
          uint32_t w[LR];
#pragma unroll
          for (int i = 0; i < LR; ++i) w[i] = w0 + i < lim ? src[(w0 + i) * TILE_M] : 0u;   // warp-uniform predicate
          if (!waited) {
            mbar_wait(&ctl->a_free[abuf], ((wi >> ashift) & 1) ^ 1);
            tc_fence_after();
            waited = true;
          }
          if (mask_m && mask_w - w0 < (uint32_t)LR) {              // the batch holding the top word of a masked input
#pragma unroll
            for (int i = 0; i < LR; ++i)
              if (w0 + i == mask_w) w[i] &= mask_m;
          }
          store_batch<LR>(w, taddr, w0, w_hi);
        }
        if (!waited) mbar_wait(&ctl->a_free[abuf], ((wi >> ashift) & 1) ^ 1);
        tmem_st_wait();                                            // the registers (hence the slot) have been read
        tc_fence_before();
        if (lane == 0) { mbar_arrive(&ctl->a_full[abuf]); mbar_arrive(&ctl->r_free[slot]); }
        if (lw == 0 && lane == 0 && wi + nslots < total) {         // refill the slot once every loader warp is done with it
          mbar_wait(&ctl->r_free[slot], ph);
          issue(wi + nslots);
        }
        __syncwarp();
      }
    } else
    for (uint32_t ps = 0; ps < a.npass; ++ps) {
      for (uint32_t k = 0; k < mine; ++k, ++wi) {
        if (ALT && (wi & 1) != half) continue;
        const uint32_t tile = blockIdx.x + k * gridDim.x;
        const uint32_t poly = tile / tpp, tin = tile % tpp;
        const uint32_t po = poly / a.inner, pi = poly % a.inner;
        const uint32_t* p = a.src + (size_t)po * a.src_outer + (size_t)pi * a.src_inner + tin * TILE_M + row;
        const uint32_t abuf = wi & amask;
        const uint32_t taddr = tmem_a + abuf * a_cols + ((quarter * 32u) << 16);
        bool waited = false;
        // the warps of a lane quarter share the row: contiguous, equal ranges of its words (multiples of 8), LR at a time
        const uint32_t wph = ALT ? a_cols : ((a_cols + HALVES - 1) / HALVES + 7) / 8 * 8;
        const uint32_t w_lo = ALT ? 0 : half * wph, w_hi = w_lo + wph < a_cols ? w_lo + wph : a_cols;
        const uint32_t lim = w_hi < a.nwords ? w_hi : a.nwords;   // words of this warp's range that exist
        for (uint32_t w0 = w_lo; w0 < w_hi; w0 += LR) {
          uint32_t w[LR];
          const uint32_t* q = p + (size_t)w0 * a.N;
          if (w0 + LR <= lim) load_full<LR>(w, q, a.N);
          else load_tail<LR>(w, q, a.N, lim > w0 ? lim - w0 : 0u);
          if (!waited) {                                           // loads are in flight while the buffer is still being read
            mbar_wait(&ctl->a_free[abuf], ((wi >> ashift) & 1) ^ 1);
            tc_fence_after();
            waited = true;
          }
          if (mask_m && mask_w - w0 < (uint32_t)LR) {              // the batch holding the top word of a masked input
#pragma unroll
            for (int i = 0; i < LR; ++i)
              if (w0 + i == mask_w) w[i] &= mask_m;
          }
          store_batch<LR>(w, taddr, w0, w_hi);
        }
        if (!waited) mbar_wait(&ctl->a_free[abuf], ((wi >> ashift) & 1) ^ 1);   // a warp without batches still keeps in step
        tmem_st_wait();
        tc_fence_before();
        if (lane == 0) mbar_arrive(&ctl->a_full[abuf]);
      }
    }
  } else {
    // ===== epilogue =====
    const uint32_t grp = warp >> 2;
    const uint32_t etid = (warp & 3) * 32 + lane;                  // 0..127 = tile row = TMEM lane
    const uint32_t lane_off = ((warp & 3) * 32u) << 16;
    if constexpr (Epi::TILE_ALT) {
      // two groups, each a whole epilogue of its own on the tiles wi = grp (mod 2): own accumulator set, own scratch
      // region, own Epi object -- no state crosses between them.  With one set only (plan fallback) group 0 does it all.
      const uint32_t nset = a.nsets;
      if (grp < nset) {
        Epi epi(ep, a, smem + a.epi_off + grp * a.epi_stride, etid, 0, 1 + grp);
        const uint32_t tset = tmem_d + grp * a.cpp * NC;
        const uint32_t nc = a.nchunks;                             // single pass
        for (uint32_t wi = grp, use = 0; wi < mine; wi += nset, ++use) {
          const uint32_t tile = blockIdx.x + wi * gridDim.x;
          const uint32_t poly = tile / tpp, n0 = (tile % tpp) * TILE_M;
          epi.begin_tile(poly / a.inner, poly % a.inner, n0);
          for (uint32_t c = 0; c < nc; ++c) {
            if (c % SPAN == 0) {
              mbar_wait(&ctl->d_full[grp][c / SPAN], use & 1);
              tc_fence_after();
            }
            uint32_t t[64];
            tmem_ld32_nowait(tset + c * NC + lane_off, t);
            tmem_ld32_nowait(tset + c * NC + 32 + lane_off, t + 32);
            tmem_ld_wait();
            tc_fence_before();
            if (lane == 0) mbar_arrive(&ctl->d_free[grp][c]);     // the accumulator chunk is in registers: hand it back
            epi.consume(c * NC, t);
            epi.consume(c * NC + 32, t + 32);
          }
          epi.end_tile();
        }
      }
    } else if constexpr (Epi::CHUNK_ALT) {
      // Whole chunks in rotation: chunk c of work item wi belongs to group (c + wi) mod GROUPS, so the chunks of a span sit
      // with several groups at once and the span's accumulator columns are back with the MMA thread within one half chunk
      // of arithmetic.  mbarrier waits only see the phase parity, so a waiter must see every completion of its barrier:
      // "span finished" is signalled on barrier [wi mod GROUPS], and since ownership depends on wi only through wi mod
      // GROUPS, a group either waits on every completion of a given barrier or on none (parity (wi / GROUPS) & 1).  (With
      // one barrier, a group without a chunk in some work item took the completion of phase wi - 1 for that of wi + 1.)
      static_assert(GROUPS == 4 && SPAN == 4, "rotation laid out for four groups and spans of four chunks");
      Epi epi(ep, a, smem + a.epi_off, etid, grp, 1);
      uint32_t wi = 0;
      for (uint32_t ps = 0; ps < a.npass; ++ps) {
        const uint32_t c0 = ps * a.cpp;
        const uint32_t nc = a.nchunks - c0 < a.cpp ? a.nchunks - c0 : a.cpp;
        for (uint32_t k = 0; k < mine; ++k, ++wi) {
          const uint32_t tile = blockIdx.x + k * gridDim.x;
          const uint32_t poly = tile / tpp, n0 = (tile % tpp) * TILE_M;
          epi.begin_tile(poly / a.inner, poly % a.inner, n0);
          // spans hold GROUPS chunks, so a group owns at most one chunk per span
          for (uint32_t c = (grp + GROUPS - wi % GROUPS) % GROUPS; c < nc; c += GROUPS) {
            const uint32_t sp = c / SPAN;
            mbar_wait(&ctl->g_full[sp][wi % GROUPS], (wi / GROUPS) & 1);
            tc_fence_after();
            uint32_t t[32];
            tmem_ld32_nowait(tmem_d + c * NC + lane_off, t);
            tmem_ld_wait();
            epi.consume((c0 + c) * NC, t);
            tmem_ld32_nowait(tmem_d + c * NC + 32 + lane_off, t);
            tmem_ld_wait();
            tc_fence_before();
            if (lane == 0) mbar_arrive(&ctl->d_free[0][c]);        // the whole chunk has been read: hand it back
            epi.consume((c0 + c) * NC + 32, t);
          }
          epi.end_tile();
        }
      }
    } else {
    Epi epi(ep, a, smem + a.epi_off, etid, grp, 1);
    uint32_t wi = 0;
    for (uint32_t ps = 0; ps < a.npass; ++ps) {
      const uint32_t c0 = ps * a.cpp;
      const uint32_t nc = a.nchunks - c0 < a.cpp ? a.nchunks - c0 : a.cpp;
      for (uint32_t k = 0; k < mine; ++k, ++wi) {
        const uint32_t tile = blockIdx.x + k * gridDim.x;
        const uint32_t poly = tile / tpp, n0 = (tile % tpp) * TILE_M;
        epi.begin_tile(poly / a.inner, poly % a.inner, n0);
        for (uint32_t c = 0; c < nc; ++c) {
          if (c % SPAN == 0) {
            mbar_wait(&ctl->d_full[0][c / SPAN], wi & 1);
            tc_fence_after();
          }
          if constexpr (GROUPS == 1) {
            uint32_t t[64];
            tmem_ld32_nowait(tmem_d + c * NC + lane_off, t);
            tmem_ld32_nowait(tmem_d + c * NC + 32 + lane_off, t + 32);
            tmem_ld_wait();
            tc_fence_before();
            if (lane == 0) mbar_arrive(&ctl->d_free[0][c]);        // the accumulator chunk is in registers: hand it back
            epi.consume((c0 + c) * NC, t);
            epi.consume((c0 + c) * NC + 32, t + 32);
          } else {
            uint32_t t[GC];
            tmem_ld_cols<GC>(tmem_d + c * NC + grp * GC + lane_off, t);
            tmem_ld_wait();
            tc_fence_before();
            if (lane == 0) mbar_arrive(&ctl->d_free[0][c]);
            epi.consume((c0 + c) * NC + grp * GC, t);
          }
        }
        epi.end_tile();
      }
    }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == MMAW) tmem_dealloc(tmem_a, a.tmem_cols);
}

template <class Epi>
inline cudaError_t launch_pipe(const PipeArgs& a_in, const typename Epi::Params& ep, size_t smem, int n_sm, cudaStream_t s,
                               const CUtensorMap* tmap = nullptr) {
  // the attribute belongs to the (kernel, device) pair: one high-water mark per device
  constexpr int MAX_DEV = 64;
  static size_t configured[MAX_DEV] = {};
  int dev = 0;
  cudaError_t e0 = cudaGetDevice(&dev);
  if (e0 != cudaSuccess) return e0;
  if (dev < 0 || dev >= MAX_DEV || smem > configured[dev]) {
    cudaError_t e = cudaFuncSetAttribute(pipe_kernel<Epi>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    if (dev >= 0 && dev < MAX_DEV) configured[dev] = smem;
  }
  PipeArgs a = a_in;
  CUtensorMap tm;
  if (tmap) tm = *tmap; else { memset(&tm, 0, sizeof(tm)); a.ring_slots = 0; }
  const uint32_t ntiles = a.npoly * (a.N / TILE_M);
  const uint32_t grid = ntiles < (uint32_t)n_sm ? ntiles : (uint32_t)n_sm;
  const cudaError_t e = launch_pdl(pipe_kernel<Epi>, grid, nthreads(Epi::GROUPS, Epi::LOAD_WARPS), smem, s, a, ep, tm);
  return e != cudaSuccess ? e : cudaGetLastError();
}
#endif  // __CUDACC__

}  // namespace pipe
}  // namespace fhe
