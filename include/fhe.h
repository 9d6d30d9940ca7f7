/* fhe.h -- C ABI of the B200-native non-RNS CKKS/BGV hot path (arxiv/paper_2607_05920, "LibFHE").
 *
 * One thing is exported: exact negacyclic multiplication of polynomials with multi-limb coefficients in
 * Z_Q[X]/(X^N+1) (Eq. 5-6) through the paper's limb -> RNS -> NTT -> pointwise -> iNTT ->
 * CRT -> limb pipeline, wrapped as the homomorphic hot path
 * mult (tensor product + relinearisation) and rescale.
 * Readings of everything the paper leaves open are listed in DESIGN.md section 3.
 *
 * Conventions (all entry points)
 *   - "d_" pointers are DEVICE memory owned by the caller, 16-byte aligned, contiguous.  "h_" pointers are HOST memory.
 *   - A polynomial is a uint32 array [L][N]: limb index before coefficient index, limb 0 least significant
 *     (radix representation X = sum_i x_i 2^(32 i), Eq. 22-23).  L = ceil(bits(Q)/32).
 *   - A ciphertext is [2][L][N] = (c0, c1) with decryption c0 + c1*s; a tensor triple is [3][L][N] = (d0, d1, d2)
 *     with decryption d0 + d1*s + d2*s^2.  A batch is the outermost dimension (the paper's `cnum`).
 *   - Outputs are canonical representatives in [0, Q) with unused top-limb bits zero.  CKKS inputs are taken
 *     mod 2^logQ (bits above logQ are ignored).  BGV inputs must already be < Q (precondition, not checked).
 *   - Hot-path calls allocate nothing, enqueue on the caller's stream (a cudaStream_t passed as void*; NULL = the
 *     legacy default stream), never synchronise and never touch host copies of data.  Outputs must not alias
 *     inputs or the workspace.  The workspace is caller-supplied device memory of at least
 *     fhe_workspace_bytes(ctx, op, batch) bytes, 256-byte aligned.
 *   - Errors are return codes only: no exceptions, no abort, nothing printed.  Argument errors are detected
 *     before anything is launched.  fhe_last_error(ctx) returns a static or ctx-owned string for the last failure.
 *   - A context is not thread-safe; use one per host thread / stream.
 */
#ifndef FHE_H_
#define FHE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fhe_ctx fhe_ctx; /* opaque: owns prime/twiddle/CRT tables (device) and the transformed evk */

typedef enum {
  FHE_OK = 0,
  FHE_ERR_ARG = 1,         /* NULL pointer, misaligned pointer, bad size, batch == 0 handled as OK no-op */
  FHE_ERR_UNSUPPORTED = 2, /* parameter combination the library does not implement; also returned by fhe_he_mult /
                              fhe_relinearize / fhe_mult_relin_rescale when that call's CRT target (constant matrix in
                              shared memory, accumulators in tensor memory) does not fit the SM while fhe_polymul's does */
  FHE_ERR_STATE = 3,       /* e.g. fhe_relinearize before fhe_set_evk */
  FHE_ERR_CUDA = 4,        /* a CUDA runtime call failed; text in fhe_last_error */
  FHE_ERR_NOMEM = 5        /* host or device allocation failed, or workspace too small */
} fhe_status;

typedef enum {            /* `op` argument of fhe_workspace_bytes */
  FHE_OP_POLYMUL = 0,
  FHE_OP_HE_MULT = 1,
  FHE_OP_RELINEARIZE = 2,
  FHE_OP_RESCALE = 3,     /* needs no workspace: returns 0 */
  FHE_OP_MULT_RELIN_RESCALE = 4,
  FHE_OP_SET_EVK = 5,
  FHE_OP_ROTATE = 6,
  FHE_OP_MULT_PLAIN = 7
} fhe_op;

typedef struct {
  uint32_t N;        /* ring degree */
  uint32_t logQ;     /* as given to fhe_ctx_create */
  uint32_t logP;
  uint64_t t;        /* 0 = CKKS, else BGV plaintext modulus */
  uint32_t bitsQ;    /* bit length of Q-1 (CKKS: logQ; BGV: logQ+1) */
  uint32_t bitsPQ;   /* bit length of P*Q-1 */
  uint32_t L;        /* uint32 limbs per coefficient mod Q */
  uint32_t L_PQ;     /* uint32 limbs per coefficient mod P*Q (the evk) */
  uint32_t K_pm;     /* NTT primes used by fhe_polymul   (product > 4*N*Q^2, see DESIGN.md 3-A5) */
  uint32_t K1;       /* NTT primes used by fhe_he_mult   (product > 8*N*Q^2) */
  uint32_t K2;       /* NTT primes used by fhe_relinearize (product > 4*N*Q*PQ) */
  uint32_t n_sm;     /* SM count of the device the context lives on */
} fhe_info;

/* Create a context on the current CUDA device.
 *   t == 0 : CKKS, Q = 2^logQ, P = 2^logP
 *   t  > 0 : BGV, t odd and < 2^31; Q = least odd integer > 2^logQ with Q = 1 (mod t), P likewise from logP
 *            (so logP == logQ gives P == Q)                                 (DESIGN.md 3-A10, A11)
 *   N a power of two, 2^8 <= N <= 2^16; 32 <= logQ; logQ, logP <= 2560.
 * Precomputes on the host and uploads: the NTT primes (30-bit, = 1 mod 2^17), psi/psi^-1 power
 * tables with Shoup companions, 2^(26 d) mod q_j and the CRT constants
 * (this build uses the direct form of Eq. 1).  Synchronises. */
fhe_status fhe_ctx_create(fhe_ctx** out, uint32_t N, uint32_t logQ, uint32_t logP, uint64_t t);
void fhe_ctx_destroy(fhe_ctx* ctx);
fhe_status fhe_ctx_info(const fhe_ctx* ctx, fhe_info* out);
const char* fhe_last_error(const fhe_ctx* ctx); /* ctx may be NULL: returns the last create-time error */

/* Copy Q (which = 0) or P (1) or P*Q (2) to h_limbs as little-endian uint32 limbs; n_limbs must be >= the
 * limb count of the value (L, L_P, L_PQ+1 suffices).  Extra limbs are zeroed.  Host-only helper for callers. */
fhe_status fhe_get_modulus(const fhe_ctx* ctx, int which, uint32_t* h_limbs, uint32_t n_limbs);

/* Bytes of device workspace the op needs for `batch` items (0 if none). */
size_t fhe_workspace_bytes(const fhe_ctx* ctx, int op, uint32_t batch);

/* Install the relinearisation key evk = (b', a') mod P*Q, d_evk = [2][L_PQ][N] (DESIGN.md 3-A2: b' = -a's + e'
 * + P s^2, resp. + t e' for BGV).  Decomposes it into the K2 relin primes and stores its forward NTT
 * ("evk-hat", [2][K2][N]) inside the context (device allocation on first call).  Once per key; enqueued on
 * `stream`; d_evk may be freed after the stream reaches this point.  d_ws: FHE_OP_SET_EVK bytes. */
fhe_status fhe_set_evk(fhe_ctx* ctx, const uint32_t* d_evk, void* d_ws, size_t ws_bytes, void* stream);

/* out[i] = a[i] * b[i] in Z_Q[X]/(X^N+1), i < batch.  d_out, d_a, d_b: [batch][L][N]. */
fhe_status fhe_polymul(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t batch,
                       void* d_ws, size_t ws_bytes, void* stream);

/* fhe_polymul for callers that cannot allocate device memory (code under CUDA graph capture, tight serving loops, harnesses
 * that forbid cudaMalloc): the same ring product with the intermediate residue matrix in a
 * 32 MiB device array that is part of the library image -- every GPU that loads the library holds it until the process
 * exits -- instead of a caller workspace.  d_out, d_a, d_b: [batch][L][N], caller-owned, as for fhe_polymul; enqueued on
 * `stream`; no cudaMalloc / cudaFree / allocating routine is called.  A batch whose fhe_workspace_bytes(FHE_OP_POLYMUL)
 * exceeds fhe_static_scratch_bytes() is rejected with FHE_ERR_NOMEM (text in fhe_last_error): use fhe_polymul then.
 * All calls on a device SHARE the array and find the previous call's contents in it (nothing in it needs clearing: the
 * decompose writes every word the later kernels read); calls that overlap on the GPU -- other streams, concurrent graph
 * launches -- race on it and must be ordered by the caller.
 * fhe_polymul_static_init looks up the array's device address (cudaGetSymbolAddress, once per device, with the context's
 * device current); fhe_polymul_static does the same on its first call, so calling init first is only needed to keep that
 * lookup out of a graph capture. */
size_t fhe_static_scratch_bytes(void);
fhe_status fhe_polymul_static_init(fhe_ctx* ctx);
fhe_status fhe_polymul_static(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t batch,
                              void* stream);

/* Tensor product (north_star item 4): d0 = c0 c0', d1 = c0 c1' + c1 c0', d2 = c1 c1' (mod Q).
 * d_out3: [batch][3][L][N]; d_ct1, d_ct2: [batch][2][L][N]. */
fhe_status fhe_he_mult(fhe_ctx* ctx, uint32_t* d_out3, const uint32_t* d_ct1, const uint32_t* d_ct2,
                       uint32_t batch, void* d_ws, size_t ws_bytes, void* stream);

/* Relinearisation (formulas DESIGN.md 3-A2..A4, A10): with x_b = d2*b', x_a = d2*a' in [0, PQ),
 *   CKKS: k = ((x + 2^(logP-1)) >> logP) mod Q
 *   BGV : r = x mod P centred, kk = (-r P^-1) mod t centred, k = ((x - r)/P - kk) mod Q
 * out = ((d0 + k_b) mod Q, (d1 + k_a) mod Q).  d_out2: [batch][2][L][N]; d_in3: [batch][3][L][N].
 * FHE_ERR_STATE if no evk is installed. */
fhe_status fhe_relinearize(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in3, uint32_t batch, void* d_ws,
                           size_t ws_bytes, void* stream);

/* CKKS rescale by 2^p (DESIGN.md 3-A3): c' = ((c + 2^(p-1)) >> p) mod 2^(logQ-p) on the
 * canonical c, every component.  d_out2, d_in2: [batch][2][L][N] (same L-limb stride; top bits zero).
 * 1 <= p_bits < logQ.  FHE_ERR_UNSUPPORTED on a BGV context.  In-place (d_out2 == d_in2) is allowed here. */
fhe_status fhe_rescale(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in2, uint32_t p_bits, uint32_t batch,
                       void* stream);

/* Convenience for the headline metric: he_mult -> relinearize -> rescale (p_bits == 0: no rescale; BGV requires 0)
 * without materialising d0/d1/d2 for the caller.  Result identical to the three calls in sequence. */
fhe_status fhe_mult_relin_rescale(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct1, const uint32_t* d_ct2,
                                  uint32_t p_bits, uint32_t batch, void* d_ws, size_t ws_bytes, void* stream);

/* Same computation as fhe_mult_relin_rescale with HOST buffers (pageable or pinned; pinned for full PCIe speed):
 * copies the inputs to the device, runs, copies the result back and returns when h_out2 is complete (`stream` and the
 * context's two copy streams are synchronised).  Batch items are independent, so the call is pipelined item by item:
 * the host->device copy of item i + 1, the kernels of item i (on `stream`) and the device->host copy of item i - 1
 * overlap.  d_ws must additionally hold the device copies: fhe_workspace_bytes(op) + 3 ciphertext batches.  Used for
 * the end-to-end ("e2e") measurement. */
fhe_status fhe_mult_relin_rescale_host(fhe_ctx* ctx, uint32_t* h_out2, const uint32_t* h_ct1, const uint32_t* h_ct2,
                                       uint32_t p_bits, uint32_t batch, void* d_ws, size_t ws_bytes, void* stream);

/* ---- NEXT-1: coefficient-wise ciphertext operations and the level drop -------------------------------
 * The paper lists them by name (add_pairwise_into, sub_pairwise_into, negate_pairwise_into, PAPER.md:654-662;
 * moddownBy_pairwise_into).  Polynomials are limb-major [L][N], `npoly` of them back to back (a batch of B
 * ciphertexts is 2 B polynomials); inputs canonical in [0, Q), outputs canonical.  In place (d_out == d_a) is allowed.
 *   fhe_add / fhe_sub / fhe_negate   (a + b) mod Q, (a - b) mod Q, (-a) mod Q, CKKS (Q = 2^logQ) and BGV (odd Q).
 *   fhe_moddown                      CKKS only: every coefficient mod 2^new_logq, 1 <= new_logq <= logQ, same L-limb stride
 *                                    (the limbs above new_logq are written as zero).  A ciphertext at the lower level is
 *                                    then used with a context created for logQ = new_logq (its evk is the original one
 *                                    reduced mod 2^(logP + new_logq): fhe_set_evk masks on load when given L_PQ' limbs). */
fhe_status fhe_add(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly, void* stream);
fhe_status fhe_sub(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly, void* stream);
fhe_status fhe_negate(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, uint32_t npoly, void* stream);
fhe_status fhe_moddown(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logq, uint32_t npoly, void* stream);
/* out = X^k * in mod (X^N + 1, Q), 0 <= k < 2N, per polynomial: a signed rotation of the coefficients.  k = N/2 multiplies
 * the CKKS slots by the imaginary unit (imult_pairwise_into), k = 3N/2 by -i.  NOT in place. */
fhe_status fhe_mul_monomial(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t k, uint32_t npoly, void* stream);

/* ---- NEXT-2: slot rotation and conjugation ------------------------------------
 * A rotation is the Galois automorphism X -> X^k (k odd, k < 2N; k = 2N - 1 conjugates) applied to both components,
 * followed by a key switch from sigma_k(s) back to s: out = (sigma(c0) + kb, ka), (kb, ka) = round(sigma(c1) * rk / P)
 * with the same divide-by-P rule as fhe_relinearize (A2/A3/A10) and a key of the same form as the evk,
 * rk = (b', a') mod PQ, b' = -a' s + e' + P sigma_k(s) (BGV: t e').
 *   fhe_set_rotation_key   installs the key for Galois element k in `slot` (0..15): decompose + forward NTT, once per key;
 *                          d_key [2][L_PQ][N] as for fhe_set_evk.
 *   fhe_rotate             d_in2, d_out2 [B][2][L][N]; d_ws >= fhe_workspace_bytes(FHE_OP_ROTATE, batch).
 *                          FHE_ERR_STATE when the slot holds no key. */
fhe_status fhe_set_rotation_key(fhe_ctx* ctx, uint32_t slot, uint32_t k, const uint32_t* d_key, void* stream);
fhe_status fhe_rotate(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in2, uint32_t slot, uint32_t batch, void* d_ws,
                      size_t ws_bytes, void* stream);

/* ---- NEXT-3: ciphertext x plaintext, pairwise and broadcast -----------------
 * out[i] = (c0_i * m_j, c1_i * m_j) mod (X^N + 1, Q) with j = i / group: group = 1 multiplies ciphertext i by its own
 * plaintext polynomial (multconstvec_pairwise), group = batch lifts ONE plaintext over the whole tensor
 * (multconst_broadcast).  d_ct, d_out2 [B][2][L][N]; d_pt [ceil(B / group)][L][N], an ENCODED plaintext (the caller rescales
 * afterwards as after any multiplication); d_ws >= fhe_workspace_bytes(FHE_OP_MULT_PLAIN, batch).  The shared operand is
 * decomposed and column-transformed once per plaintext; the same kernels as fhe_polymul do the rest. */
fhe_status fhe_mult_plain(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                          uint32_t group, void* d_ws, size_t ws_bytes, void* stream);

/* ---- NEXT-3, constants (addconst / multconst with a scalar: names only; reading in DESIGN.md 3) ------
 *   fhe_add_plain     out[i] = (c0_i + m_j, c1_i) mod Q, j = i / group (group = 1: pairwise, group = batch: broadcast).
 *                     d_ct, d_out2 [B][2][L][N]; d_pt [ceil(B / group)][L][N] canonical in [0, Q).  In place
 *                     (d_out2 == d_ct) is allowed.  CKKS and BGV.
 *   fhe_mult_scalar   every coefficient of `npoly` polynomials [L][N] times the integer k mod Q, |k| < 2^31 (k = INT32_MIN is
 *                     FHE_ERR_ARG); in place allowed.  CKKS and BGV (BGV: FHE_ERR_UNSUPPORTED when logQ < 66, where the
 *                     single-word quotient estimate does not hold).
 * One streaming kernel each, a thread per coefficient; no workspace. */
fhe_status fhe_add_plain(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                         uint32_t group, void* stream);
fhe_status fhe_mult_scalar(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, int32_t k, uint32_t npoly, void* stream);

/* ---- NEXT-4: BGV modulus switching (named only; reading DESIGN.md 3, A20) ---------------
 * Every coefficient c in [0, Q) of `npoly` polynomials [L][N] becomes c' in [0, Q'), Q' = the modulus of the same construction
 * above 2^new_logQ (least odd integer that is 1 mod t):  x = c Q',  r = x mod Q centred,  k = (-r Q^-1) mod t centred,
 * c' = ((x - r)/Q - k) mod Q'  -- the integer nearest to c Q'/Q that keeps the plaintext exact, the noise shrinks by Q'/Q.
 * Output in the same L-limb stride (limbs above Q' are zero); a ciphertext at the lower level is then used with a context
 * created for logQ = new_logQ.  In place allowed.  BGV only (FHE_ERR_UNSUPPORTED on CKKS, and when logQ < 96 or
 * new_logQ < 34, where the kernel's shortcuts for Q = 2^logQ + e do not hold); 34 <= new_logQ < logQ. */
fhe_status fhe_modswitch(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logQ, uint32_t npoly, void* stream);

/* ---- debug / unit-parity entry points (same kernels as the hot path, one step at a time) ------------------- */

/* Host copies of the first `count` NTT primes and the primitive 2N-th roots psi_j the tables were built from. */
fhe_status fhe_debug_primes(const fhe_ctx* ctx, uint32_t* h_q, uint32_t* h_psi, uint32_t count);
/* S1: d_res [npoly][K][N] = residues of d_limbs [npoly][Lin][N] mod the first K primes.
 * mask_bits > 0: the input is first reduced mod 2^mask_bits (CKKS load masking). */
fhe_status fhe_debug_decompose(fhe_ctx* ctx, uint32_t* d_res, const uint32_t* d_limbs, uint32_t npoly, uint32_t Lin,
                               uint32_t K, uint32_t mask_bits, void* stream);
/* S2 / S4 (Eq. 8-9) in place on d_res [npoly][K][N].  Forward output is in bit-reversed index
 * order: res[bitrev(i)] = sum_j a_j psi^((2i+1) j).  inverse != 0: expects that order, returns natural order,
 * scaled by N^-1 only (no CRT constant folded in). */
fhe_status fhe_debug_ntt(fhe_ctx* ctx, uint32_t* d_res, uint32_t npoly, uint32_t K, int inverse, void* stream);
/* The CKKS relinearisation CRT decides the one carry out of the low logP bits of x from 96-bit truncated constants and
 * recomputes a coefficient exactly when the `bits` fractional bits below the rounding position are all ones (default
 * and maximum 58: the truncation error is below 2^-58, so nothing else can be wrong).  A smaller value
 * only sends more coefficients down the exact path -- results are identical -- which is how the tests reach it. */
fhe_status fhe_debug_crt_ambiguity(fhe_ctx* ctx, uint32_t bits);
/* Path selection by shape.  Small conversions (K <= 32 primes, <= 16 limbs, K x limbs <= 192) run on the CUDA cores, one
 * thread per pair of coefficients, because a tile of the tensor-core pipeline costs more than it moves there; N = 2^12 runs every
 * product's transforms in ONE kernel (whole prime-polynomial in shared memory), larger N in three passes.  mode 0: that
 * choice (by measurement); 1: the large-shape paths everywhere (tensor-core conversions, three-pass NTT); 2: the small-shape
 * paths wherever they exist (the whole-transform NTT also at N = 2^13, where the three passes measure 8-13 % faster).
 * Results are identical in every mode -- this is how the tests cover each path at the shapes where it is not the default. */
fhe_status fhe_debug_force_pipeline(fhe_ctx* ctx, int mode);
/* Calibration for the roofline report: register-only throughput, in operations per second over the
 * whole device, of mode 0: the forward NTT butterfly exactly as the kernels execute it (Eq. 8: one
 * Shoup modular multiplication, one add, one subtract, lazy corrections); 1: mad.lo.u32; 2: mul.hi.u32.  Allocates
 * a scratch buffer, launches a few milliseconds of work on `stream` and synchronises: not a hot-path call. */
fhe_status fhe_debug_int_peak(fhe_ctx* ctx, int mode, double* per_second, void* stream);
/* Number of kernel launches the context has enqueued so far (for bench.py's gpu_launches). */
uint64_t fhe_debug_launch_count(const fhe_ctx* ctx);
/* Per-kernel device timing for the roofline report.  enable != 0: every later launch is bracketed by a CUDA event
 * pair on its stream (the only case in which a hot-path call creates anything); enable == 0: off, events freed.
 * fhe_debug_timing_read synchronises on the recorded events and returns the summed duration and launch count of one
 * kernel class: 0 decompose, 1 forward NTT, 2 inverse NTT, 3 pointwise, 4 CRT(+post), 5 rescale. */
fhe_status fhe_debug_timing(fhe_ctx* ctx, int enable);
fhe_status fhe_debug_timing_read(fhe_ctx* ctx, int kernel_class, double* ms_total, uint64_t* launches);

#ifdef __cplusplus
}
#endif
#endif /* FHE_H_ */
