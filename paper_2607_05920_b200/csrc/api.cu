// api.cu -- the hot-path entry points: argument checks, then kernel launches on the caller's stream.  No allocation,
// no synchronisation, no host copies (except the explicit *_host end-to-end variant).
#include "fhe_internal.cuh"

using namespace fhe;

namespace {

inline Context* C(fhe_ctx* p) { return reinterpret_cast<Context*>(p); }
inline const Context* C(const fhe_ctx* p) { return reinterpret_cast<const Context*>(p); }
inline bool misaligned(const void* p, size_t a) { return (reinterpret_cast<uintptr_t>(p) & (a - 1)) != 0; }

fhe_status err(Context* c, fhe_status st, const char* msg) { c->err = msg; return st; }
fhe_status cuda_fail(Context* c, cudaError_t e, const char* where) {
  c->err = std::string(where) + ": " + cudaGetErrorString(e);
  return FHE_ERR_CUDA;
}
// Tables, keys, copy streams and the launch configuration all belong to the device the context was created on.
fhe_status check_device(Context* c) {
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess || d != c->device) return err(c, FHE_ERR_STATE, "the context's CUDA device is not the current device");
  return FHE_OK;
}
#define CK(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) return cuda_fail(c, e_, where); } while (0)

inline size_t align256(size_t x) { return (x + 255) & ~(size_t)255; }

size_t ws_polymul(const Context* c, uint32_t b) { return align256((size_t)b * 2 * c->K_pm * c->N * 4); }
size_t ws_tensor(const Context* c, uint32_t b) { return align256((size_t)b * 4 * c->K1 * c->N * 4); }
// residues [B][2][K2][N], then the flag bitmap of the exact CRT path, one bit per output coefficient (kernels_crt.cu)
size_t ws_relin_res(const Context* c, uint32_t b) { return align256((size_t)b * 2 * c->K2 * c->N * 4); }
size_t ws_relin(const Context* c, uint32_t b) { return ws_relin_res(c, b) + align256((size_t)b * 2 * (c->N / 32) * 4); }
size_t ws_d3(const Context* c, uint32_t b) { return align256((size_t)b * 3 * c->L * c->N * 4); }
size_t ws_evk(const Context* c) { return 0; }   // evk-hat is transformed in place inside the context

// he_mult core: ct1, ct2 [B][2][L][N] -> out3 [B][3][L][N]; ws: [B][4][K1][N]
fhe_status do_he_mult(Context* c, uint32_t* d_out3, const uint32_t* d_ct1, const uint32_t* d_ct2, uint32_t B,
                      uint32_t* ws, cudaStream_t s) {
  const uint32_t N = c->N, L = c->L, K = c->K1;
  const size_t rp = (size_t)K * N;           // residue poly stride
  const uint32_t mask = c->t == 0 ? c->logQ : 0;
  // slots (a0, a1, b0, b1) per batch item: ct1 polys go to slots 0,1 ; ct2 polys to slots 2,3
  CK(launch_decompose(c, ws, 4 * rp, rp, d_ct1, (size_t)2 * L * N, (size_t)L * N, B, 2, L, K, mask, s), "decompose ct1");
  // the second factor carries the final constant of the inverse transforms (scaled decompose image, fhe_internal.cuh)
  CK(launch_decompose(c, ws + 2 * rp, 4 * rp, rp, d_ct2, (size_t)2 * L * N, (size_t)L * N, B, 2, L, K, mask, s, true, &c->tgt_tensor), "decompose ct2");
  // forward columns, fused rows (tensor product in registers), inverse columns: slots 0..2 <- INTT(d0^, d1^, d2^)
  CK(launch_ntt_product(c, ws, nullptr, B, K, PW_TENSOR, s), "ntt tensor");
  CK(launch_crt(c, c->tgt_tensor, c->post_tensor, d_out3, (size_t)3 * L * N, (size_t)L * N, ws, 4 * rp, rp, nullptr, 0, 0,
                B, 3, s), "crt");
  return FHE_OK;
}

// relin core: in3 [B][3][L][N] -> out2 [B][2][L][N]; ws: [B][2][K2][N]; rescale_bits fused into the CRT epilogue
fhe_status do_relin(Context* c, uint32_t* d_out2, const uint32_t* d_in3, uint32_t B, uint32_t* ws, uint32_t rescale_bits,
                    cudaStream_t s, const uint32_t* d_key_hat = nullptr) {
  if (!d_key_hat) d_key_hat = c->d_evk_hat;
  const uint32_t N = c->N, L = c->L, K = c->K2;
  const size_t rp = (size_t)K * N;
  const uint32_t mask = c->t == 0 ? c->logQ : 0;
  CK(launch_decompose(c, ws, 2 * rp, 0, d_in3 + (size_t)2 * L * N, (size_t)3 * L * N, 0, B, 1, L, K, mask, s), "decompose d2");
  CK(launch_ntt_product(c, ws, const_cast<uint32_t*>(d_key_hat), B, K, PW_RELIN, s), "ntt relin");   // the key carries the final constant
  PostParams pp = c->post_relin;
  pp.rescale_bits = rescale_bits;
  pp.amb_bits = c->amb_bits;
  uint32_t* flags = (uint32_t*)((char*)ws + ws_relin_res(c, B));
  CK(launch_crt(c, c->tgt_relin, pp, d_out2, (size_t)2 * L * N, (size_t)L * N, ws, 2 * rp, rp, d_in3, (size_t)3 * L * N,
                (size_t)L * N, B, 2, s, flags), "crt relin");
  return FHE_OK;
}

}  // namespace

extern "C" {

size_t fhe_workspace_bytes(const fhe_ctx* ctx, int op, uint32_t batch) {
  if (!ctx) return 0;
  const Context* c = C(ctx);
  switch (op) {
    case FHE_OP_POLYMUL: return ws_polymul(c, batch);
    case FHE_OP_HE_MULT: return ws_tensor(c, batch);
    case FHE_OP_RELINEARIZE: return ws_relin(c, batch);
    case FHE_OP_RESCALE: return 0;
    case FHE_OP_MULT_RELIN_RESCALE: {
      size_t a = ws_tensor(c, batch), b = ws_relin(c, batch);
      return (a > b ? a : b) + ws_d3(c, batch);
    }
    case FHE_OP_SET_EVK: return ws_evk(c);
    case FHE_OP_ROTATE: return ws_relin(c, batch) + ws_d3(c, batch);
    case FHE_OP_MULT_PLAIN: return ws_polymul(c, 2 * batch);
    default: return 0;
  }
}

// decompose + forward NTT of a key (b', a') mod PQ into *slot ([2][K2][N], allocated on first use)
static fhe_status install_key(Context* c, uint32_t** slot, const uint32_t* d_key, cudaStream_t s) {
  const size_t bytes = (size_t)2 * c->K2 * c->N * 4;
  if (!*slot) {
    void* p = nullptr;
    if (cudaMalloc(&p, bytes) != cudaSuccess) { cudaGetLastError(); return err(c, FHE_ERR_NOMEM, "key allocation failed"); }
    *slot = (uint32_t*)p;
  }
  const uint32_t mask = c->t == 0 ? c->logQ + c->logP : 0;
  CK(launch_decompose(c, *slot, 0, (size_t)c->K2 * c->N, d_key, 0, (size_t)c->L_PQ * c->N, 1, 2, c->L_PQ, c->K2, mask, s), "decompose key");
  CK(launch_ntt_fwd(c, *slot, 1, 2, 2, c->K2, s), "ntt key");
  CK(launch_scale_rows(c, *slot, 2, c->K2, c->tgt_relin.d_scale, s), "scale key");   // the key carries the relin products' final constant
  return FHE_OK;
}

fhe_status fhe_set_evk(fhe_ctx* ctx, const uint32_t* d_evk, void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  (void)d_ws; (void)ws_bytes;
  if (!d_evk || misaligned(d_evk, 16)) return err(c, FHE_ERR_ARG, "d_evk NULL or misaligned");
  c->have_evk = false;
  fhe_status st = install_key(c, &c->d_evk_hat, d_evk, (cudaStream_t)stream);
  if (st != FHE_OK) return st;
  c->have_evk = true;
  return FHE_OK;
}

fhe_status fhe_set_rotation_key(fhe_ctx* ctx, uint32_t slot, uint32_t k, const uint32_t* d_key, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (slot >= (uint32_t)Context::MAX_ROT_KEYS) return err(c, FHE_ERR_ARG, "key slot out of range");
  if (!(k & 1) || k >= 2 * c->N) return err(c, FHE_ERR_ARG, "Galois element must be odd and below 2N");
  if (!d_key || misaligned(d_key, 16)) return err(c, FHE_ERR_ARG, "d_key NULL or misaligned");
  c->rot_k[slot] = 0;
  fhe_status st = install_key(c, &c->d_rot_hat[slot], d_key, (cudaStream_t)stream);
  if (st != FHE_OK) return st;
  c->rot_k[slot] = k;
  return FHE_OK;
}

fhe_status fhe_rotate(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in2, uint32_t slot, uint32_t batch, void* d_ws,
                      size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_in2 || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_in2, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (slot >= (uint32_t)Context::MAX_ROT_KEYS || !c->rot_k[slot]) return err(c, FHE_ERR_STATE, "no rotation key in this slot");
  if (c->N < 256) return err(c, FHE_ERR_UNSUPPORTED, "N < 256");
  if (!c->fit_relin) return err(c, FHE_ERR_UNSUPPORTED, "relinearisation CRT target too large for the conversion pipeline");
  if (ws_bytes < ws_relin(c, batch) + ws_d3(c, batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  cudaStream_t s = (cudaStream_t)stream;
  uint32_t* d3 = (uint32_t*)d_ws;
  uint32_t* ws = (uint32_t*)((char*)d_ws + ws_d3(c, batch));
  CK(launch_automorphism(c, d3, d_in2, c->rot_k[slot], batch, s), "automorphism");
  return do_relin(c, d_out2, d3, batch, ws, 0, s, c->d_rot_hat[slot]);
}

// out[i] = a[i] * b[i / group] mod (X^N + 1, Q) for i < npoly; ws: [npoly + ceil(npoly / group)][K_pm][N]
static fhe_status do_polymul(Context* c, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly,
                             uint32_t group, uint32_t* ws, cudaStream_t s) {
  const uint32_t N = c->N, L = c->L, K = c->K_pm, nb = (npoly + group - 1) / group;
  const size_t rp = (size_t)K * N;
  uint32_t* ra = ws;
  uint32_t* rb = ra + (size_t)npoly * rp;
  const uint32_t mask = c->t == 0 ? c->logQ : 0;
  CK(launch_decompose(c, ra, 0, rp, d_a, 0, (size_t)L * N, 1, npoly, L, K, mask, s), "decompose a");
  CK(launch_decompose(c, rb, 0, rp, d_b, 0, (size_t)L * N, 1, nb, L, K, mask, s, true, &c->tgt_pm), "decompose b");   // carries the final constant
  CK(launch_ntt_product(c, ra, rb, npoly, K, PW_POLYMUL, s, group), "ntt polymul");
  CK(launch_crt(c, c->tgt_pm, c->post_pm, d_out, 0, (size_t)L * N, ra, 0, rp, nullptr, 0, 0, 1, npoly, s), "crt");
  return FHE_OK;
}

fhe_status fhe_polymul(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t batch,
                       void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out || !d_a || !d_b || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out, 16) || misaligned(d_a, 16) || misaligned(d_b, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (ws_bytes < ws_polymul(c, batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  return do_polymul(c, d_out, d_a, d_b, batch, 1, (uint32_t*)d_ws, (cudaStream_t)stream);
}

fhe_status fhe_mult_plain(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                          uint32_t group, void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_ct || !d_pt || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_ct, 16) || misaligned(d_pt, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (group == 0) return err(c, FHE_ERR_ARG, "group must be at least 1");
  if (ws_bytes < ws_polymul(c, 2 * batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  // both components of ciphertext i times plaintext i / group: 2 batch polynomials, operand shared by 2 group of them
  return do_polymul(c, d_out2, d_ct, d_pt, 2 * batch, 2 * group, (uint32_t*)d_ws, (cudaStream_t)stream);
}

fhe_status fhe_he_mult(fhe_ctx* ctx, uint32_t* d_out3, const uint32_t* d_ct1, const uint32_t* d_ct2, uint32_t batch,
                       void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out3 || !d_ct1 || !d_ct2 || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out3, 16) || misaligned(d_ct1, 16) || misaligned(d_ct2, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (ws_bytes < ws_tensor(c, batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  if (!c->fit_tensor) return err(c, FHE_ERR_UNSUPPORTED, "tensor-product CRT target too large for the conversion pipeline");
  return do_he_mult(c, d_out3, d_ct1, d_ct2, batch, (uint32_t*)d_ws, (cudaStream_t)stream);
}

fhe_status fhe_relinearize(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in3, uint32_t batch, void* d_ws,
                           size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_in3 || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_in3, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (!c->have_evk) return err(c, FHE_ERR_STATE, "no evk installed (call fhe_set_evk first)");
  if (ws_bytes < ws_relin(c, batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  if (!c->fit_relin) return err(c, FHE_ERR_UNSUPPORTED, "relinearisation CRT target too large for the conversion pipeline");
  return do_relin(c, d_out2, d_in3, batch, (uint32_t*)d_ws, 0, (cudaStream_t)stream);
}

fhe_status fhe_rescale(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_in2, uint32_t p_bits, uint32_t batch,
                       void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (c->t != 0) return err(c, FHE_ERR_UNSUPPORTED, "rescale is CKKS-only");
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_in2) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_in2, 16)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (p_bits < 1 || p_bits >= c->logQ) return err(c, FHE_ERR_ARG, "p_bits out of range");
  CK(launch_rescale(c, d_out2, d_in2, batch * 2, p_bits, (cudaStream_t)stream), "rescale");
  return FHE_OK;
}

fhe_status fhe_mult_relin_rescale(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct1, const uint32_t* d_ct2,
                                  uint32_t p_bits, uint32_t batch, void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_ct1 || !d_ct2 || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_ct1, 16) || misaligned(d_ct2, 16) || misaligned(d_ws, 256)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (!c->have_evk) return err(c, FHE_ERR_STATE, "no evk installed (call fhe_set_evk first)");
  if (c->t != 0 && p_bits != 0) return err(c, FHE_ERR_UNSUPPORTED, "rescale is CKKS-only");
  if (p_bits >= c->logQ) return err(c, FHE_ERR_ARG, "p_bits out of range");
  if (ws_bytes < fhe_workspace_bytes(ctx, FHE_OP_MULT_RELIN_RESCALE, batch)) return err(c, FHE_ERR_NOMEM, "workspace too small");
  if (!c->fit_tensor || !c->fit_relin) return err(c, FHE_ERR_UNSUPPORTED, "CRT target too large for the conversion pipeline");
  cudaStream_t s = (cudaStream_t)stream;
  uint32_t* d3 = (uint32_t*)d_ws;
  uint32_t* ws = (uint32_t*)((char*)d_ws + ws_d3(c, batch));
  fhe_status st = do_he_mult(c, d3, d_ct1, d_ct2, batch, ws, s);
  if (st != FHE_OK) return st;
  return do_relin(c, d_out2, d3, batch, ws, p_bits, s);
}

fhe_status fhe_mult_relin_rescale_host(fhe_ctx* ctx, uint32_t* h_out2, const uint32_t* h_ct1, const uint32_t* h_ct2,
                                       uint32_t p_bits, uint32_t batch, void* d_ws, size_t ws_bytes, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!h_out2 || !h_ct1 || !h_ct2 || !d_ws) return err(c, FHE_ERR_ARG, "NULL pointer");
  const size_t ctb = align256((size_t)batch * 2 * c->L * c->N * 4);
  const size_t inner = fhe_workspace_bytes(ctx, FHE_OP_MULT_RELIN_RESCALE, batch);
  if (ws_bytes < inner + 3 * ctb) return err(c, FHE_ERR_NOMEM, "workspace too small");
  cudaStream_t s = (cudaStream_t)stream;
  char* base = (char*)d_ws + inner;
  uint32_t* d1 = (uint32_t*)base; uint32_t* d2 = (uint32_t*)(base + ctb); uint32_t* d_o = (uint32_t*)(base + 2 * ctb);
  // Batch items are independent, so the call is pipelined in pieces of `per` items over three streams: piece i + 1 is
  // on its way to the device (copy stream) while piece i runs on the caller's stream and piece i - 1 goes back to
  // the host (second copy stream): the PCIe transfers of both directions overlap each other and the kernels.
  const uint32_t per = (batch + Context::HOST_PIECES - 1) / Context::HOST_PIECES;
  const uint32_t pieces = (batch + per - 1) / per;
  const size_t item_words = (size_t)2 * c->L * c->N;
  // An error in the middle must not leave copies into / out of the caller's host buffers in flight behind the return:
  // every exit drains the three streams first.
  auto drain = [&]() { cudaStreamSynchronize(c->s_h2d); cudaStreamSynchronize(s); cudaStreamSynchronize(c->s_d2h); };
#define CKH(call, where) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { drain(); return cuda_fail(c, e_, where); } } while (0)
  CKH(cudaEventRecord(c->ev_start, s), "event");
  CKH(cudaStreamWaitEvent(c->s_h2d, c->ev_start, 0), "wait");         // the staging buffers are free once `s` gets here
  CKH(cudaStreamWaitEvent(c->s_d2h, c->ev_start, 0), "wait");
  for (uint32_t i = 0; i < pieces; ++i) {
    const uint32_t b0 = i * per, nb = batch - b0 < per ? batch - b0 : per;
    const size_t off = (size_t)b0 * item_words, bytes = (size_t)nb * item_words * 4;
    CKH(cudaMemcpyAsync(d1 + off, h_ct1 + off, bytes, cudaMemcpyHostToDevice, c->s_h2d), "H2D ct1");
    CKH(cudaMemcpyAsync(d2 + off, h_ct2 + off, bytes, cudaMemcpyHostToDevice, c->s_h2d), "H2D ct2");
    CKH(cudaEventRecord(c->ev_in[i], c->s_h2d), "event");
  }
  for (uint32_t i = 0; i < pieces; ++i) {
    const uint32_t b0 = i * per, nb = batch - b0 < per ? batch - b0 : per;
    const size_t off = (size_t)b0 * item_words, bytes = (size_t)nb * item_words * 4;
    CKH(cudaStreamWaitEvent(s, c->ev_in[i], 0), "wait");
    fhe_status st = fhe_mult_relin_rescale(ctx, d_o + off, d1 + off, d2 + off, p_bits, nb, d_ws, inner, stream);
    if (st != FHE_OK) { drain(); return st; }
    CKH(cudaEventRecord(c->ev_done[i], s), "event");
    CKH(cudaStreamWaitEvent(c->s_d2h, c->ev_done[i], 0), "wait");
    CKH(cudaMemcpyAsync(h_out2 + off, d_o + off, bytes, cudaMemcpyDeviceToHost, c->s_d2h), "D2H out");
  }
  CKH(cudaStreamSynchronize(c->s_d2h), "sync");
  CKH(cudaStreamSynchronize(s), "sync");
#undef CKH
  return FHE_OK;
}

// ---- NEXT-1: coefficient-wise operations (kernels_elem.cu) --------------------------------------------------------------
static fhe_status elem_call(fhe_ctx* ctx, int op, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly,
                            uint32_t bits, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (npoly == 0) return FHE_OK;
  if (!d_out || !d_a || (op <= 1 && !d_b)) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out, 16) || misaligned(d_a, 16) || (op <= 1 && misaligned(d_b, 16))) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (c->N < 256) return err(c, FHE_ERR_UNSUPPORTED, "N < 256");
  CK(launch_elem(c, op, d_out, d_a, d_b, npoly, bits, (cudaStream_t)stream), "elementwise");
  return FHE_OK;
}
fhe_status fhe_add(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly, void* stream) {
  return elem_call(ctx, 0, d_out, d_a, d_b, npoly, ctx ? C(ctx)->logQ : 0, stream);
}
fhe_status fhe_sub(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t npoly, void* stream) {
  return elem_call(ctx, 1, d_out, d_a, d_b, npoly, ctx ? C(ctx)->logQ : 0, stream);
}
fhe_status fhe_negate(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, uint32_t npoly, void* stream) {
  return elem_call(ctx, 2, d_out, d_a, nullptr, npoly, ctx ? C(ctx)->logQ : 0, stream);
}
fhe_status fhe_mul_monomial(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t k, uint32_t npoly, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (npoly == 0) return FHE_OK;
  if (!d_out || !d_in || d_out == d_in) return err(c, FHE_ERR_ARG, "NULL or aliasing pointer");
  if (misaligned(d_out, 16) || misaligned(d_in, 16)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (k >= 2 * c->N) return err(c, FHE_ERR_ARG, "k must be below 2N");
  if (c->N < 256) return err(c, FHE_ERR_UNSUPPORTED, "N < 256");
  CK(launch_monomial(c, d_out, d_in, k, npoly, (cudaStream_t)stream), "monomial");
  return FHE_OK;
}
// ---- NEXT-3: constants ----------------------------------------------------------------------------------------------------
fhe_status fhe_add_plain(fhe_ctx* ctx, uint32_t* d_out2, const uint32_t* d_ct, const uint32_t* d_pt, uint32_t batch,
                         uint32_t group, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (batch == 0) return FHE_OK;
  if (!d_out2 || !d_ct || !d_pt) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out2, 16) || misaligned(d_ct, 16) || misaligned(d_pt, 16)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (group == 0) return err(c, FHE_ERR_ARG, "group must be at least 1");
  if (c->N < 256) return err(c, FHE_ERR_UNSUPPORTED, "N < 256");
  CK(launch_add_plain(c, d_out2, d_ct, d_pt, batch, group, (cudaStream_t)stream), "add_plain");
  return FHE_OK;
}
fhe_status fhe_mult_scalar(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, int32_t k, uint32_t npoly, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (npoly == 0) return FHE_OK;
  if (!d_out || !d_in) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out, 16) || misaligned(d_in, 16)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (k == INT32_MIN) return err(c, FHE_ERR_ARG, "|k| must be below 2^31");
  if (c->N < 256) return err(c, FHE_ERR_UNSUPPORTED, "N < 256");
  if (c->t != 0) {   // the quotient estimate needs Q = 2^logQ + e with e < 2^(logQ - 33) (kernels_elem.cu)
    std::vector<uint32_t> e(c->h_Q.begin(), c->h_Q.begin() + c->L);
    e[c->logQ >> 5] &= ~(1u << (c->logQ & 31));
    bool ok = c->logQ >= 34 + 32;
    for (uint32_t l = 1; l < c->L; ++l) ok = ok && e[l] == 0;       // e below 2^32 <= 2^(logQ - 33) - 1 then
    if (!ok) return err(c, FHE_ERR_UNSUPPORTED, "mult_scalar (BGV): Q - 2^logQ too large for this logQ");
  }
  CK(launch_mult_scalar(c, d_out, d_in, k, npoly, (cudaStream_t)stream), "mult_scalar");
  return FHE_OK;
}
fhe_status fhe_moddown(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logq, uint32_t npoly, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (c->t != 0) return err(c, FHE_ERR_UNSUPPORTED, "moddown is CKKS-only");
  if (new_logq < 1 || new_logq > c->logQ) return err(c, FHE_ERR_ARG, "new_logq out of range");
  return elem_call(ctx, 3, d_out, d_in, nullptr, npoly, new_logq, stream);
}

// ---- NEXT-4: BGV modulus switch ----------------------------------------------------------------------------------------------
fhe_status fhe_modswitch(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_in, uint32_t new_logQ, uint32_t npoly, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (c->t == 0) return err(c, FHE_ERR_UNSUPPORTED, "modswitch is BGV-only (CKKS: fhe_rescale / fhe_moddown)");
  if (npoly == 0) return FHE_OK;
  if (!d_out || !d_in) return err(c, FHE_ERR_ARG, "NULL pointer");
  if (misaligned(d_out, 16) || misaligned(d_in, 16)) return err(c, FHE_ERR_ARG, "misaligned pointer");
  if (new_logQ >= c->logQ) return err(c, FHE_ERR_ARG, "new_logQ must be below logQ");
  if (c->logQ < 96 || new_logQ < 34) return err(c, FHE_ERR_UNSUPPORTED, "modswitch needs logQ >= 96 and new_logQ >= 34");
  const uint64_t e = modulus_offset(c->logQ, c->t), e2 = modulus_offset(new_logQ, c->t);   // both < 2 t < 2^32
  CK(launch_modswitch(c, d_out, d_in, new_logQ, (uint32_t)e, (uint32_t)e2, npoly, (cudaStream_t)stream), "modswitch");
  return FHE_OK;
}

fhe_status fhe_debug_force_pipeline(fhe_ctx* ctx, int mode) {
  if (!ctx || mode < 0 || mode > 2) return FHE_ERR_ARG;
  C(ctx)->force_pipe = mode;
  return FHE_OK;
}

fhe_status fhe_debug_crt_ambiguity(fhe_ctx* ctx, uint32_t bits) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (bits < 1 || bits > TOP_AMB) return err(c, FHE_ERR_ARG, "bits out of range");
  c->amb_bits = bits;
  return FHE_OK;
}

fhe_status fhe_debug_int_peak(fhe_ctx* ctx, int mode, double* per_second, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (!per_second || mode < 0 || mode > 2) return err(c, FHE_ERR_ARG, "bad argument");
  CK(measure_int_peak(c, mode, per_second, (cudaStream_t)stream), "int peak");
  return FHE_OK;
}

fhe_status fhe_debug_decompose(fhe_ctx* ctx, uint32_t* d_res, const uint32_t* d_limbs, uint32_t npoly, uint32_t Lin,
                               uint32_t K, uint32_t mask_bits, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (!d_res || !d_limbs || K == 0 || K > c->Kmax || Lin == 0 || Lin > MAX_LIMBS_IN) return err(c, FHE_ERR_ARG, "bad argument");
  CK(launch_decompose(c, d_res, 0, (size_t)K * c->N, d_limbs, 0, (size_t)Lin * c->N, 1, npoly, Lin, K, mask_bits, (cudaStream_t)stream, false), "decompose");
  return FHE_OK;
}

fhe_status fhe_debug_ntt(fhe_ctx* ctx, uint32_t* d_res, uint32_t npoly, uint32_t K, int inverse, void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = C(ctx);
  if (fhe_status ds = check_device(c)) return ds;
  if (!d_res || K == 0 || K > c->Kmax) return err(c, FHE_ERR_ARG, "bad argument");
  if (inverse) CK(launch_ntt_inv(c, d_res, npoly, 1, 1, K, c->d_scale_plain, (cudaStream_t)stream), "ntt inv");
  else CK(launch_ntt_fwd(c, d_res, npoly, 1, 1, K, (cudaStream_t)stream), "ntt fwd");
  return FHE_OK;
}

}  // extern "C"
