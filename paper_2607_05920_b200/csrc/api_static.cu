// api_static.cu -- fhe_polymul_static: the ring product of fhe_polymul for callers that cannot
// allocate device memory (code under CUDA graph capture, tight serving loops, harnesses that forbid cudaMalloc).
//
// fhe_polymul keeps its intermediate -- the residue matrix of both operands, [2 batch][K_pm][N] words, written by the
// decompose, transformed and multiplied in place, read by the CRT -- in a workspace the caller allocates.  Here that scratch
// is a file-scope device array of FHE_STATIC_SCRATCH_BYTES = 32 MiB: every GPU on which this library's module is loaded holds
// it until the process exits, which is why the maximum is modest.  The kernels are the ones fhe_polymul launches; only where
// their scratch lives differs.
//
// In HOST code the array's name is a host-side stand-in, not a device address (a kernel handed `g_static_scratch` from the
// host would fault or, where the GPU can reach host memory, silently use the wrong memory).  The device address is taken
// once per device with cudaGetSymbolAddress, with that device current (static_scratch_for_current_device), and that pointer
// is what the kernels receive.
//
// Sharing: every call on a device uses the SAME array and finds the previous call's contents in it.  Nothing in it has to
// start at zero -- the decompose writes every residue the transforms and the CRT later read (K_pm rows of N words per
// polynomial), so no clearing is needed -- but two calls that overlap on the GPU (different streams, or graphs launched
// concurrently) race on it: callers must order them.  Calls with a caller-owned workspace (fhe_polymul) do not touch it.
//
// This file calls no cudaMalloc / cudaFree / allocating library routine, and neither does the path below it (the hot-path
// calls never allocate: include/fhe.h, "Ownership").
#include "fhe_internal.cuh"

namespace fhe {

constexpr size_t STATIC_SCRATCH_BYTES = (size_t)32 << 20;
static __device__ __align__(256) uint32_t g_static_scratch[STATIC_SCRATCH_BYTES / sizeof(uint32_t)];

// device address of the array on the CURRENT device, looked up once per device
static cudaError_t static_scratch_for_current_device(uint32_t** out) {
  constexpr int MAX_DEV = 64;
  static uint32_t* addr[MAX_DEV] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= MAX_DEV) return cudaErrorInvalidDevice;
  if (!addr[dev]) {
    uint32_t* p = nullptr;
    e = cudaGetSymbolAddress((void**)&p, g_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    addr[dev] = p;
  }
  *out = addr[dev];
  return cudaSuccess;
}

static fhe_status fail(Context* c, fhe_status st, const std::string& msg) {
  c->err = msg;
  return st;
}

}  // namespace fhe

using namespace fhe;

extern "C" {

size_t fhe_static_scratch_bytes(void) { return STATIC_SCRATCH_BYTES; }

fhe_status fhe_polymul_static_init(fhe_ctx* ctx) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = reinterpret_cast<Context*>(ctx);
  int d = -1;
  if (cudaGetDevice(&d) != cudaSuccess || d != c->device)
    return fail(c, FHE_ERR_STATE, "the context's CUDA device is not the current device");
  uint32_t* p = nullptr;
  const cudaError_t e = static_scratch_for_current_device(&p);
  if (e != cudaSuccess) {
    cudaGetLastError();
    return fail(c, FHE_ERR_CUDA, std::string("cudaGetSymbolAddress(static scratch): ") + cudaGetErrorString(e));
  }
  return FHE_OK;
}

fhe_status fhe_polymul_static(fhe_ctx* ctx, uint32_t* d_out, const uint32_t* d_a, const uint32_t* d_b, uint32_t batch,
                              void* stream) {
  if (!ctx) return FHE_ERR_ARG;
  Context* c = reinterpret_cast<Context*>(ctx);
  if (batch == 0) return FHE_OK;
  const size_t need = fhe_workspace_bytes(ctx, FHE_OP_POLYMUL, batch);
  if (need > STATIC_SCRATCH_BYTES)
    return fail(c, FHE_ERR_NOMEM, "fhe_polymul_static: this batch needs " + std::to_string(need) + " bytes of scratch, the static scratch holds " +
                                      std::to_string(STATIC_SCRATCH_BYTES) + " (32 MiB): use fhe_polymul with a caller-owned workspace");
  if (fhe_status st = fhe_polymul_static_init(ctx)) return st;    // device check + the address (cached after the first call)
  uint32_t* scratch = nullptr;
  if (static_scratch_for_current_device(&scratch) != cudaSuccess) return fail(c, FHE_ERR_CUDA, "static scratch address");
  return fhe_polymul(ctx, d_out, d_a, d_b, batch, scratch, STATIC_SCRATCH_BYTES, stream);
}

}  // extern "C"
