// starkv_decode_attn_static: decode attention for callers that cannot allocate (code under CUDA graph capture, tight
// serving loops, harnesses that forbid cudaMalloc).  It is starkv_decode_attn -- the same kernels, chosen the same way
// -- with the decode workspace (latent-space query image, split-K partials [batch][split][head][4 + r_v] fp32, sliced
// combine partials; DESIGN.md section 6 "HBM layout") taken from a file-scope device array instead of a caller buffer.
//
//   * The array is STARKV_STATIC_SCRATCH_BYTES (8 MiB) of device memory per GPU that loads libstarkv.so, held until
//     the process exits.  8 MiB covers BASELINE.json configs C2-C5 (largest: C4, 7.2 MB); a call that needs more is
//     refused with STARKV_ERR_WORKSPACE and a text that names both sizes (starkv_last_error).
//   * In host code the array's NAME is a host-side stand-in, not a device address: a kernel given it would fault or,
//     where the GPU can reach host memory, silently use the wrong memory.  The device address is looked up here, in
//     the translation unit that defines the array, with cudaGetSymbolAddress -- once per device, with that device
//     current (the entry point refuses a context whose device is not the current one before it looks) -- and only
//     that address is ever handed to a kernel.
//   * The entry point calls no cudaMalloc / cudaFree / cudaHostAlloc and no allocating library routine: argument
//     checks, the size check, kernel launches.  (The first call on a device resolves the address and, like any first
//     launch, loads the kernels; make that call outside a graph capture.)
//   * Every call on a device shares the array, and it keeps the last call's contents.  Nothing in it has to start at
//     zero: every region a call reads (query image, partials of every split including empty ranges, slice partials) is
//     written earlier in the same call, so stale bytes of a previous call -- of any shape -- are never read
//     (tests/test_zz_no_alloc.py alternates shapes).  Calls that overlap on the GPU (two streams, two contexts or two
//     host threads on one device) RACE on the array: serialise them, or give the others their own workspace through
//     starkv_decode_attn.
#include <stdio.h>

#include "ctx.h"

static_assert(STARKV_STATIC_SCRATCH_BYTES % 256 == 0, "whole 256-byte lines");
static __device__ __align__(256) unsigned char sk_static_scratch[STARKV_STATIC_SCRATCH_BYTES];

namespace {

constexpr int SK_MAX_DEVICES = 64;
void* g_scratch_addr[SK_MAX_DEVICES];   // device address of sk_static_scratch on device i (0 = not looked up yet)

// Device address of the array on the CURRENT device, which the caller has checked to be `device`.
cudaError_t scratch_address(int device, void** out) {
  if (device < 0 || device >= SK_MAX_DEVICES) return cudaErrorInvalidDevice;
  if (!g_scratch_addr[device]) {
    void* p = nullptr;
    const cudaError_t e = cudaGetSymbolAddress(&p, sk_static_scratch);
    if (e != cudaSuccess) return e;
    if (!p) return cudaErrorInvalidSymbol;
    g_scratch_addr[device] = p;   // (two threads racing here store the same value)
  }
  *out = g_scratch_addr[device];
  return cudaSuccess;
}

}  // namespace

int starkv_decode_attn_static(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                              const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* out) {
  if (!ctx || batch <= 0 || max_pages <= 0) return STARKV_ERR_INVALID_ARG;
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) {
    (void)cudaGetLastError();
    return STARKV_ERR_CUDA;
  }
  if (dev != ctx->device) {
    snprintf(ctx->err, sizeof(ctx->err), "starkv_decode_attn_static: the context belongs to device %d, device %d is current",
             ctx->device, dev);
    return STARKV_ERR_INVALID_ARG;
  }
  const size_t need = starkv_workspace_bytes(ctx, batch, max_pages);
  if (need > (size_t)STARKV_STATIC_SCRATCH_BYTES) {
    snprintf(ctx->err, sizeof(ctx->err),
             "starkv_decode_attn_static: this call needs %zu bytes of scratch, the static array holds %zu "
             "(use starkv_decode_attn with a workspace of your own, or fewer splits / a smaller batch)",
             need, (size_t)STARKV_STATIC_SCRATCH_BYTES);
    return STARKV_ERR_WORKSPACE;
  }
  void* scratch = nullptr;
  SK_CUDA_CHECK(ctx, scratch_address(dev, &scratch));
  return starkv_decode_attn(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, scratch,
                            (size_t)STARKV_STATIC_SCRATCH_BYTES, out);
}
