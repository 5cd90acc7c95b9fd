// Internal context of libstarkv.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/starkv.h"
#include "decode_plan.h"
#include "starkv_layout.h"

struct starkv_ctx {
  StarkvLayout L;
  cudaStream_t stream;
  int device;
  int n_sm;
  int smem_optin;        // max dynamic shared memory per block (opt-in)
  int smem_per_sm;       // shared memory per SM
  int n_splits_override; // 0 = automatic
  int last_launches;
  const char* last_append;   // projection kernel of the last starkv_append (starkv_last_append_kernel_name)
  int fast_ok;           // tensor-core decode kernel covers this descriptor
  DecodePlan plan;
  TmPlan tm;             // TMEM-operand kernel of the integer modes (decode_tm.cu); tm.ok = it covers this descriptor
  int variant;           // decode kernel choice, SK_VARIANT_* (starkv_set_option "decode_variant"); 0 = automatic
  int append_tc5;        // prefill projection on the TMA + tcgen05 GEMM (default 1; starkv_set_option "append_tc5" 0 = mma.sync)
  int host_graph;        // HOST-buffer entry points replay a cached CUDA graph (starkv_set_option "host_graph")
  int pdl;               // launch the step's kernels with programmatic dependent launch (starkv_set_option "pdl")
  int timing_on;         // record events around the main decode kernel
  int timing_valid;
  cudaEvent_t ev0, ev1;
  // HOST-buffer entry points: pinned staging + one instantiated CUDA graph per call signature, so that a step costs
  // one cudaGraphLaunch instead of a dozen driver calls
  void* pin;              // pinned host staging of starkv_decode_attn_host: [q][seq_lens][out]
  size_t pin_bytes;
  void* pin2;             // pinned host staging of starkv_append_host: [k][v][seq_ids][positions]
  size_t pin2_bytes;
  cudaEvent_t pin_free;   // recorded after the last graph that reads the append staging area
  int pin_busy;
  struct HostGraph {
    cudaGraphExec_t exec;
    const void* p[8];
    long long v[10];
  };
  static const int kHostGraphs = 8;   // cached call signatures per entry point (e.g. one per block table in use)
  HostGraph g_dec[8], g_app[8];
  int g_dec_next, g_app_next;         // round-robin replacement
  // cudaFuncSetAttribute bookkeeping, per context (= per device: a context belongs to the device it was created on):
  // kernel -> largest dynamic shared-memory size granted (-1 = only the carve-out preference has been set)
  struct KernelAttr { const void* fn; int smem; };
  mutable KernelAttr attrs[48];
  mutable int n_attrs;
  int* tickets;          // SK_TICKETS zeroed ints in device memory (allocated at create): arrival counters of the sliced
                         // combine, one per (sequence, head), reset by the last arriver
  char err[512];
};
#define SK_TICKETS 16384
#define SK_APPEND_TICKETS 128   // after them: one arrival counter per group (KV head / values) of the small append

// decode kernel variants (starkv_set_decode_variant)
enum { SK_VARIANT_AUTO = 0, SK_VARIANT_MMA = 1, SK_VARIANT_TC5 = 2, SK_VARIANT_TM = 3, SK_VARIANT_GENERIC = 4 };

int sk_cuda_fail(starkv_ctx* ctx, cudaError_t e, const char* what);

#define SK_CUDA_CHECK(ctx, expr)                    \
  do {                                              \
    cudaError_t _e = (expr);                        \
    if (_e != cudaSuccess) return sk_cuda_fail((ctx), _e, #expr); \
  } while (0)

// The decode kernel runs with the maximum shared-memory carve-out.  Every other kernel of the step asks for the
// same carve-out, so that no L1/shared reconfiguration (an SM drain of several microseconds) sits between
// consecutive launches of a step.
// The attributes are per device, so the "already set" state lives in the context, not in function-local statics.
static inline starkv_ctx::KernelAttr* sk_attr_slot(const starkv_ctx* ctx, const void* fn, bool* fresh) {
  for (int i = 0; i < ctx->n_attrs; ++i)
    if (ctx->attrs[i].fn == fn) { *fresh = false; return &ctx->attrs[i]; }
  *fresh = true;
  if (ctx->n_attrs >= 48) return nullptr;   // table full: the caller sets the attribute every time
  ctx->attrs[ctx->n_attrs].fn = fn;
  ctx->attrs[ctx->n_attrs].smem = -1;
  return &ctx->attrs[ctx->n_attrs++];
}
template <typename K>
static inline cudaError_t sk_prefer_smem(const starkv_ctx* ctx, K kernel) {
  bool fresh;
  sk_attr_slot(ctx, (const void*)kernel, &fresh);
  if (!fresh) return cudaSuccess;
  return cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
}
template <typename K>
static inline cudaError_t sk_need_smem(const starkv_ctx* ctx, K kernel, int bytes) {
  bool fresh;
  starkv_ctx::KernelAttr* a = sk_attr_slot(ctx, (const void*)kernel, &fresh);
  if (a && a->smem < 0) {
    // the attribute belongs to the device's copy of the kernel, which other contexts share: start from what is
    // already granted and only ever raise it (a context with a smaller plan must not shrink another one's limit)
    cudaFuncAttributes fa;
    if (cudaFuncGetAttributes(&fa, kernel) == cudaSuccess) a->smem = fa.maxDynamicSharedSizeBytes;
    else cudaGetLastError();
  }
  if (a && a->smem >= bytes) return cudaSuccess;
  const cudaError_t e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes);
  if (e == cudaSuccess && a) a->smem = bytes;
  return e;
}
#define SK_PREFER_SMEM(ctx, kernel) SK_CUDA_CHECK((ctx), sk_prefer_smem((ctx), (kernel)))

// Programmatic dependent launch (PDL): the kernels of a step are launched with the stream-serialization
// attribute, trigger their dependents at once and wait for their predecessor (griddepcontrol.wait) before touching
// global memory, so a kernel's launch latency and CTA ramp overlap the tail of the one before it.  Every such
// kernel waits, hence completion stays transitive: kernel K done implies kernel K-1 done.
#ifdef __CUDACC__
__device__ __forceinline__ void sk_pdl_enter() {
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  asm volatile("griddepcontrol.wait;" ::: "memory");
}
// The two halves separately, for a kernel that does dependency-free work first: shared-memory set-up and reads of
// CALLER-OWNED inputs that no kernel of this library ever writes (seq_lens, block tables).  Such inputs are final
// when the first kernel of a PDL chain starts (a predecessor outside the chain never triggers early, so the chain's
// head starts only after it completed), hence they may be read before the wait.
__device__ __forceinline__ void sk_pdl_trigger() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void sk_pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
template <typename... KArgs, typename... Args>
static inline cudaError_t sk_launch(const starkv_ctx* ctx, void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem,
                                    Args... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = grid;
  cfg.blockDim = block;
  cfg.dynamicSmemBytes = smem;
  cfg.stream = ctx->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = ctx->pdl ? 1 : 0;
  return cudaLaunchKernelEx(&cfg, kern, args...);
}
#endif

struct AppendSmallArgs;

// codec.cu
int sk_pack(starkv_ctx* ctx, const void* lk, const void* lv, int n_tokens, void* pages);
int sk_unpack(starkv_ctx* ctx, const void* pages, int n_tokens, int8_t* codes, uint16_t* scales, float* deq);
int sk_append(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
              const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride,
              int64_t k_head_stride, int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v,
              const void* A_k, const void* A_v, void* ws, size_t ws_bytes);
size_t sk_append_ws_bytes(const starkv_ctx* ctx, int n_new);
// append_gemm.cu: prefill append (n_new >= 64) by TMA + tcgen05; 2 = done (quantiser and paged write fused), 1 = z holds
// fp16(X . A), 0 = not covered (the caller falls back)
int sk_append_gemm(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
                   const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride, int64_t k_head_stride, int d_in_k,
                   const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k, const void* A_v, void* z);
int sk_append_small_ok(const starkv_ctx* ctx, int n_new);   // the one-launch append covers n_new tokens
int sk_append_small_fused(const starkv_ctx* ctx, int n_new, int n_part, int limit);   // A1-A4 in one launch (else A1, then append_write_kernel)
int sk_append_small_write(starkv_ctx* ctx, const AppendSmallArgs* a);   // A2-A4 from the partials of an un-fused A1 launch
void sk_append_small_args(const starkv_ctx* ctx, AppendSmallArgs* a, void* pool, const int32_t* table, int max_pages,
                          const int32_t* seq_ids, const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride,
                          int64_t k_head_stride, int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v,
                          const void* A_k, const void* A_v, void* ws);

// decode.cu / decode_generic.cu
struct SkWorkspace {   // carve-up of the caller's decode workspace
  size_t qimg_off;     // latent-space query images, per sequence
  size_t qimg_stride;
  size_t part_off;     // split-K partials
  size_t slice_off;    // sliced combine: per-slice up-projection partials
  size_t host_off;     // staging for the _host variant (q, seq_lens, out)
  size_t total;
  int n_splits;
};
void sk_plan_workspace(const starkv_ctx* ctx, int batch, int max_pages, SkWorkspace* w);
int sk_decode_generic(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                      const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws,
                      size_t ws_bytes, void* out, int rope = 0, float rope_theta = 0.f, const int32_t* pos_offset = nullptr);
int sk_decode_fast(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                   const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws,
                   size_t ws_bytes, void* out, const AppendSmallArgs* app = nullptr);   // app: the step's append, run in the first launch
int sk_fast_supported(const starkv_ctx* ctx);
int sk_fast_plan(starkv_ctx* ctx);   // fills ctx->plan, ctx->fast_ok
int sk_tm_plan(starkv_ctx* ctx);     // fills ctx->tm
int sk_decode_tm(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                 const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                 void* out, const AppendSmallArgs* app = nullptr);   // app: the step's append, run in the first launch
