// C ABI of libstarkv.so (include/starkv.h): argument checks, context, dispatch.  No compute here.
#include <stdio.h>
#include <stdlib.h>
#include <string.h>

#include "append_small.cuh"
#include "ctx.h"

int sk_cuda_fail(starkv_ctx* ctx, cudaError_t e, const char* what) {
  if (ctx) snprintf(ctx->err, sizeof(ctx->err), "%s: %s (%s)", cudaGetErrorName(e), cudaGetErrorString(e), what);
  (void)cudaGetLastError();   // clear the non-sticky error state
  return STARKV_ERR_CUDA;
}

static bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }

// A context belongs to the device it was created on (kernel attributes, tickets, pinned staging): a call made with
// another device current is refused instead of launching there.
static bool sk_device_ok(starkv_ctx* ctx) {
  int dev = -1;
  if (cudaGetDevice(&dev) != cudaSuccess) { (void)cudaGetLastError(); return false; }
  if (dev != ctx->device) {
    snprintf(ctx->err, sizeof(ctx->err), "context created on device %d, called with device %d current", ctx->device, dev);
    return false;
  }
  return true;
}

// ---- pinned staging and graph cache of the HOST-buffer entry points ----
static const size_t kPinDecode = 0;
// grow a pinned staging block; the graph that captured the old address is dropped
static int sk_pin_reserve(starkv_ctx* ctx, void** pin, size_t* have, size_t bytes, starkv_ctx::HostGraph* g) {
  if (*have >= bytes) return STARKV_OK;
  for (int i = 0; i < starkv_ctx::kHostGraphs; ++i)
    if (g[i].exec) { cudaGraphExecDestroy(g[i].exec); g[i].exec = nullptr; }
  SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
  if (*pin) cudaFreeHost(*pin);
  *pin = nullptr;
  *have = 0;
  if (bytes < ((size_t)1 << 16)) bytes = (size_t)1 << 16;
  SK_CUDA_CHECK(ctx, cudaHostAlloc(pin, bytes, cudaHostAllocDefault));
  *have = bytes;
  return STARKV_OK;
}
static starkv_ctx::HostGraph* sk_graph_find(starkv_ctx::HostGraph* gs, const void* const* p, const long long* v) {
  for (int k = 0; k < starkv_ctx::kHostGraphs; ++k) {
    starkv_ctx::HostGraph& g = gs[k];
    if (!g.exec) continue;
    bool ok = true;
    for (int i = 0; i < 8 && ok; ++i) ok = g.p[i] == p[i];
    for (int i = 0; i < 10 && ok; ++i) ok = g.v[i] == v[i];
    if (ok) return &g;
  }
  return nullptr;
}
static starkv_ctx::HostGraph* sk_graph_slot(starkv_ctx::HostGraph* gs, int* next) {
  starkv_ctx::HostGraph* g = &gs[*next];
  *next = (*next + 1) % starkv_ctx::kHostGraphs;
  if (g->exec) { cudaGraphExecDestroy(g->exec); g->exec = nullptr; }
  return g;
}
// graphs are not used on the legacy / per-thread default streams (not capturable) or inside a caller's capture
static bool sk_stream_capturing(starkv_ctx* ctx) {
  if (ctx->stream == nullptr || ctx->stream == cudaStreamLegacy || ctx->stream == cudaStreamPerThread) return true;
  cudaStreamCaptureStatus st = cudaStreamCaptureStatusNone;
  if (cudaStreamIsCapturing(ctx->stream, &st) != cudaSuccess) { (void)cudaGetLastError(); return true; }
  return st != cudaStreamCaptureStatusNone;
}

extern "C" {

int starkv_create(starkv_ctx** out, const starkv_desc* d, void* cuda_stream) {
  if (!out) return STARKV_ERR_INVALID_ARG;
  *out = nullptr;
  if (!d || !d->rank_k) return STARKV_ERR_INVALID_ARG;
  if (d->layout_id != 1) return STARKV_ERR_UNSUPPORTED;
  if (d->bits_hi != 16 && !d->rank_k_hi) return STARKV_ERR_INVALID_ARG;
  if (d->n_kv_heads <= 0 || d->n_kv_heads > STARKV_MAX_KV_HEADS) return STARKV_ERR_INVALID_ARG;
  starkv_ctx* ctx = (starkv_ctx*)calloc(1, sizeof(starkv_ctx));
  if (!ctx) return STARKV_ERR_INVALID_ARG;
  const float sm = d->sm_scale > 0.f ? d->sm_scale : 1.0f / sqrtf((float)(d->head_dim > 0 ? d->head_dim : 1));
  const int rc = starkv_build_layout(&ctx->L, d->n_q_heads, d->n_kv_heads, d->head_dim, d->rank_k, d->rank_k_hi, d->rank_v,
                                     d->rank_v_hi, d->bits_hi, d->bits_lo, d->page_tokens, sm);
  if (rc != 0) {
    free(ctx);
    return rc == -2 ? STARKV_ERR_UNSUPPORTED : STARKV_ERR_INVALID_ARG;
  }
  ctx->stream = (cudaStream_t)cuda_stream;
  cudaError_t e = cudaGetDevice(&ctx->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, ctx->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->smem_optin, cudaDevAttrMaxSharedMemoryPerBlockOptin, ctx->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&ctx->smem_per_sm, cudaDevAttrMaxSharedMemoryPerMultiprocessor, ctx->device);
  if (e != cudaSuccess) {   // no usable device: fail loudly, there is no CPU path
    (void)cudaGetLastError();
    free(ctx);
    return STARKV_ERR_CUDA;
  }
  ctx->pdl = 1;
  ctx->append_tc5 = 1;
  if (cudaMalloc((void**)&ctx->tickets, (SK_TICKETS + SK_APPEND_TICKETS) * sizeof(int)) != cudaSuccess ||
      cudaMemset(ctx->tickets, 0, (SK_TICKETS + SK_APPEND_TICKETS) * sizeof(int)) != cudaSuccess) {
    (void)cudaGetLastError();
    if (ctx->tickets) cudaFree(ctx->tickets);
    ctx->tickets = nullptr;   // the sliced combine is skipped
  }
  sk_fast_plan(ctx);
  sk_tm_plan(ctx);
  *out = ctx;
  return STARKV_OK;
}

void starkv_destroy(starkv_ctx* ctx) {
  if (!ctx) return;
  if (ctx->ev0) cudaEventDestroy(ctx->ev0);
  if (ctx->ev1) cudaEventDestroy(ctx->ev1);
  for (int i = 0; i < starkv_ctx::kHostGraphs; ++i) {
    if (ctx->g_dec[i].exec) cudaGraphExecDestroy(ctx->g_dec[i].exec);
    if (ctx->g_app[i].exec) cudaGraphExecDestroy(ctx->g_app[i].exec);
  }
  if (ctx->pin_free) cudaEventDestroy(ctx->pin_free);
  if (ctx->tickets) cudaFree(ctx->tickets);
  if (ctx->pin) cudaFreeHost(ctx->pin);
  if (ctx->pin2) cudaFreeHost(ctx->pin2);
  free(ctx);
}

size_t starkv_page_bytes(const starkv_ctx* ctx) { return ctx ? (size_t)ctx->L.page_bytes : 0; }

size_t starkv_workspace_bytes(const starkv_ctx* ctx, int batch, int max_pages) {
  if (!ctx || batch <= 0 || max_pages <= 0) return 0;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  return w.total;
}

size_t starkv_append_workspace_bytes(const starkv_ctx* ctx, int n_new) { return ctx ? sk_append_ws_bytes(ctx, n_new) : 0; }

int starkv_pack(starkv_ctx* ctx, const void* lk, const void* lv, int n_tokens, void* pages) {
  if (!ctx || !sk_device_ok(ctx)) return STARKV_ERR_INVALID_ARG;
  if (n_tokens > 0 && (!aligned16(lk) || !aligned16(lv) || !aligned16(pages))) return STARKV_ERR_INVALID_ARG;
  return sk_pack(ctx, lk, lv, n_tokens, pages);
}

int starkv_unpack(starkv_ctx* ctx, const void* pages, int n_tokens, int8_t* codes, uint16_t* scales, float* deq) {
  if (!ctx || !sk_device_ok(ctx)) return STARKV_ERR_INVALID_ARG;
  if (n_tokens > 0 && !aligned16(pages)) return STARKV_ERR_INVALID_ARG;
  return sk_unpack(ctx, pages, n_tokens, codes, scales, deq);
}

int starkv_append(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
                  const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride, int64_t k_head_stride,
                  int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k, const void* A_v,
                  void* ws, size_t ws_bytes) {
  if (!ctx || !sk_device_ok(ctx)) return STARKV_ERR_INVALID_ARG;
  if (n_new > 0 && (!aligned16(pool) || !aligned16(ws))) return STARKV_ERR_INVALID_ARG;
  return sk_append(ctx, pool, table, max_pages, seq_ids, positions, n_new, k_new, k_row_stride, k_head_stride, d_in_k,
                   v_new, v_row_stride, d_in_v, A_k, A_v, ws, ws_bytes);
}

// which decode kernel family a call runs on: the TMEM-operand kernel where it covers the descriptor (integer modes),
// else the mma.sync / tcgen05-PV kernels of decode_fast.cu, else the scalar kernel
static int sk_decode_choice(const starkv_ctx* ctx) {
  if (ctx->variant == SK_VARIANT_GENERIC) return SK_VARIANT_GENERIC;
  if (ctx->tm.ok && (ctx->variant == SK_VARIANT_AUTO || ctx->variant == SK_VARIANT_TM)) return SK_VARIANT_TM;
  if (ctx->fast_ok) return ctx->plan.um ? SK_VARIANT_TC5 : SK_VARIANT_MMA;
  return SK_VARIANT_GENERIC;
}

static int check_decode_args(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                             const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, void* out) {
  if (!ctx || batch <= 0 || max_pages <= 0 || !sk_device_ok(ctx)) return STARKV_ERR_INVALID_ARG;
  if (!q || !pool || !table || !seq_lens || !B_k || !B_v || !ws || !out) return STARKV_ERR_INVALID_ARG;
  if (!aligned16(q) || !aligned16(B_k) || !aligned16(B_v) || !aligned16(ws) || !aligned16(out)) return STARKV_ERR_INVALID_ARG;
  if (((uintptr_t)pool & 127) != 0) return STARKV_ERR_INVALID_ARG;
  return STARKV_OK;
}

int starkv_decode_attn(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                       const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                       void* out) {
  const int rc = check_decode_args(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, out);
  if (rc) return rc;
  switch (sk_decode_choice(ctx)) {
    case SK_VARIANT_TM: return sk_decode_tm(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out);
    case SK_VARIANT_GENERIC: return sk_decode_generic(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out);
    default: return sk_decode_fast(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out);
  }
}

int starkv_decode_attn_latent(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                              const int32_t* seq_lens, int batch, const void* B_k, void* ws, size_t ws_bytes, void* out_latent) {
  // B_k stands in for B_v in the shared argument check (latent-output mode has no B_v); a null B_v selects the
  // merge-only combine in sk_launch_combine
  const int rc = check_decode_args(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_k, ws, out_latent);
  if (rc) return rc;
  switch (sk_decode_choice(ctx)) {
    case SK_VARIANT_TM: return sk_decode_tm(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, nullptr, ws, ws_bytes, out_latent);
    case SK_VARIANT_GENERIC: return sk_decode_generic(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, nullptr, ws, ws_bytes, out_latent);
    default: return sk_decode_fast(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, nullptr, ws, ws_bytes, out_latent);
  }
}

int starkv_decode_step(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
                       const int32_t* positions, int batch, const void* k_new, int64_t k_row_stride, int64_t k_head_stride,
                       int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k, const void* A_v,
                       void* append_ws, size_t append_ws_bytes, const void* q, const int32_t* seq_lens, const void* B_k,
                       const void* B_v, void* ws, size_t ws_bytes, void* out) {
  int rc = check_decode_args(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, out);
  if (rc) return rc;
  if (!seq_ids || !positions || !k_new || !v_new || !A_k || !A_v || !append_ws || !aligned16(append_ws) || d_in_k <= 0 ||
      d_in_v <= 0)
    return STARKV_ERR_INVALID_ARG;
  if (append_ws_bytes < sk_append_ws_bytes(ctx, batch)) return STARKV_ERR_WORKSPACE;
  AppendSmallArgs a;
  const int choice = sk_decode_choice(ctx);
  if (choice != SK_VARIANT_GENERIC && sk_append_small_ok(ctx, batch))
    sk_append_small_args(ctx, &a, pool, table, max_pages, seq_ids, positions, batch, k_new, k_row_stride, k_head_stride, d_in_k,
                         v_new, v_row_stride, d_in_v, A_k, A_v, append_ws);
  else
    a.n_part = 0;
  if (a.n_part > 0) {
    // The append's projection shares the query image's launch.  Where the serial tail of the one-launch form stays short
    // (<= 2K partial sums: measured, codec.cu) it is the whole append (three launches per step); else the quantiser / paged
    // write follows as a launch of its own (four).
    a.fused = sk_append_small_fused(ctx, batch, a.n_part, 2048);
    if (choice == SK_VARIANT_TM) return sk_decode_tm(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out, &a);
    return sk_decode_fast(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out, &a);
  }
  rc = sk_append(ctx, pool, table, max_pages, seq_ids, positions, batch, k_new, k_row_stride, k_head_stride, d_in_k, v_new,
                 v_row_stride, d_in_v, A_k, A_v, append_ws, append_ws_bytes);
  if (rc) return rc;
  const int n_app = ctx->last_launches;
  rc = starkv_decode_attn(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out);
  ctx->last_launches += n_app;
  return rc;
}

int starkv_decode_attn_generic(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                               const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws,
                               size_t ws_bytes, void* out) {
  const int rc = check_decode_args(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, out);
  if (rc) return rc;
  return sk_decode_generic(ctx, q, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out);
}

int starkv_decode_attn_rope(starkv_ctx* ctx, const void* q_rotated, const void* pool, const int32_t* table, int max_pages,
                            const int32_t* seq_lens, const int32_t* pos_offset, float rope_theta, int batch, const void* B_k,
                            const void* B_v, void* ws, size_t ws_bytes, void* out) {
  const int rc = check_decode_args(ctx, q_rotated, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, out);
  if (rc) return rc;
  if (!(rope_theta > 1.f) || (ctx->L.head_dim & 1)) return STARKV_ERR_INVALID_ARG;
  return sk_decode_generic(ctx, q_rotated, pool, table, max_pages, seq_lens, batch, B_k, B_v, ws, ws_bytes, out, 1, rope_theta,
                           pos_offset);
}

// enqueue-only body shared by the direct and the captured path: copies from `q_src` / `len_src`, decode, copy to `out_dst`
static int sk_decode_host_enqueue(starkv_ctx* ctx, const void* q_src, const void* pool, const int32_t* table, int max_pages,
                                  const int32_t* len_src, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                                  void* out_dst, bool staged) {
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  const size_t qbytes = (size_t)batch * ctx->L.n_q_heads * ctx->L.head_dim * 2;
  const size_t qb = (qbytes + 255) / 256 * 256;
  const size_t lb = ((size_t)batch * 4 + 255) / 256 * 256;
  uint8_t* dq = (uint8_t*)ws + w.host_off;   // device staging [q][seq_lens][out], same layout as the pinned block
  int32_t* dlen = (int32_t*)(dq + qb);
  uint8_t* dout = dq + qb + lb;
  if (staged) {   // sources are the library's pinned block [q][seq_lens]: one copy for both
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dq, q_src, qb + (size_t)batch * 4, cudaMemcpyHostToDevice, ctx->stream));
  } else {
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dq, q_src, qbytes, cudaMemcpyHostToDevice, ctx->stream));
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dlen, len_src, (size_t)batch * 4, cudaMemcpyHostToDevice, ctx->stream));
  }
  const int rc = starkv_decode_attn(ctx, dq, pool, table, max_pages, dlen, batch, B_k, B_v, ws, ws_bytes, dout);
  if (rc) return rc;
  SK_CUDA_CHECK(ctx, cudaMemcpyAsync(out_dst, dout, qbytes, cudaMemcpyDeviceToHost, ctx->stream));
  return STARKV_OK;
}

int starkv_decode_attn_host(starkv_ctx* ctx, const void* q_host, const void* pool, const int32_t* table, int max_pages,
                            const int32_t* seq_lens_host, int batch, const void* B_k, const void* B_v, void* ws,
                            size_t ws_bytes, void* out_host) {
  if (!ctx || batch <= 0 || max_pages <= 0 || !q_host || !seq_lens_host || !out_host || !ws) return STARKV_ERR_INVALID_ARG;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  const size_t qbytes = (size_t)batch * ctx->L.n_q_heads * ctx->L.head_dim * 2;
  const size_t qb = (qbytes + 255) / 256 * 256, lb = ((size_t)batch * 4 + 255) / 256 * 256;
  if (ctx->timing_on || sk_stream_capturing(ctx)) {   // plain path: event timing wants the kernels un-captured
    const int rc = sk_decode_host_enqueue(ctx, q_host, pool, table, max_pages, seq_lens_host, batch, B_k, B_v, ws, ws_bytes, out_host, false);
    if (rc) return rc;
    SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    return STARKV_OK;
  }
  // pinned staging: [q][seq_lens][out] at the start of the block; the append staging lives behind it
  const size_t dec_bytes = 2 * qb + lb;
  {
    const int rc = sk_pin_reserve(ctx, &ctx->pin, &ctx->pin_bytes, dec_bytes, ctx->g_dec);
    if (rc) return rc;
  }
  uint8_t* pq = (uint8_t*)ctx->pin + kPinDecode;
  uint8_t* plen = pq + qb;
  uint8_t* pout = plen + lb;
  const bool use_graph = ctx->host_graph != 0;
  if (!use_graph) {   // default: direct enqueue, one H2D copy (q + seq_lens) from the pinned block, one D2H copy
    memcpy(pq, q_host, qbytes);
    memcpy(plen, seq_lens_host, (size_t)batch * 4);
    const int rc = sk_decode_host_enqueue(ctx, pq, pool, table, max_pages, (const int32_t*)plen, batch, B_k, B_v, ws, ws_bytes, pout, true);
    if (rc) return rc;
    SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    memcpy(out_host, pout, qbytes);
    return STARKV_OK;
  }
  const void* kp[8] = {pool, table, B_k, B_v, ws, ctx->pin, nullptr, nullptr};
  const long long kv[10] = {max_pages, batch, (long long)ws_bytes, ctx->n_splits_override, 0, 0, 0, 0, 0, 0};
  starkv_ctx::HostGraph* hg = sk_graph_find(ctx->g_dec, kp, kv);
  if (!hg) {
    hg = sk_graph_slot(ctx->g_dec, &ctx->g_dec_next);
    // un-captured warm-up run: sets the kernels' function attributes (not capturable) and validates the arguments
    memcpy(pq, q_host, qbytes);
    memcpy(plen, seq_lens_host, (size_t)batch * 4);
    int rc = sk_decode_host_enqueue(ctx, pq, pool, table, max_pages, (const int32_t*)plen, batch, B_k, B_v, ws, ws_bytes, pout, true);
    if (rc) return rc;
    SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    cudaGraph_t graph = nullptr;
    SK_CUDA_CHECK(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
    rc = sk_decode_host_enqueue(ctx, pq, pool, table, max_pages, (const int32_t*)plen, batch, B_k, B_v, ws, ws_bytes, pout, true);
    const cudaError_t ce = cudaStreamEndCapture(ctx->stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    SK_CUDA_CHECK(ctx, ce);
    const cudaError_t ie = cudaGraphInstantiate(&hg->exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ie != cudaSuccess) hg->exec = nullptr;
    SK_CUDA_CHECK(ctx, ie);
    memcpy(hg->p, kp, sizeof(kp));
    memcpy(hg->v, kv, sizeof(kv));
    memcpy(out_host, pout, qbytes);   // the warm-up run already produced this call's result
    return STARKV_OK;
  }
  memcpy(pq, q_host, qbytes);
  memcpy(plen, seq_lens_host, (size_t)batch * 4);
  SK_CUDA_CHECK(ctx, cudaGraphLaunch(hg->exec, ctx->stream));
  SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
  memcpy(out_host, pout, qbytes);
  return STARKV_OK;
}

size_t starkv_append_host_workspace_bytes(const starkv_ctx* ctx, int n_new, int k_row_elems, int v_row_elems) {
  if (!ctx || n_new <= 0 || k_row_elems < 0 || v_row_elems < 0) return 0;
  const size_t up = 255;
  // projection scratch, then staging for [k_new][v_new][seq_ids][positions] and -- starkv_decode_step_host only --
  // [q][seq_lens] for n_new sequences, so that one copy brings a whole step's inputs
  const size_t qb = ((size_t)n_new * ctx->L.n_q_heads * ctx->L.head_dim * 2 + up) & ~up;
  return sk_append_ws_bytes(ctx, n_new) + (((size_t)n_new * k_row_elems * 2 + up) & ~up) +
         (((size_t)n_new * v_row_elems * 2 + up) & ~up) + 3 * (((size_t)n_new * 4 + up) & ~up) + qb;
}

// enqueue-only body shared by the direct and the captured path
static int sk_append_host_enqueue(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const void* seq_src,
                                  const void* pos_src, int n_new, const void* k_src, int k_row_elems, int64_t k_head_stride,
                                  int d_in_k, const void* v_src, int v_row_elems, int d_in_v, const void* A_k, const void* A_v,
                                  void* ws, bool staged_block) {
  const size_t up = 255;
  const size_t zb = sk_append_ws_bytes(ctx, n_new);
  const size_t kb = (size_t)n_new * k_row_elems * 2, vb = (size_t)n_new * v_row_elems * 2, ib = (size_t)n_new * 4;
  uint8_t* dk = (uint8_t*)ws + zb;
  uint8_t* dv = dk + ((kb + up) & ~up);
  int32_t* dseq = (int32_t*)(dv + ((vb + up) & ~up));
  int32_t* dpos = (int32_t*)((uint8_t*)dseq + ((ib + up) & ~up));
  const void* vdev = v_src != k_src ? (const void*)dv : (const void*)dk;
  const bool staged = staged_block && v_src != k_src;   // [k][v][seq_ids][positions] in the device staging layout
  if (staged) {   // sources already in the device staging layout (pinned block of starkv_append_host): one copy
    const size_t total = ((kb + up) & ~up) + ((vb + up) & ~up) + ((ib + up) & ~up) + ib;
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dk, k_src, total, cudaMemcpyHostToDevice, ctx->stream));
  } else {
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dk, k_src, kb, cudaMemcpyHostToDevice, ctx->stream));
    if (v_src != k_src) SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dv, v_src, vb, cudaMemcpyHostToDevice, ctx->stream));
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dseq, seq_src, ib, cudaMemcpyHostToDevice, ctx->stream));
    SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dpos, pos_src, ib, cudaMemcpyHostToDevice, ctx->stream));
  }
  return starkv_append(ctx, pool, table, max_pages, dseq, dpos, n_new, dk, k_row_elems, k_head_stride, d_in_k, vdev,
                       v_row_elems, d_in_v, A_k, A_v, ws, zb);
}

int starkv_append_host(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids_host,
                       const int32_t* positions_host, int n_new, const void* k_new_host, int k_row_elems,
                       int64_t k_head_stride, int d_in_k, const void* v_new_host, int v_row_elems, int d_in_v,
                       const void* A_k, const void* A_v, void* ws, size_t ws_bytes) {
  if (!ctx || n_new < 0) return STARKV_ERR_INVALID_ARG;
  if (n_new == 0) return STARKV_OK;
  if (!seq_ids_host || !positions_host || !k_new_host || !v_new_host || !ws || !aligned16(ws)) return STARKV_ERR_INVALID_ARG;
  if (ws_bytes < starkv_append_host_workspace_bytes(ctx, n_new, k_row_elems, v_row_elems)) return STARKV_ERR_WORKSPACE;
  const size_t up = 255;
  const size_t kb = (size_t)n_new * k_row_elems * 2, vb = (size_t)n_new * v_row_elems * 2, ib = (size_t)n_new * 4;
  const bool same = v_new_host == k_new_host;
  const size_t kbp = (kb + up) & ~up, vbp = same ? 0 : ((vb + up) & ~up), ibp = (ib + up) & ~up;
  const bool use_graph = ctx->host_graph != 0;
  const size_t need = kbp + vbp + 2 * ibp;
  if (n_new > 64 || need > ((size_t)4 << 20) || ctx->stream == nullptr || ctx->stream == cudaStreamLegacy ||
      ctx->stream == cudaStreamPerThread)   // staging is for decode-time appends on a stream of the caller's own
    return sk_append_host_enqueue(ctx, pool, table, max_pages, seq_ids_host, positions_host, n_new, k_new_host, k_row_elems,
                                  k_head_stride, d_in_k, v_new_host, v_row_elems, d_in_v, A_k, A_v, ws, false);
  // the previous graph launch may still be reading the staging block (this call does not synchronise)
  if (ctx->pin_busy) {
    SK_CUDA_CHECK(ctx, cudaEventSynchronize(ctx->pin_free));
    ctx->pin_busy = 0;
  }
  {
    const int rc = sk_pin_reserve(ctx, &ctx->pin2, &ctx->pin2_bytes, need, ctx->g_app);
    if (rc) return rc;
  }
  uint8_t* pk = (uint8_t*)ctx->pin2;
  uint8_t* pv = same ? pk : pk + kbp;
  uint8_t* pseq = pk + kbp + vbp;
  uint8_t* ppos = pseq + ibp;
  memcpy(pk, k_new_host, kb);
  if (!same) memcpy(pv, v_new_host, vb);
  memcpy(pseq, seq_ids_host, ib);
  memcpy(ppos, positions_host, ib);
  if (!ctx->pin_free) SK_CUDA_CHECK(ctx, cudaEventCreateWithFlags(&ctx->pin_free, cudaEventDisableTiming));
  if (!use_graph || sk_stream_capturing(ctx)) {   // default: direct enqueue, one H2D copy from the pinned block
    const int rc = sk_append_host_enqueue(ctx, pool, table, max_pages, pseq, ppos, n_new, pk, k_row_elems, k_head_stride, d_in_k,
                                          pv, v_row_elems, d_in_v, A_k, A_v, ws, true);
    if (rc) return rc;
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->pin_free, ctx->stream));
    ctx->pin_busy = 1;
    return STARKV_OK;
  }
  const void* kp[8] = {pool, table, A_k, A_v, ws, ctx->pin2, nullptr, nullptr};
  const long long kv[10] = {max_pages, n_new, k_row_elems, (long long)k_head_stride, d_in_k, v_row_elems, d_in_v, same ? 1 : 0, 0, 0};
  starkv_ctx::HostGraph* hg = sk_graph_find(ctx->g_app, kp, kv);
  if (!hg) {
    hg = sk_graph_slot(ctx->g_app, &ctx->g_app_next);
    // un-captured warm-up run (function attributes, argument checks); it also performs this call's append
    int rc = sk_append_host_enqueue(ctx, pool, table, max_pages, pseq, ppos, n_new, pk, k_row_elems, k_head_stride, d_in_k, pv,
                                    v_row_elems, d_in_v, A_k, A_v, ws, true);
    if (rc) return rc;
    SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
    cudaGraph_t graph = nullptr;
    SK_CUDA_CHECK(ctx, cudaStreamBeginCapture(ctx->stream, cudaStreamCaptureModeThreadLocal));
    rc = sk_append_host_enqueue(ctx, pool, table, max_pages, pseq, ppos, n_new, pk, k_row_elems, k_head_stride, d_in_k, pv,
                                v_row_elems, d_in_v, A_k, A_v, ws, true);
    const cudaError_t ce = cudaStreamEndCapture(ctx->stream, &graph);
    if (rc) { if (graph) cudaGraphDestroy(graph); return rc; }
    SK_CUDA_CHECK(ctx, ce);
    const cudaError_t ie = cudaGraphInstantiate(&hg->exec, graph, 0);
    cudaGraphDestroy(graph);
    if (ie != cudaSuccess) hg->exec = nullptr;
    SK_CUDA_CHECK(ctx, ie);
    memcpy(hg->p, kp, sizeof(kp));
    memcpy(hg->v, kv, sizeof(kv));
    return STARKV_OK;
  }
  SK_CUDA_CHECK(ctx, cudaGraphLaunch(hg->exec, ctx->stream));
  SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->pin_free, ctx->stream));
  ctx->pin_busy = 1;
  return STARKV_OK;
}

// One whole decode step from HOST buffers: the inputs of the append and of the decode travel in one pinned block (two
// host-to-device copies, one per device staging area), then starkv_decode_step, one device-to-host copy, one
// synchronisation.  Against starkv_append_host + starkv_decode_attn_host it saves two kernel launches, an event
// hand-shake and a call.
int starkv_decode_step_host(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids_host,
                            const int32_t* positions_host, int batch, const void* k_new_host, int k_row_elems,
                            int64_t k_head_stride, int d_in_k, const void* v_new_host, int v_row_elems, int d_in_v,
                            const void* A_k, const void* A_v, void* append_ws, size_t append_ws_bytes, const void* q_host,
                            const int32_t* seq_lens_host, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                            void* out_host) {
  if (!ctx || batch <= 0 || max_pages <= 0 || !sk_device_ok(ctx)) return STARKV_ERR_INVALID_ARG;
  if (!seq_ids_host || !positions_host || !k_new_host || !v_new_host || !q_host || !seq_lens_host || !out_host || !append_ws ||
      !ws || !aligned16(append_ws) || !aligned16(ws) || k_row_elems <= 0 || v_row_elems <= 0)
    return STARKV_ERR_INVALID_ARG;
  if (append_ws_bytes < starkv_append_host_workspace_bytes(ctx, batch, k_row_elems, v_row_elems)) return STARKV_ERR_WORKSPACE;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  const size_t up = 255;
  const size_t kb = (size_t)batch * k_row_elems * 2, vb = (size_t)batch * v_row_elems * 2, ib = (size_t)batch * 4;
  const bool same = v_new_host == k_new_host;
  const size_t kbp = (kb + up) & ~up, vbp = same ? 0 : ((vb + up) & ~up), ibp = (ib + up) & ~up;
  const size_t qbytes = (size_t)batch * ctx->L.n_q_heads * ctx->L.head_dim * 2;
  const size_t qb = (qbytes + up) & ~up, lb = ibp;
  const size_t app_bytes = kbp + vbp + 2 * ibp, need = app_bytes + 2 * qb + lb;
  if (batch > 64 || need > ((size_t)4 << 20) || ctx->stream == nullptr || ctx->stream == cudaStreamLegacy ||
      ctx->stream == cudaStreamPerThread || ctx->timing_on || sk_stream_capturing(ctx)) {
    // (the pinned staging is for a stream of the caller's own; elsewhere: the two calls)
    const int rc = starkv_append_host(ctx, pool, table, max_pages, seq_ids_host, positions_host, batch, k_new_host, k_row_elems,
                                      k_head_stride, d_in_k, v_new_host, v_row_elems, d_in_v, A_k, A_v, append_ws, append_ws_bytes);
    if (rc) return rc;
    return starkv_decode_attn_host(ctx, q_host, pool, table, max_pages, seq_lens_host, batch, B_k, B_v, ws, ws_bytes, out_host);
  }
  if (ctx->pin_busy) {   // an earlier starkv_append_host may still be reading the block
    SK_CUDA_CHECK(ctx, cudaEventSynchronize(ctx->pin_free));
    ctx->pin_busy = 0;
  }
  {
    const int rc = sk_pin_reserve(ctx, &ctx->pin2, &ctx->pin2_bytes, need, ctx->g_app);
    if (rc) return rc;
  }
  // pinned block: [k][v][seq_ids][positions] | [q][seq_lens] | [out]
  uint8_t* pk = (uint8_t*)ctx->pin2;
  uint8_t* pv = same ? pk : pk + kbp;
  uint8_t* pseq = pk + kbp + vbp;
  uint8_t* ppos = pseq + ibp;
  uint8_t* pq = pk + app_bytes;
  uint8_t* plen = pq + qb;
  uint8_t* pout = plen + lb;
  memcpy(pk, k_new_host, kb);
  if (!same) memcpy(pv, v_new_host, vb);
  memcpy(pseq, seq_ids_host, ib);
  memcpy(ppos, positions_host, ib);
  memcpy(pq, q_host, qbytes);
  memcpy(plen, seq_lens_host, ib);
  // device staging, same layout, behind the projection scratch of the append workspace: ONE copy brings the step's inputs.
  // The result is written by the combine kernel straight into the pinned block (cudaHostAlloc memory is mapped into the
  // device's address space under unified addressing; posted writes, visible to the host once the stream has drained), so
  // there is no copy back.
  const size_t zb = sk_append_ws_bytes(ctx, batch);
  uint8_t* dk = (uint8_t*)append_ws + zb;
  uint8_t* dv = same ? dk : dk + kbp;
  int32_t* dseq = (int32_t*)(dk + kbp + vbp);
  int32_t* dpos = (int32_t*)((uint8_t*)dseq + ibp);
  uint8_t* dq = dk + app_bytes;
  int32_t* dlen = (int32_t*)(dq + qb);
  // ... and where the caller's own `out_host` is page-locked (and so mapped), straight into it: no host copy either
  void* out_dev = pout;
  {
    cudaPointerAttributes at;
    if (cudaPointerGetAttributes(&at, out_host) == cudaSuccess) {
      if (at.type == cudaMemoryTypeHost && at.devicePointer && aligned16(at.devicePointer)) out_dev = at.devicePointer;
    } else {
      (void)cudaGetLastError();
    }
  }
  SK_CUDA_CHECK(ctx, cudaMemcpyAsync(dk, pk, app_bytes + qb + ib, cudaMemcpyHostToDevice, ctx->stream));
  const int rc = starkv_decode_step(ctx, pool, table, max_pages, dseq, dpos, batch, dk, k_row_elems, k_head_stride, d_in_k, dv,
                                    v_row_elems, d_in_v, A_k, A_v, append_ws, zb, dq, dlen, B_k, B_v, ws, ws_bytes, out_dev);
  if (rc) return rc;
  SK_CUDA_CHECK(ctx, cudaStreamSynchronize(ctx->stream));
  if (out_dev == pout) memcpy(out_host, pout, qbytes);
  return STARKV_OK;
}

int starkv_set_kernel_timing(starkv_ctx* ctx, int on) {
  if (!ctx) return STARKV_ERR_INVALID_ARG;
  if (on && !ctx->ev0) {
    SK_CUDA_CHECK(ctx, cudaEventCreate(&ctx->ev0));
    SK_CUDA_CHECK(ctx, cudaEventCreate(&ctx->ev1));
  }
  ctx->timing_on = on ? 1 : 0;
  ctx->timing_valid = 0;
  return STARKV_OK;
}

int starkv_last_decode_kernel_ms(starkv_ctx* ctx, float* ms) {
  if (!ctx || !ms || !ctx->timing_valid) return STARKV_ERR_INVALID_ARG;
  SK_CUDA_CHECK(ctx, cudaEventSynchronize(ctx->ev1));
  SK_CUDA_CHECK(ctx, cudaEventElapsedTime(ms, ctx->ev0, ctx->ev1));
  return STARKV_OK;
}

int starkv_set_splits(starkv_ctx* ctx, int n_splits) {
  if (!ctx || n_splits < 0) return STARKV_ERR_INVALID_ARG;
  ctx->n_splits_override = n_splits;
  return STARKV_OK;
}

int starkv_last_launches(const starkv_ctx* ctx) { return ctx ? ctx->last_launches : 0; }

const char* starkv_last_append_kernel_name(const starkv_ctx* ctx) { return ctx && ctx->last_append ? ctx->last_append : ""; }

const char* starkv_decode_kernel_name(const starkv_ctx* ctx) {
  if (!ctx) return "decode_generic_kernel";
  switch (sk_decode_choice(ctx)) {
    case SK_VARIANT_TM: return "decode_tm_kernel";
    case SK_VARIANT_TC5: return "decode_tc5_kernel";
    case SK_VARIANT_MMA: return "decode_fast_kernel";
    default: return "decode_generic_kernel";
  }
}

int starkv_set_option(starkv_ctx* ctx, const char* name, int value) {
  if (!ctx || !name) return STARKV_ERR_INVALID_ARG;
  if (!strcmp(name, "pdl")) { ctx->pdl = value != 0; return STARKV_OK; }
  if (!strcmp(name, "host_graph")) { ctx->host_graph = value != 0; return STARKV_OK; }
  if (!strcmp(name, "append_tc5")) { ctx->append_tc5 = value != 0; return STARKV_OK; }
  if (!strcmp(name, "decode_variant")) {
    if (value < SK_VARIANT_AUTO || value > SK_VARIANT_GENERIC) return STARKV_ERR_INVALID_ARG;
    const int before = ctx->variant;
    ctx->variant = value;
    sk_fast_plan(ctx);   // the mma.sync / tcgen05-PV choice is part of the plan
    const int got = sk_decode_choice(ctx);
    if (value != SK_VARIANT_AUTO && got != value) {   // the descriptor is not covered by that kernel
      ctx->variant = before;
      sk_fast_plan(ctx);
      return STARKV_ERR_UNSUPPORTED;
    }
    return STARKV_OK;
  }
  return STARKV_ERR_INVALID_ARG;
}

const char* starkv_strerror(int code) {
  switch (code) {
    case STARKV_OK: return "ok";
    case STARKV_ERR_INVALID_ARG: return "invalid argument";
    case STARKV_ERR_UNSUPPORTED: return "unsupported configuration";
    case STARKV_ERR_WORKSPACE: return "workspace too small";
    case STARKV_ERR_CUDA: return "CUDA error";
    default: return "unknown error";
  }
}

const char* starkv_last_error(const starkv_ctx* ctx) { return ctx ? ctx->err : ""; }

}  // extern "C"
