/* starkv.h -- C ABI of libstarkv.so: decode attention read directly from a low-rank,
 * mixed-precision-quantised KV cache (STAR-KV, arxiv/paper_2606_08382), hand-written CUDA for
 * sm_100a.  Citations are PAPER.md:L<line> (+ section / equation); "DESIGN.md" is the repo's
 * design file (cache page format v1, readings of the paper).
 *
 * Conventions
 *   - Every `const void*` / `void*` data argument is a DEVICE pointer unless the name ends in
 *     `_host` or the comment says HOST.  The descriptor and its rank tables are HOST memory and
 *     are copied at starkv_create.
 *   - The caller owns every buffer.  starkv_create allocates the context's own device state (64 KB of zeroed
 *     arrival counters); after that the DEVICE-pointer entry points allocate nothing, on the device or the host.
 *     The two `_host` entry points are the exception: on first use (and when a call needs more) they allocate a
 *     pinned host staging block, and with the "host_graph" option they instantiate and cache CUDA graphs; all of
 *     it is freed by starkv_destroy.  The library keeps no reference to caller buffers between calls and never
 *     mutates `seq_lens` or `block_table`.
 *   - Preconditions on index inputs (not checked on the host; the kernels stay memory-safe when they are broken, the
 *     result is then unspecified): 0 <= seq_lens[b] <= max_pages * page_tokens (longer is clamped to the table);
 *     block_table entries of the pages in use are valid page indices of the pool (negative entries are read as
 *     page 0 by decode and skipped by append); append positions lie inside the table (others are skipped).
 *   - Every call only enqueues work on the context's CUDA stream and returns (no host sync);
 *     all entry points are CUDA-graph capturable.  The `_host` variants are the exception: they
 *     copy host buffers in, run, copy the result out and synchronise the stream.
 *   - Return value: 0 = STARKV_OK, negative = error (see enum).  No exception or abort crosses
 *     the ABI.  Inputs must be finite; NaN/Inf in the data are not detected.
 *   - Device pointers must be 16-byte aligned; the page pool 128-byte aligned.
 *   - A context is bound to the device current at starkv_create and to one stream; it is not thread-safe (one
 *     caller at a time per context; different contexts are independent).
 */
#ifndef STARKV_H
#define STARKV_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

enum {
  STARKV_OK = 0,
  STARKV_ERR_INVALID_ARG = -1, /* null / misaligned pointer, bad rank table, bad sizes          */
  STARKV_ERR_UNSUPPORTED = -2, /* bit pair, layout_id, page_tokens or head count not built      */
  STARKV_ERR_WORKSPACE = -3,   /* workspace_bytes smaller than starkv_workspace_bytes()         */
  STARKV_ERR_CUDA = -4         /* a CUDA runtime call failed; text via starkv_last_error()      */
};

/* Cache / attention descriptor (POD, HOST memory).
 *   Keys: head-wise decomposition, one latent cache L_k^h [l, r_h] and one reconstruction
 *   B_k^h [r_h, d_h] per KV head, rank adaptive per head (§4.3.1, §4.3.3).
 *   Values: joint decomposition, one latent L_v [l, r_v] per token shared by all heads,
 *   reconstruction B_v [r_v, H_kv*d_h] (same passages).
 *   Precision split: the leading rank_*_hi channels (highest singular values) are stored at
 *   bits_hi, the rest at bits_lo, quantised per token (§4.4, Eq.12). */
typedef struct {
  int32_t n_q_heads;        /* H_q                                                             */
  int32_t n_kv_heads;       /* H_kv, divides H_q; query head i reads KV head i / (H_q/H_kv)     */
  int32_t head_dim;         /* d_h, multiple of 16, <= 256                                      */
  const int32_t* rank_k;    /* HOST [n_kv_heads] r_h: multiple of 8, 8 <= r_h <= head_dim       */
  const int32_t* rank_k_hi; /* HOST [n_kv_heads] leading high-precision channels: multiple of 8,
                               0 < r_hi <= r_h (ignored when bits_hi == 16)                     */
  int32_t rank_v;           /* r_v: multiple of 8, <= n_kv_heads*head_dim                       */
  int32_t rank_v_hi;        /* multiple of 8, 0 < rank_v_hi <= rank_v                           */
  int32_t bits_hi, bits_lo; /* {16,16} fp16 latents; {8,4}; {8,8}; {4,4}                        */
  int32_t page_tokens;      /* tokens per cache page, multiple of 16 (fast path: 64)            */
  int32_t layout_id;        /* 1 = DESIGN.md "Cache page format v1"                             */
  float sm_scale;           /* softmax scale; <= 0 selects 1/sqrt(head_dim)      */
} starkv_desc;

typedef struct starkv_ctx starkv_ctx; /* opaque: descriptor copy, page byte map, stream */

/* Create a context.  `cuda_stream` is a cudaStream_t (NULL = default stream) on the current
 * device; all later calls enqueue on it.  Errors: INVALID_ARG, UNSUPPORTED, CUDA. */
int starkv_create(starkv_ctx** out, const starkv_desc* desc, void* cuda_stream);
void starkv_destroy(starkv_ctx* ctx);

/* Bytes of one cache page (DESIGN.md format v1: every block padded to 16 B, the page to 128 B). */
size_t starkv_page_bytes(const starkv_ctx* ctx);

/* Bytes of scratch starkv_decode_attn needs for `batch` sequences of at most `max_pages` pages
 * (latent-space queries + split-K partials).  Deterministic in (ctx, batch, max_pages). */
size_t starkv_workspace_bytes(const starkv_ctx* ctx, int batch, int max_pages);

/* Bytes of scratch starkv_append needs for n_new tokens (fp16 latents of the new tokens). */
size_t starkv_append_workspace_bytes(const starkv_ctx* ctx, int n_new);

/* starkv_pack: quantise + pack caller latents into consecutive pages (rows A2-A4 of the hot
 * path on caller-supplied latents).  PAPER.md Eq.12: Z^ = [Q_hi(Z_out) Q_lo(Z_in)], per
 * token; reading of Q in DESIGN.md (symmetric absmax, s = RN_fp16(max|z|/qmax),
 * c = clamp(RNE(z/s), +-qmax), stored offset-binary).
 *   latents_k  fp16 [n_tokens, sum r_h] row-major (head h = columns koff[h] .. koff[h]+r_h)
 *   latents_v  fp16 [n_tokens, r_v]
 *   pages_out  ceil(n_tokens/page_tokens) pages, fully written: slots >= n_tokens and all
 *              padding bytes are zero, so whole pages are bit-comparable. */
int starkv_pack(starkv_ctx* ctx, const void* latents_k, const void* latents_v, int n_tokens,
                void* pages_out);

/* starkv_unpack: inverse of starkv_pack on the first n_tokens slots of consecutive pages.
 * Any output may be NULL.
 *   codes_out    int8  [n_tokens, sum r_h + r_v] signed codes c (quantised modes only)
 *   scales_out   fp16 bits [n_tokens, 2*H_kv + 2]: K (h, blk) then V (blk) (quantised only)
 *   dequant_out  fp32  [n_tokens, sum r_h + r_v] = c*s exactly (or the fp16 latent) */
int starkv_unpack(starkv_ctx* ctx, const void* pages_in, int n_tokens, int8_t* codes_out,
                  uint16_t* scales_out, float* dequant_out);

/* starkv_append: compress-on-append.  PAPER.md §3.2: K' = x (Sigma V)_K per head,
 * V' = x (Sigma V)_V joint; then Eq.12 quantisation and a paged write.  Token j of the n_new
 * new tokens goes to sequence seq_ids[j] at position positions[j]: page
 * block_table[seq_ids[j]*max_pages + positions[j]/page_tokens], slot positions[j]%page_tokens.
 * Other slots of the page are left untouched.  KV head h reads row j of its input at
 * k_new + j*k_row_stride + h*k_head_stride (strides in ELEMENTS), width d_in_k, and multiplies
 * by columns [koff[h], koff[h]+r_h) of A_k:
 *   dense-KV mode   k_head_stride = head_dim, d_in_k = head_dim, d_in_v = H_kv*head_dim
 *   hidden mode     k_head_stride = 0, k_new = v_new = x, d_in_k = d_in_v = d_model
 *   A_k fp16 [d_in_k, sum r_h] row-major, A_v fp16 [d_in_v, r_v] row-major; fp32 accumulation,
 *   one rounding to fp16, then quantise.  seq_ids / positions / block_table: device int32.
 * Two new tokens must not target the same (sequence, position). */
int starkv_append(starkv_ctx* ctx, void* page_pool, const int32_t* block_table, int max_pages,
                  const int32_t* seq_ids, const int32_t* positions, int n_new,
                  const void* k_new, int64_t k_row_stride, int64_t k_head_stride, int d_in_k,
                  const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k,
                  const void* A_v, void* workspace, size_t workspace_bytes);

/* starkv_decode_attn: one decode step of attention read directly from the latent cache
 * (rows D1-D9).  For sequence b with l = seq_lens[b], query head i, KV head g = i/(H_q/H_kv):
 *   q~_i = sm_scale * q_i B_k^gT            (latent-space query; §3.3 L62-68 reordering)
 *   s_t  = q~_i . L_k^g[t]   t in [0, l)     (== sm_scale * q_i . (L_k^g B_k^g)[t], L58)
 *   p    = softmax(s)                        (§3.1)
 *   out_i = ((p L_v)) B_v[:, g*d_h:(g+1)*d_h]   ("(p V') U_V")
 * with L = code*scale dequantised in registers.  l = 0 gives a zero row.  No RoPE (A1).
 *   q fp16 [batch, H_q, d_h]; B_k fp16 [sum r_h, d_h]; B_v fp16 [r_v, H_kv*d_h];
 *   block_table int32 [batch, max_pages]; seq_lens int32 [batch], seq_lens[b] <= max_pages*P;
 *   out fp16 [batch, H_q, d_h]. */
int starkv_decode_attn(starkv_ctx* ctx, const void* q, const void* page_pool,
                       const int32_t* block_table, int max_pages, const int32_t* seq_lens,
                       int batch, const void* B_k, const void* B_v, void* workspace,
                       size_t workspace_bytes, void* out);

/* NEXT-3, latent-output mode: the same attention, but the result is the LATENT row
 *   o~_i = softmax(s_i) . L_v      fp16 [batch, H_q, r_v]
 * and the up-projection by B_v is left to an output projection with U_V absorbed (section 3.3: "(p . V') .
 * U_V", W'_out^i = W_out^i U_V^i).  Arguments as starkv_decode_attn without B_v; same kernels up to the split-K
 * partials, then a merge-only combine.  l = 0 gives a zero row.  Same workspace size and error codes. */
int starkv_decode_attn_latent(starkv_ctx* ctx, const void* q, const void* page_pool,
                              const int32_t* block_table, int max_pages, const int32_t* seq_lens,
                              int batch, const void* B_k, void* workspace, size_t workspace_bytes,
                              void* out_latent);

/* starkv_decode_step: one whole decode step = starkv_append of ONE new token per sequence (n_new = batch, token b at
 * seq_ids[b] / positions[b]) followed by starkv_decode_attn over seq_lens (which already count the new token), with
 * the same arguments, meanings and results as those two calls made back to back on the context's stream -- the cache
 * bytes and `out` are bit-identical to theirs.  What it adds is launch fusion: where a tensor-core decode kernel covers
 * the descriptor and batch <= 16, the append's projection and the latent-space query image run in ONE launch; where
 * the one-launch append applies as well (batch x widest rank x K splits <= 2048: measured faster up to there) that launch also holds the quantiser
 * and the paged write, so the step is three launches (pre, decode, combine) instead of five, else the quantiser /
 * paged write is a launch of its own (four).  Elsewhere it makes the two calls.  append_workspace >=
 * starkv_append_workspace_bytes(ctx, batch), workspace >= starkv_workspace_bytes(...);
 * the two workspaces must not overlap.  Same error codes; on error nothing, the append only, or both may have been
 * enqueued. */
int starkv_decode_step(starkv_ctx* ctx, void* page_pool, const int32_t* block_table, int max_pages,
                       const int32_t* seq_ids, const int32_t* positions, int batch,
                       const void* k_new, int64_t k_row_stride, int64_t k_head_stride, int d_in_k,
                       const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k,
                       const void* A_v, void* append_workspace, size_t append_workspace_bytes,
                       const void* q, const int32_t* seq_lens, const void* B_k, const void* B_v,
                       void* workspace, size_t workspace_bytes, void* out);

/* starkv_decode_attn_static: starkv_decode_attn for callers that cannot allocate (code under CUDA graph capture, tight
 * serving loops, harnesses that forbid cudaMalloc): same arguments, meanings, kernels and result, but NO workspace
 * argument -- the decode scratch (query image, split-K partials) lives in a file-scope device array of
 * STARKV_STATIC_SCRATCH_BYTES that every GPU which loads the library holds until the process exits.  The call makes no
 * cudaMalloc / cudaFree / allocating library call.  A call whose starkv_workspace_bytes(ctx, batch, max_pages) exceeds the
 * array returns STARKV_ERR_WORKSPACE (starkv_last_error names both sizes); 8 MiB covers BASELINE.json configs C2-C5.
 * All calls on a device share the array and it keeps the last call's contents (nothing in it needs to start at zero:
 * each call writes every region before reading it); calls that OVERLAP on the GPU -- two streams, contexts or threads
 * on one device -- race on it: serialise them or use starkv_decode_attn with a workspace per stream.  The first call on
 * a device resolves the array's device address (cudaGetSymbolAddress) and loads the kernels: make it outside a
 * graph capture.  Other error codes as starkv_decode_attn. */
#define STARKV_STATIC_SCRATCH_BYTES (8u << 20)
int starkv_decode_attn_static(starkv_ctx* ctx, const void* q, const void* page_pool,
                              const int32_t* block_table, int max_pages, const int32_t* seq_lens,
                              int batch, const void* B_k, const void* B_v, void* out);

/* Same operation through the plain scalar kernel (any page_tokens / head count; fp32 math,
 * exact dequantisation).  Slow; used as a second implementation in tests and for shapes the
 * tensor-core kernel does not cover. */
int starkv_decode_attn_generic(starkv_ctx* ctx, const void* q, const void* page_pool,
                               const int32_t* block_table, int max_pages,
                               const int32_t* seq_lens, int batch, const void* B_k,
                               const void* B_v, void* workspace, size_t workspace_bytes,
                               void* out);

/* NEXT-1: decode attention with the paper's own key path -- latent keys are cached PRE-RoPE; per token
 * the kernel dequantises, reconstructs K = L_k B_k, applies rotary position embedding at the token's position and then
 * scores against the query (PAPER.md 3.3 L62-68: "RoPE ... is inserted between W_Q and U_K, preventing offline
 * fusion"; A.6 L619-627).  Same arguments as starkv_decode_attn, plus:
 *   q_rotated   the query AFTER its own rotation (the caller rotates q at the current position, as for dense attention)
 *   pos_offset  device int32 [batch] or NULL: token t of sequence b sits at position pos_offset[b] + t (NULL = 0)
 *   rope_theta  the base (10000 for LLaMA-2, 500000 for LLaMA-3.x); must be > 1
 * Pairing: half-split (channel i with i + head_dim/2, angle position * theta^(-2i/head_dim)) -- the paper does not state
 * it; reading R1.  This entry point runs a scalar, correctness-first kernel (r_h * head_dim multiply-adds per
 * token and head; r_h <= 128); values, split-K and combine are the ones of starkv_decode_attn.  Same error codes. */
int starkv_decode_attn_rope(starkv_ctx* ctx, const void* q_rotated, const void* page_pool,
                            const int32_t* block_table, int max_pages, const int32_t* seq_lens,
                            const int32_t* pos_offset, float rope_theta, int batch, const void* B_k,
                            const void* B_v, void* workspace, size_t workspace_bytes, void* out);

/* The two HOST-buffer variants below stage their host inputs in a pinned block owned by the context when the
 * context has a stream of its own (not the legacy / per-thread default stream): the caller's buffers are read
 * before the call returns, one host-to-device copy carries all inputs of the call, and with the "host_graph" option (starkv_set_option) in
 * the environment the copies and kernels of a call signature are replayed as one cached CUDA graph. */

/* HOST-buffer variant (bench.py "e2e"): q_host / seq_lens_host / out_host are HOST pointers
 * (pinned for best speed); the call copies q and seq_lens to device scratch inside `workspace`
 * (sized by starkv_workspace_bytes, which reserves room for them), runs the decode step,
 * copies `out` back and synchronises the stream.  The cache, block table and factors stay on
 * the device (they are the resident state of a serving process). */
int starkv_decode_attn_host(starkv_ctx* ctx, const void* q_host, const void* page_pool,
                            const int32_t* block_table, int max_pages,
                            const int32_t* seq_lens_host, int batch, const void* B_k,
                            const void* B_v, void* workspace, size_t workspace_bytes,
                            void* out_host);

/* HOST-buffer variant of starkv_append (bench.py "e2e"): k_new_host [n_new, k_row_elems] and
 * v_new_host [n_new, v_row_elems] fp16, seq_ids_host / positions_host int32 [n_new] are HOST
 * pointers (pinned for best speed); strides are the row element counts (k_row_stride =
 * k_row_elems, v_row_stride = v_row_elems).  In hidden mode pass v_new_host == k_new_host (copied
 * once).  The call copies them into `workspace` (sized by starkv_append_host_workspace_bytes, which
 * also leaves room for the q and seq_lens of starkv_decode_step_host) and enqueues the append; it does NOT synchronise (copies and kernels are ordered on the stream;
 * the host buffers must stay unchanged until the stream reaches the end of the call). */
size_t starkv_append_host_workspace_bytes(const starkv_ctx* ctx, int n_new, int k_row_elems,
                                          int v_row_elems);
int starkv_append_host(starkv_ctx* ctx, void* page_pool, const int32_t* block_table, int max_pages,
                       const int32_t* seq_ids_host, const int32_t* positions_host, int n_new,
                       const void* k_new_host, int k_row_elems, int64_t k_head_stride, int d_in_k,
                       const void* v_new_host, int v_row_elems, int d_in_v, const void* A_k,
                       const void* A_v, void* workspace, size_t workspace_bytes);

/* starkv_decode_step with HOST buffers (bench.py "e2e"): starkv_append_host of one new token per sequence followed by
 * starkv_decode_attn_host, as ONE call.  The host inputs of both are gathered in one page-locked block the context owns
 * and reach the device in ONE copy (into the staging area behind the projection scratch of `append_workspace`, which
 * starkv_append_host_workspace_bytes sizes for k_new, v_new, seq_ids, positions, q and seq_lens of `batch` sequences);
 * then the launch-fused step; the result is written by the last kernel directly into page-locked host memory -- into
 * `out_host` itself when that is page-locked (cudaHostAlloc / cudaHostRegister, 16-byte aligned), else into the
 * context's block and copied from there -- so there is no device-to-host copy; one stream synchronisation ends the call.
 * *_host arguments are HOST pointers, read before the call returns; out_host is complete when it returns.  The cache,
 * block table and factors stay on the device.  append_workspace >= starkv_append_host_workspace_bytes(ctx, batch,
 * k_row_elems, v_row_elems), workspace >= starkv_workspace_bytes(ctx, batch, max_pages), both DEVICE memory.  Same
 * results (bit for bit) and error codes as the two calls; on the default / legacy stream, under capture, with kernel
 * timing on or for batch > 64 it simply makes them. */
int starkv_decode_step_host(starkv_ctx* ctx, void* page_pool, const int32_t* block_table, int max_pages,
                            const int32_t* seq_ids_host, const int32_t* positions_host, int batch,
                            const void* k_new_host, int k_row_elems, int64_t k_head_stride, int d_in_k,
                            const void* v_new_host, int v_row_elems, int d_in_v, const void* A_k,
                            const void* A_v, void* append_workspace, size_t append_workspace_bytes,
                            const void* q_host, const int32_t* seq_lens_host, const void* B_k,
                            const void* B_v, void* workspace, size_t workspace_bytes, void* out_host);

/* Kernel timing (bench.py "roofline"): when on, the decode calls record CUDA events on the
 * context's stream directly before and after the main split-K kernel (rows D2-D7).
 * starkv_last_decode_kernel_ms waits for the second event and returns the elapsed milliseconds of
 * the last decode call's main kernel in *ms (STARKV_ERR_INVALID_ARG if timing was off). */
int starkv_set_kernel_timing(starkv_ctx* ctx, int on);
int starkv_last_decode_kernel_ms(starkv_ctx* ctx, float* ms);

/* Tuning knob (0 = automatic): number of split-K ranges per sequence for the next decode calls. */
int starkv_set_splits(starkv_ctx* ctx, int n_splits);

/* Number of kernel launches the last decode/append/pack/unpack call enqueued (for bench.py's
 * gpu_launches claim). */
int starkv_last_launches(const starkv_ctx* ctx);

/* Name of the main split-K kernel (rows D2-D7) starkv_decode_attn launches for this context:
 * "decode_tm_kernel" (integer modes: both products on tcgen05 with their A operands in tensor memory),
 * "decode_tc5_kernel" (integer modes: value product on tcgen05, scores on mma.sync),
 * "decode_fast_kernel" (mma.sync; the fp16 mode) or "decode_generic_kernel" (shapes the tensor-core
 * kernels do not cover).  Static string, never NULL.  Selection: DESIGN.md section 6. */
const char* starkv_decode_kernel_name(const starkv_ctx* ctx);
/* Name of the projection kernel the last starkv_append / starkv_append_host call of this context ran ("" before the first):
 * "append_small_kernel" (n_new <= 16, one launch), "append_gemm_kernel" (TMA + tcgen05), "append_project_mma_kernel",
 * "append_project_kernel" (scalar; unaligned rows). */
const char* starkv_last_append_kernel_name(const starkv_ctx* ctx);

/* Per-context options; the library reads NO environment variables.  Returns STARKV_OK,
 * STARKV_ERR_INVALID_ARG (unknown name / value) or STARKV_ERR_UNSUPPORTED (the context keeps its
 * previous setting).
 *   "decode_variant"  0 automatic (default), 1 mma.sync kernel, 2 tcgen05 value product,
 *                     3 TMEM-operand kernel, 4 scalar kernel; UNSUPPORTED when that kernel does
 *                     not cover the descriptor.  For tests and measurements.
 *   "pdl"             1 (default) launches the kernels of a step with programmatic dependent launch.
 *   "host_graph"      1 makes the HOST-buffer entry points replay a cached CUDA graph per call
 *                     signature (default 0).
 *   "append_tc5"      prefill projection (n_new >= 64): 1 = TMA + tcgen05 GEMM (default), 0 = mma.sync kernel. */
int starkv_set_option(starkv_ctx* ctx, const char* name, int value);

const char* starkv_strerror(int code);
/* Text of the last CUDA error seen by this context ("" if none). */
const char* starkv_last_error(const starkv_ctx* ctx);

#ifdef __cplusplus
}
#endif
#endif /* STARKV_H */
