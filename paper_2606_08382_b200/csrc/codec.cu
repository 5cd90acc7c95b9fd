// Page codec and compress-on-append kernels (rows A1-A4 and U of the hot path).
//   PAPER.md §3.2 L58 (K' = x (Sigma V)_K per head, V' = x (Sigma V)_V joint),
//   PAPER.md §4.4 L204-210 / Eq.12 L208 (leading channels at bits_hi, trailing at bits_lo, per token),
//   DESIGN.md "Cache page format v1" (token-major K blocks, channel-major V blocks, offset-binary fields).
#include <stdlib.h>

#include "append_small.cuh"
#include "common.cuh"
#include "ctx.h"

namespace {

// ---------------------------------------------------------------------------------------------
// pack: one CTA builds one whole page image in shared memory, then writes it out coalesced.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) pack_kernel(const __grid_constant__ StarkvLayout L,
                                                   const __half* __restrict__ lk,
                                                   const __half* __restrict__ lv, int n_tokens,
                                                   uint8_t* __restrict__ pages) {
  extern __shared__ __align__(16) uint8_t img[];
  float* vs = reinterpret_cast<float*>(img + L.page_bytes);  // [2][P] value scales as float
  const int P = L.page_tokens;
  const int page = blockIdx.x;
  const int t0 = page * P;
  const bool quant = L.bits_hi != 16;

  for (int i = threadIdx.x; i < L.page_bytes / 16; i += blockDim.x) reinterpret_cast<uint4*>(img)[i] = make_uint4(0, 0, 0, 0);
  __syncthreads();

  // keys: one (slot, head, blk) unit per thread -> whole bytes of a token-major row
  for (int u = threadIdx.x; u < L.n_kv_heads * 2 * P; u += blockDim.x) {
    const int slot = u % P, hb = u / P, h = hb >> 1, blk = hb & 1;
    const int tok = t0 + slot;
    if (tok >= n_tokens) continue;
    const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
    if (n == 0) continue;
    const __half* z = lk + (size_t)tok * L.sum_rank_k + L.koff[h] + (blk ? L.k_hi_n[h] : 0);
    const int bits = blk ? L.bits_lo : L.bits_hi;
    uint8_t* row = img + (blk ? L.k_lo_off[h] : L.k_hi_off[h]) + (size_t)slot * (n * bits / 8);
    if (!quant) {
      for (int c = 0; c < n; ++c) reinterpret_cast<__half*>(row)[c] = z[c];
      continue;
    }
    float amax = 0.f;
    for (int c = 0; c < n; ++c) amax = fmaxf(amax, fabsf(__half2float(z[c])));
    const int qmax = sk_qmax(bits);
    const __half s16 = sk_scale_of(amax, qmax);
    const float s = __half2float(s16);
    reinterpret_cast<uint16_t*>(img + L.k_scale_off)[(h * 2 + blk) * P + slot] = sk_half_bits(s16);
    if (bits == 8) {
      for (int c = 0; c < n; ++c) row[c] = (uint8_t)(sk_code_of(__half2float(z[c]), s, qmax) + 128);
    } else {
      for (int c = 0; c < n; c += 2) {
        const int u0 = sk_code_of(__half2float(z[c]), s, qmax) + 8;
        const int u1 = sk_code_of(__half2float(z[c + 1]), s, qmax) + 8;
        row[c >> 1] = (uint8_t)(u0 | (u1 << 4));
      }
    }
  }

  // value scales: one (slot, blk) unit per thread
  if (quant) {
    for (int u = threadIdx.x; u < 2 * P; u += blockDim.x) {
      const int slot = u % P, blk = u / P;
      const int tok = t0 + slot;
      const int n = blk ? L.v_lo_n : L.v_hi_n;
      float s = 0.f;
      if (tok < n_tokens && n > 0) {
        const __half* z = lv + (size_t)tok * L.rank_v + (blk ? L.v_hi_n : 0);
        float amax = 0.f;
        for (int c = 0; c < n; ++c) amax = fmaxf(amax, fabsf(__half2float(z[c])));
        const __half s16 = sk_scale_of(amax, sk_qmax(blk ? L.bits_lo : L.bits_hi));
        reinterpret_cast<uint16_t*>(img + L.v_scale_off)[blk * P + slot] = sk_half_bits(s16);
        s = __half2float(s16);
      }
      vs[blk * P + slot] = s;
    }
  }
  __syncthreads();

  // value fields, channel-major: consecutive threads take consecutive channels (coalesced reads)
  for (int blk = 0; blk < 2; ++blk) {
    const int n = blk ? L.v_lo_n : L.v_hi_n;
    if (n == 0) continue;
    const int bits = blk ? L.bits_lo : L.bits_hi;
    const int c0 = blk ? L.v_hi_n : 0;
    uint8_t* base = img + (blk ? L.v_lo_off : L.v_hi_off);
    if (bits == 16) {
      for (int i = threadIdx.x; i < n * P; i += blockDim.x) {
        const int ch = i % n, slot = i / n, tok = t0 + slot;
        if (tok < n_tokens) reinterpret_cast<__half*>(base)[ch * P + slot] = lv[(size_t)tok * L.rank_v + c0 + ch];
      }
    } else if (bits == 8) {
      for (int i = threadIdx.x; i < n * P; i += blockDim.x) {
        const int ch = i % n, slot = i / n, tok = t0 + slot;
        if (tok < n_tokens)
          base[ch * P + slot] =
              (uint8_t)(sk_code_of(__half2float(lv[(size_t)tok * L.rank_v + c0 + ch]), vs[blk * P + slot], 127) + 128);
      }
    } else {
      for (int i = threadIdx.x; i < n * (P / 2); i += blockDim.x) {
        const int ch = i % n, k = i / n;
        int byte = 0;
        for (int e = 0; e < 2; ++e) {
          const int slot = 2 * k + e, tok = t0 + slot;
          if (tok < n_tokens) {
            const int u = sk_code_of(__half2float(lv[(size_t)tok * L.rank_v + c0 + ch]), vs[blk * P + slot], 7) + 8;
            byte |= u << (4 * e);
          }
        }
        base[ch * (P / 2) + k] = (uint8_t)byte;
      }
    }
  }
  __syncthreads();
  uint4* dst = reinterpret_cast<uint4*>(pages + (size_t)page * L.page_bytes);
  for (int i = threadIdx.x; i < L.page_bytes / 16; i += blockDim.x) dst[i] = reinterpret_cast<uint4*>(img)[i];
}

// ---------------------------------------------------------------------------------------------
// unpack
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void sk_locate(const StarkvLayout& L, int col, int slot, int& bits, int& field_byte,
                                          int& nib, int& scale_idx) {
  // field_byte: byte offset inside the page of the byte holding the field (fp16: first byte);
  // nib: 0/1 nibble selector for 4-bit; scale_idx: index into the page's fp16 scale arrays
  // (K: (h*2+blk)*P+slot relative to k_scale_off; V: encoded as -(1 + blk*P + slot)).
  const int P = L.page_tokens;
  const bool quant = L.bits_hi != 16;
  if (col < L.sum_rank_k) {
    const int h = sk_head_of_col(L, col);
    const int cc = col - L.koff[h];
    const int blk = (quant && cc >= L.k_hi_n[h]) ? 1 : 0;
    const int idx = blk ? cc - L.k_hi_n[h] : cc;
    const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
    bits = blk ? L.bits_lo : L.bits_hi;
    const int base = (blk ? L.k_lo_off[h] : L.k_hi_off[h]) + slot * (n * bits / 8);
    field_byte = base + idx * bits / 8;
    nib = (bits == 4) ? (idx & 1) : 0;
    scale_idx = (h * 2 + blk) * P + slot;
  } else {
    const int cc = col - L.sum_rank_k;
    const int blk = (quant && cc >= L.v_hi_n) ? 1 : 0;
    const int idx = blk ? cc - L.v_hi_n : cc;
    bits = blk ? L.bits_lo : L.bits_hi;
    const int base = (blk ? L.v_lo_off : L.v_hi_off) + idx * (P * bits / 8);
    field_byte = base + slot * bits / 8;
    nib = (bits == 4) ? (slot & 1) : 0;
    scale_idx = -(1 + blk * P + slot);
  }
}

__global__ void unpack_kernel(const __grid_constant__ StarkvLayout L, const uint8_t* __restrict__ pages,
                              int n_tokens, int8_t* __restrict__ codes, uint16_t* __restrict__ scales,
                              float* __restrict__ deq) {
  const int P = L.page_tokens;
  const int R = L.sum_rank_k + L.rank_v;
  const bool quant = L.bits_hi != 16;
  const long long total = (long long)n_tokens * R;
  for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < total;
       i += (long long)gridDim.x * blockDim.x) {
    const int tok = (int)(i / R), col = (int)(i % R);
    const uint8_t* pg = pages + (size_t)(tok / P) * L.page_bytes;
    int bits, fb, nib, si;
    sk_locate(L, col, tok % P, bits, fb, nib, si);
    if (!quant) {
      if (deq) deq[i] = __half2float(*reinterpret_cast<const __half*>(pg + fb));
      continue;
    }
    int u = pg[fb];
    if (bits == 4) u = (u >> (4 * nib)) & 0xF;
    const int c = u - (1 << (bits - 1));
    if (codes) codes[i] = (int8_t)c;
    if (deq) {
      const uint16_t sb = si >= 0 ? reinterpret_cast<const uint16_t*>(pg + L.k_scale_off)[si]
                                  : reinterpret_cast<const uint16_t*>(pg + L.v_scale_off)[-si - 1];
      deq[i] = (float)c * __half2float(__ushort_as_half(sb));
    }
  }
  if (quant && scales) {
    const long long ts = (long long)n_tokens * L.n_scales;
    for (long long i = blockIdx.x * (long long)blockDim.x + threadIdx.x; i < ts;
         i += (long long)gridDim.x * blockDim.x) {
      const int tok = (int)(i / L.n_scales), k = (int)(i % L.n_scales);
      const uint8_t* pg = pages + (size_t)(tok / P) * L.page_bytes;
      const int slot = tok % P;
      scales[i] = k < 2 * L.n_kv_heads ? reinterpret_cast<const uint16_t*>(pg + L.k_scale_off)[k * P + slot]
                                       : reinterpret_cast<const uint16_t*>(pg + L.v_scale_off)[(k - 2 * L.n_kv_heads) * P + slot];
    }
  }
}

// ---------------------------------------------------------------------------------------------
// append, step A1: latent projection  z = fp16( X . A )  (fp32 accumulation)
//   blockIdx.x < H_kv : key head h (input row at k_new + j*row_stride + h*head_stride, d_in_k wide)
//   blockIdx.x >= H_kv: 128-column chunk of the joint value projection
//   blockIdx.y        : tile of APP_TOK new tokens
// ---------------------------------------------------------------------------------------------
constexpr int APP_TOK = 16;
constexpr int APP_KC = 64;

__global__ void __launch_bounds__(128) append_project_kernel(
    const __grid_constant__ StarkvLayout L, int n_new, const __half* __restrict__ k_new, long long k_row_stride,
    long long k_head_stride, int d_in_k, const __half* __restrict__ v_new, long long v_row_stride, int d_in_v,
    const __half* __restrict__ A_k, const __half* __restrict__ A_v, __half* __restrict__ z) {
  __shared__ float xs[APP_TOK][APP_KC + 1];
  const int R = L.sum_rank_k + L.rank_v;
  const int j0 = blockIdx.y * APP_TOK;
  const bool is_k = (int)blockIdx.x < L.n_kv_heads;
  const int h = blockIdx.x;
  const __half* x0;
  long long xstride;
  int d_in, ncols, col_out0, lda;
  const __half* A;
  if (is_k) {
    x0 = k_new + (long long)h * k_head_stride; xstride = k_row_stride; d_in = d_in_k;
    ncols = L.rank_k[h]; col_out0 = L.koff[h]; A = A_k + L.koff[h]; lda = L.sum_rank_k;
  } else {
    const int c0 = (blockIdx.x - L.n_kv_heads) * 128;
    x0 = v_new; xstride = v_row_stride; d_in = d_in_v;
    ncols = min(128, L.rank_v - c0); col_out0 = L.sum_rank_k + c0; A = A_v + c0; lda = L.rank_v;
  }
  for (int cbase = 0; cbase < ncols; cbase += 128) {
    const int c = cbase + threadIdx.x;
    float acc[APP_TOK];
#pragma unroll
    for (int t = 0; t < APP_TOK; ++t) acc[t] = 0.f;
    for (int k0 = 0; k0 < d_in; k0 += APP_KC) {
      __syncthreads();
      for (int i = threadIdx.x; i < APP_TOK * APP_KC; i += blockDim.x) {
        const int t = i / APP_KC, k = i % APP_KC;
        const int j = j0 + t;
        xs[t][k] = (j < n_new && k0 + k < d_in) ? __half2float(x0[(long long)j * xstride + k0 + k]) : 0.f;
      }
      __syncthreads();
      if (c < ncols) {
        const int kmax = min(APP_KC, d_in - k0);
        for (int k = 0; k < kmax; ++k) {
          const float a = __half2float(A[(size_t)(k0 + k) * lda + c]);
#pragma unroll
          for (int t = 0; t < APP_TOK; ++t) acc[t] = fmaf(xs[t][k], a, acc[t]);
        }
      }
    }
    if (c < ncols) {
#pragma unroll
      for (int t = 0; t < APP_TOK; ++t)
        if (j0 + t < n_new) z[(size_t)(j0 + t) * R + col_out0 + c] = __float2half_rn(acc[t]);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// append for a handful of new tokens (decode-time append, n_new <= 16): projection, quantiser and paged write in one
// launch (append_small.cuh).  grid (column tiles of keys then values, K splits), 256 threads.
// ---------------------------------------------------------------------------------------------
template <bool FUSED>
__global__ void __launch_bounds__(APS_THREADS) append_small_kernel(const __grid_constant__ StarkvLayout L,
                                                                  const __grid_constant__ AppendSmallArgs a) {
  __shared__ __align__(16) float sm[APS_SM_FLOATS];
  sk_pdl_enter();
  append_small_body<FUSED>(L, a, blockIdx.x, blockIdx.y, sm);
}

// ---------------------------------------------------------------------------------------------
// append, step A1 for many new tokens (prefill): z = fp16(X . A) on tensor cores (mma.sync m16n8k16, fp32
// accumulation).  CTA tile 64 tokens x 64 latent columns, K step 32, 4 warps (2 x 2, warp tile 32 x 32),
// 4-stage cp.async pipeline (prefetch distance 3, one block barrier per K step), ldmatrix fragments (A operand from the token-major X tile, B operand by
// ldmatrix.trans from the k-major A tile).  grid (column tiles of keys then values, token tiles).
// Requires 16-byte aligned rows: d_in % 8 == 0, row strides % 8 == 0 (else the scalar kernel runs).
// ---------------------------------------------------------------------------------------------
constexpr int GM = 64, GN = 64, GK = 32, GST = 4;
constexpr int GXS = GK + 8;   // X tile row stride in halves (80 B: conflict-free ldmatrix)
constexpr int GAS = GN + 8;   // A tile row stride in halves (144 B)

__device__ __forceinline__ void cp_async16(void* smem_dst, const void* gsrc, bool pred) {
  const uint32_t d = (uint32_t)__cvta_generic_to_shared(smem_dst);
  const int n = pred ? 16 : 0;   // src-size 0: zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(d), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ uint32_t pack_f2h2(float lo, float hi) {
  const __half2 h = __floats2half2_rn(lo, hi);
  return *reinterpret_cast<const uint32_t*>(&h);
}
__device__ __forceinline__ void cp_async16_s(uint32_t smem_dst, const void* gsrc, bool pred) {
  const int n = pred ? 16 : 0;   // src-size 0: zero fill
  asm volatile("cp.async.cg.shared.global [%0], [%1], 16, %2;" ::"r"(smem_dst), "l"(gsrc), "r"(n) : "memory");
}
__device__ __forceinline__ void ldsm_x4(uint32_t (&r)[4], const void* p) {
  const uint32_t a = (uint32_t)__cvta_generic_to_shared(p);
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t (&r)[4], const void* p) {
  const uint32_t a = (uint32_t)__cvta_generic_to_shared(p);
  asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];" : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]) : "r"(a));
}
__device__ __forceinline__ void hmma16816(float (&d)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

__global__ void __launch_bounds__(128) append_project_mma_kernel(
    const __grid_constant__ StarkvLayout L, int n_new, int n_key_tiles, const __half* __restrict__ k_new,
    long long k_row_stride, long long k_head_stride, int d_in_k, const __half* __restrict__ v_new, long long v_row_stride,
    int d_in_v, const __half* __restrict__ A_k, const __half* __restrict__ A_v, __half* __restrict__ z) {
  __shared__ __align__(16) __half xs[GST][GM * GXS];
  __shared__ __align__(16) __half as[GST][GK * GAS];
  const int R = L.sum_rank_k + L.rank_v;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int wm = warp >> 1, wn = warp & 1;
  const __half* x0;
  long long xstride;
  int d_in, ncols, col_out0, lda;
  const __half* A;
  if ((int)blockIdx.x < n_key_tiles) {
    int h = 0, t = blockIdx.x;
    while (t >= (L.rank_k[h] + GN - 1) / GN) { t -= (L.rank_k[h] + GN - 1) / GN; ++h; }
    const int c0 = t * GN;
    x0 = k_new + (long long)h * k_head_stride; xstride = k_row_stride; d_in = d_in_k;
    ncols = min(GN, L.rank_k[h] - c0); col_out0 = L.koff[h] + c0; A = A_k + L.koff[h] + c0; lda = L.sum_rank_k;
  } else {
    const int c0 = (blockIdx.x - n_key_tiles) * GN;
    x0 = v_new; xstride = v_row_stride; d_in = d_in_v;
    ncols = min(GN, L.rank_v - c0); col_out0 = L.sum_rank_k + c0; A = A_v + c0; lda = L.rank_v;
  }
  const int m0 = blockIdx.y * GM;
  auto load_tiles = [&](int buf, int k0) {
    // X tile: 64 rows x 32 halves = 256 chunks of 16 B, 2 per thread
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int ci = tid + 128 * u, row = ci >> 2, kc = (ci & 3) * 8;
      const bool ok = m0 + row < n_new && k0 + kc < d_in;
      const __half* src = x0 + (long long)(ok ? m0 + row : 0) * xstride + (ok ? k0 + kc : 0);
      cp_async16(&xs[buf][row * GXS + kc], src, ok);
    }
    // A tile: 32 rows (k) x 64 halves = 256 chunks
#pragma unroll
    for (int u = 0; u < 2; ++u) {
      const int ci = tid + 128 * u, row = ci >> 3, nc = (ci & 7) * 8;
      const bool ok = k0 + row < d_in && nc < ncols;
      const __half* src = A + (size_t)(ok ? k0 + row : 0) * lda + (ok ? nc : 0);
      cp_async16(&as[buf][row * GAS + nc], src, ok);
    }
    asm volatile("cp.async.commit_group;" ::: "memory");
  };
  float acc[2][4][4];
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[a][b][e] = 0.f;
  const int nk = (d_in + GK - 1) / GK;
  // prologue: tiles 0 .. GST-2 (empty groups keep the group count uniform)
#pragma unroll
  for (int p = 0; p < GST - 1; ++p) {
    if (p < nk) load_tiles(p, p * GK);
    else asm volatile("cp.async.commit_group;" ::: "memory");
  }
  for (int kt = 0; kt < nk; ++kt) {
    const int buf = kt % GST;
    asm volatile("cp.async.wait_group %0;" ::"n"(GST - 2) : "memory");   // tile kt has landed (this thread's copies)
    __syncthreads();   // ... everyone's; and every warp is done with the stage tile kt + GST - 1 goes into
    if (kt + GST - 1 < nk) load_tiles((kt + GST - 1) % GST, (kt + GST - 1) * GK);
    else asm volatile("cp.async.commit_group;" ::: "memory");
#pragma unroll
    for (int ks = 0; ks < GK; ks += 16) {
      uint32_t af[2][4], bf[2][4];
      // A operand: rows = tokens.  lanes 0-15 address rows 0-15 at k 0, lanes 16-31 the same rows at k + 8
#pragma unroll
      for (int a = 0; a < 2; ++a)
        ldsm_x4(af[a], &xs[buf][(wm * 32 + a * 16 + (lane & 15)) * GXS + ks + (lane >> 4) * 8]);
      // B operand (k-major tile, transposed load): matrices (k 0-7, n 0-7), (k 8-15, n 0-7), (k 0-7, n 8-15), (k 8-15, n 8-15)
#pragma unroll
      for (int b = 0; b < 2; ++b)
        ldsm_x4_trans(bf[b], &as[buf][(ks + (lane & 7) + ((lane >> 3) & 1) * 8) * GAS + wn * 32 + b * 16 + (lane >> 4) * 8]);
#pragma unroll
      for (int a = 0; a < 2; ++a)
#pragma unroll
        for (int b = 0; b < 4; ++b) hmma16816(acc[a][b], af[a], bf[b >> 1][(b & 1) * 2], bf[b >> 1][(b & 1) * 2 + 1]);
    }
  }
  // epilogue: one rounding to fp16, rows = tokens
#pragma unroll
  for (int a = 0; a < 2; ++a)
#pragma unroll
    for (int b = 0; b < 4; ++b) {
      const int col = wn * 32 + b * 8 + 2 * (lane & 3);
      if (col < ncols) {
#pragma unroll
        for (int hh = 0; hh < 2; ++hh) {
          const int row = m0 + wm * 32 + a * 16 + (lane >> 2) + 8 * hh;
          if (row < n_new)
            *reinterpret_cast<__half2*>(z + (size_t)row * R + col_out0 + col) =
                __floats2half2_rn(acc[a][b][2 * hh], acc[a][b][2 * hh + 1]);
        }
      }
    }
}

// ---------------------------------------------------------------------------------------------
// append, steps A2-A4 for n > 16 new tokens: per-token scales, codes, pack, paged write.  One CTA per new token.
// Keys (token-major rows): one warp per (head, precision block), lanes over channels.
// Values are channel-major, so a byte (4-bit) or 8 bytes (8-bit) of a channel row hold neighbouring SLOTS.  When the
// token belongs to an aligned slot octet of its page whose 8 tokens are consecutive entries of this call (a prefill
// chunk in position order: the common case), the octet's FIRST token's CTA does the values of all eight: it loads their
// value latents, takes the 16 scales, and one thread per channel assembles and stores the channel's whole word; the
// other seven CTAs skip the values.  Any other token sets its 4-bit fields with atomicAnd/atomicOr on the containing
// word so that concurrent appends to neighbouring slots cannot lose an update.
// ---------------------------------------------------------------------------------------------
constexpr int AW_THREADS = 512;

__global__ void __launch_bounds__(AW_THREADS) append_write_kernel(const __grid_constant__ StarkvLayout L,
                                                                  const __half* __restrict__ z, const float* __restrict__ zp,
                                                                  int n_part, int n_new, const int32_t* __restrict__ seq_ids,
                                                                  const int32_t* __restrict__ positions,
                                                                  const int32_t* __restrict__ table, int max_pages,
                                                                  uint8_t* __restrict__ pool) {
  extern __shared__ __align__(16) uint8_t sm[];
  __half* zr = reinterpret_cast<__half*>(sm);                                    // [R] this token's latents
  __half* zo = zr + ((L.sum_rank_k + L.rank_v + 7) & ~7);                         // [8][rank_v] the octet's value latents
  __shared__ float vsc[8][2];
  __shared__ int s_oct;   // 0 = no octet (per-field path), 1 = octet leader, 2 = octet member (the leader writes the values)
  sk_pdl_enter();
  const int j = blockIdx.x;
  const int P = L.page_tokens;
  const int R = L.sum_rank_k + L.rank_v;
  const bool quant = L.bits_hi != 16;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int pos = positions[j], sid = seq_ids[j];
  if (pos < 0 || pos / P >= max_pages || sid < 0) return;   // caller error: skip the token rather than write wildly
  const int pidx = table[(size_t)sid * max_pages + pos / P];
  if (pidx < 0) return;
  uint8_t* pg = pool + (size_t)pidx * L.page_bytes;
  const int slot = pos % P;
  const int jb = j - (slot & 7);   // call index of the octet's first token, if the octet is in this call in order
  if (tid == 0) s_oct = 0;
  __syncthreads();
  if (!zp && jb >= 0 && jb + 8 <= n_new) {
    if (tid < 8) {
      const bool ok = seq_ids[jb + tid] == sid && positions[jb + tid] == pos - (slot & 7) + tid;
      const unsigned all = __ballot_sync(0xffu, ok);
      if (tid == 0 && all == 0xffu) s_oct = (slot & 7) == 0 ? 1 : 2;
    }
  }
  if (zp) {   // fp32 partial sums zp[part][token][column] of append_small_kernel<false>, added in order, one rounding
    for (int i = tid; i < R; i += AW_THREADS) {
      float v[APS_KS_MAX];   // all K splits in flight at once, then added in order
#pragma unroll
      for (int p = 0; p < APS_KS_MAX; ++p) v[p] = p < n_part ? __ldcg(zp + ((size_t)p * n_new + j) * R + i) : 0.f;
      float acc = 0.f;
#pragma unroll
      for (int p = 0; p < APS_KS_MAX; ++p) acc += v[p];
      zr[i] = __float2half_rn(acc);
    }
  } else {
    for (int i = tid; i < R / 8; i += AW_THREADS) reinterpret_cast<uint4*>(zr)[i] = reinterpret_cast<const uint4*>(z + (size_t)j * R)[i];
  }
  __syncthreads();
  const int oct = s_oct;
  if (oct == 1) {
    const int v8 = L.rank_v / 8;
    for (int i = tid; i < 8 * v8; i += AW_THREADS)
      reinterpret_cast<uint4*>(zo)[i] = reinterpret_cast<const uint4*>(z + (size_t)(jb + i / v8) * R + L.sum_rank_k)[i % v8];
  }

  // keys: one warp per (head, precision block), lanes over channels
  for (int u = warp; u < L.n_kv_heads * 2; u += AW_THREADS / 32) {
    const int h = u >> 1, blk = u & 1;
    const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
    if (!quant) {
      if (blk) continue;
      __half* row = reinterpret_cast<__half*>(pg + L.k_hi_off[h]) + (size_t)slot * n;
      for (int c = lane; c < n; c += 32) row[c] = zr[L.koff[h] + c];
      continue;
    }
    uint16_t* sc = reinterpret_cast<uint16_t*>(pg + L.k_scale_off) + (h * 2 + blk) * P + slot;
    if (n == 0) {
      if (lane == 0) *sc = 0;
      continue;
    }
    const __half* zz = zr + L.koff[h] + (blk ? L.k_hi_n[h] : 0);
    const int bits = blk ? L.bits_lo : L.bits_hi;
    const int qmax = sk_qmax(bits);
    float amax = 0.f;
    for (int c = lane; c < n; c += 32) amax = fmaxf(amax, fabsf(__half2float(zz[c])));
#pragma unroll
    for (int o = 16; o; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
    const __half s16 = sk_scale_of(amax, qmax);
    const float sf = __half2float(s16);
    if (lane == 0) *sc = sk_half_bits(s16);
    uint8_t* row = pg + (blk ? L.k_lo_off[h] : L.k_hi_off[h]) + (size_t)slot * (n * bits / 8);
    if (bits == 8) {
      for (int c = lane; c < n; c += 32) row[c] = (uint8_t)(sk_code_of(__half2float(zz[c]), sf, qmax) + 128);
    } else {
      for (int c = lane; c < n / 2; c += 32) {
        const int u0 = sk_code_of(__half2float(zz[2 * c]), sf, qmax) + 8;
        const int u1 = sk_code_of(__half2float(zz[2 * c + 1]), sf, qmax) + 8;
        row[c] = (uint8_t)(u0 | (u1 << 4));
      }
    }
  }
  if (oct == 2) return;   // (CTA-uniform) the octet's first token writes this token's values
  __syncthreads();        // zo is complete

  // values: scales of the token (or of the octet's eight tokens), then the channel-major fields
  const int n_tok = oct == 1 ? 8 : 1;
  const __half* zv0 = oct == 1 ? zo : zr + L.sum_rank_k;   // token t's value latents at zv0 + t * rank_v
  if (quant) {
    for (int u = warp; u < n_tok * 2; u += AW_THREADS / 32) {
      const int t = u >> 1, w = u & 1;
      const int n = w ? L.v_lo_n : L.v_hi_n;
      const __half* zv = zv0 + (size_t)t * L.rank_v + (w ? L.v_hi_n : 0);
      float amax = 0.f;
      for (int c = lane; c < n; c += 32) amax = fmaxf(amax, fabsf(__half2float(zv[c])));
#pragma unroll
      for (int o = 16; o; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      if (lane == 0) {
        const __half s16 = n ? sk_scale_of(amax, sk_qmax(w ? L.bits_lo : L.bits_hi)) : __float2half(0.f);
        vsc[t][w] = __half2float(s16);
        reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[w * P + slot + t] = sk_half_bits(s16);
      }
    }
    __syncthreads();
  }
  for (int c = tid; c < L.rank_v; c += AW_THREADS) {
    const int blk = (quant && c >= L.v_hi_n) ? 1 : 0;
    const int idx = blk ? c - L.v_hi_n : c;
    const int bits = blk ? L.bits_lo : L.bits_hi;
    uint8_t* base = pg + (blk ? L.v_lo_off : L.v_hi_off);
    const __half* zc = zv0 + c;
    if (oct == 1) {   // slots [slot, slot + 8) of the channel row at once
      if (bits == 16) {
        uint32_t w[4];
#pragma unroll
        for (int t = 0; t < 8; t += 2)
          w[t >> 1] = (uint32_t)__half_as_ushort(zc[(size_t)t * L.rank_v]) | ((uint32_t)__half_as_ushort(zc[(size_t)(t + 1) * L.rank_v]) << 16);
        *reinterpret_cast<uint4*>(base + ((size_t)idx * P + slot) * 2) = make_uint4(w[0], w[1], w[2], w[3]);
      } else if (bits == 8) {
        uint32_t w[2] = {0u, 0u};
#pragma unroll
        for (int t = 0; t < 8; ++t)
          w[t >> 2] |= (uint32_t)(sk_code_of(__half2float(zc[(size_t)t * L.rank_v]), vsc[t][blk], 127) + 128) << (8 * (t & 3));
        *reinterpret_cast<uint2*>(base + (size_t)idx * P + slot) = make_uint2(w[0], w[1]);
      } else {
        uint32_t w = 0u;
#pragma unroll
        for (int t = 0; t < 8; ++t) w |= (uint32_t)(sk_code_of(__half2float(zc[(size_t)t * L.rank_v]), vsc[t][blk], 7) + 8) << (4 * t);
        *reinterpret_cast<uint32_t*>(base + (size_t)idx * (P / 2) + (slot >> 1)) = w;
      }
    } else if (bits == 16) {
      reinterpret_cast<__half*>(base)[(size_t)idx * P + slot] = zc[0];
    } else if (bits == 8) {
      base[(size_t)idx * P + slot] = (uint8_t)(sk_code_of(__half2float(zc[0]), vsc[0][blk], 127) + 128);
    } else {
      const unsigned u = (unsigned)(sk_code_of(__half2float(zc[0]), vsc[0][blk], 7) + 8);
      const size_t byte = (size_t)idx * (P / 2) + (slot >> 1);
      unsigned* word = reinterpret_cast<unsigned*>(base + (byte & ~(size_t)3));
      const int sh = 8 * (int)(byte & 3) + 4 * (slot & 1);
      atomicAnd(word, ~(0xFu << sh));
      atomicOr(word, u << sh);
    }
  }
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host side
// ---------------------------------------------------------------------------------------------
int sk_pack(starkv_ctx* ctx, const void* lk, const void* lv, int n_tokens, void* pages) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (n_tokens < 0) return STARKV_ERR_INVALID_ARG;
  if (n_tokens == 0) return STARKV_OK;
  if (!lk || !lv || !pages) return STARKV_ERR_INVALID_ARG;
  const int n_pages = (n_tokens + L.page_tokens - 1) / L.page_tokens;
  const size_t smem = (size_t)L.page_bytes + 2 * L.page_tokens * sizeof(float);
  if ((int)smem > ctx->smem_optin) return STARKV_ERR_UNSUPPORTED;
  SK_CUDA_CHECK(ctx, sk_need_smem(ctx, pack_kernel, (int)smem));
  pack_kernel<<<n_pages, 256, smem, ctx->stream>>>(L, (const __half*)lk, (const __half*)lv, n_tokens, (uint8_t*)pages);
  ctx->last_launches = 1;
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  return STARKV_OK;
}

int sk_unpack(starkv_ctx* ctx, const void* pages, int n_tokens, int8_t* codes, uint16_t* scales, float* deq) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (n_tokens < 0) return STARKV_ERR_INVALID_ARG;
  if (n_tokens == 0) return STARKV_OK;
  if (!pages) return STARKV_ERR_INVALID_ARG;
  const long long total = (long long)n_tokens * (L.sum_rank_k + L.rank_v);
  const int blocks = (int)((total + 255) / 256 < 148 * 16 ? (total + 255) / 256 : 148 * 16);
  unpack_kernel<<<blocks, 256, 0, ctx->stream>>>(L, (const uint8_t*)pages, n_tokens, codes, scales, deq);
  ctx->last_launches = 1;
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  return STARKV_OK;
}

size_t sk_append_ws_bytes(const starkv_ctx* ctx, int n_new) {
  const size_t R = (size_t)ctx->L.sum_rank_k + ctx->L.rank_v;
  const size_t n = (size_t)(n_new > 0 ? n_new : 0);
  const size_t b = n <= (size_t)APS_TOK ? n * R * 4 * APS_KS_MAX : n * R * 2;
  return (b + 255) / 256 * 256;
}

int sk_append_small_ok(const starkv_ctx* ctx, int n_new) {
  return n_new > 0 && n_new <= APS_TOK && n_new * ctx->L.rank_v <= APS_ZR_MAX && ctx->tickets != nullptr &&
         ctx->L.n_kv_heads + 1 <= SK_APPEND_TICKETS;
}

void sk_append_small_args(const starkv_ctx* ctx, AppendSmallArgs* a, void* pool, const int32_t* table, int max_pages,
                          const int32_t* seq_ids, const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride,
                          int64_t k_head_stride, int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v,
                          const void* A_k, const void* A_v, void* ws) {
  const StarkvLayout& L = ctx->L;
  int nkt = 0;
  for (int h = 0; h < L.n_kv_heads; ++h) nkt += (L.rank_k[h] + APS_COLS - 1) / APS_COLS;
  const int d_max = d_in_k > d_in_v ? d_in_k : d_in_v;
  const int n_tiles = nkt + (L.rank_v + APS_COLS - 1) / APS_COLS;
  int n_part = (d_max + APS_KCH - 1) / APS_KCH;
  if (n_part > APS_KS_MAX) n_part = APS_KS_MAX;
  a->n_new = n_new; a->n_key_tiles = nkt; a->n_tiles = n_tiles; a->n_part = n_part;
  a->k_new = (const __half*)k_new; a->k_row_stride = k_row_stride; a->k_head_stride = k_head_stride; a->d_in_k = d_in_k;
  a->v_new = (const __half*)v_new; a->v_row_stride = v_row_stride; a->d_in_v = d_in_v;
  a->A_k = (const __half*)A_k; a->A_v = (const __half*)A_v; a->zp = (float*)ws;
  a->seq_ids = seq_ids; a->positions = positions; a->table = table; a->max_pages = max_pages; a->pool = (uint8_t*)pool;
  a->tickets = ctx->tickets + SK_TICKETS;
  a->fused = 1;
  a->x_vec = (((uintptr_t)k_new | (uintptr_t)v_new) & 15) == 0 && ((k_row_stride | k_head_stride | v_row_stride) & 7) == 0 &&
             ((d_in_k | d_in_v) & 7) == 0;
}

// One launch for A1-A4 when the serial tail of a group's last CTA stays small: at most `limit` partial sums to add.
// Measured: against A1 + append_write_kernel the single launch loses above ~2K sums, as a call of its own (C2, 4096 sums:
// 54.6 vs 52.3 us per step) and inside starkv_decode_step, where either form shares its first launch with the query
// image (C2 49.9 vs 47.3 us, C5 55.9 vs 54.4 per layer; C3, 1024 sums: 40.3 vs 41.0, the single launch wins).
int sk_append_small_fused(const starkv_ctx* ctx, int n_new, int n_part, int limit) {
  const StarkvLayout& L = ctx->L;
  int widest = L.rank_v;
  for (int h = 0; h < L.n_kv_heads; ++h) widest = L.rank_k[h] > widest ? L.rank_k[h] : widest;
  return (long long)n_new * widest * n_part <= limit;
}

// A2-A4 after a launch that ran append_small_body<false> with these arguments (the step's pre kernel): quantise, pack
// and write from the K-split partials.
int sk_append_small_write(starkv_ctx* ctx, const AppendSmallArgs* a) {
  const StarkvLayout& L = ctx->L;
  const size_t smem = ((size_t)((L.sum_rank_k + L.rank_v + 7) & ~7) + 8 * (size_t)L.rank_v) * 2;
  if ((int)smem > ctx->smem_optin) return STARKV_ERR_UNSUPPORTED;
  if (smem > 48 * 1024) SK_CUDA_CHECK(ctx, sk_need_smem(ctx, append_write_kernel, (int)smem));
  SK_PREFER_SMEM(ctx, append_write_kernel);
  SK_CUDA_CHECK(ctx, sk_launch(ctx, append_write_kernel, dim3(a->n_new), dim3(AW_THREADS), smem, L, (const __half*)a->zp,
                               (const float*)a->zp, a->n_part, a->n_new, a->seq_ids, a->positions, a->table, a->max_pages, a->pool));
  ctx->last_append = "append_small_kernel";
  return STARKV_OK;
}

int sk_append(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
              const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride, int64_t k_head_stride,
              int d_in_k, const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k, const void* A_v,
              void* ws, size_t ws_bytes) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (n_new < 0 || max_pages <= 0 || d_in_k <= 0 || d_in_v <= 0) return STARKV_ERR_INVALID_ARG;
  if (n_new == 0) return STARKV_OK;
  if (!pool || !table || !seq_ids || !positions || !k_new || !v_new || !A_k || !A_v || !ws) return STARKV_ERR_INVALID_ARG;
  if (ws_bytes < sk_append_ws_bytes(ctx, n_new)) return STARKV_ERR_WORKSPACE;
  __half* z = (__half*)ws;
  const size_t smem = ((size_t)((L.sum_rank_k + L.rank_v + 7) & ~7) + 8 * (size_t)L.rank_v) * 2;   // of append_write_kernel
  if (!sk_append_small_ok(ctx, n_new) && (int)smem > ctx->smem_optin) return STARKV_ERR_UNSUPPORTED;
  const float* zp = nullptr;
  int n_part = 1;
  if (sk_append_small_ok(ctx, n_new)) {
    AppendSmallArgs a;
    sk_append_small_args(ctx, &a, pool, table, max_pages, seq_ids, positions, n_new, k_new, k_row_stride, k_head_stride, d_in_k,
                         v_new, v_row_stride, d_in_v, A_k, A_v, ws);
    ctx->last_append = "append_small_kernel";
    if (sk_append_small_fused(ctx, n_new, a.n_part, 2048)) {
      SK_PREFER_SMEM(ctx, append_small_kernel<true>);
      SK_CUDA_CHECK(ctx, sk_launch(ctx, append_small_kernel<true>, dim3(a.n_tiles, a.n_part), dim3(APS_THREADS), 0, L, a));
      ctx->last_launches = 1;
      return STARKV_OK;
    }
    SK_PREFER_SMEM(ctx, append_small_kernel<false>);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, append_small_kernel<false>, dim3(a.n_tiles, a.n_part), dim3(APS_THREADS), 0, L, a));
    zp = (const float*)ws;
    n_part = a.n_part;
  } else if (d_in_k % 8 == 0 && d_in_v % 8 == 0 && k_row_stride % 8 == 0 && k_head_stride % 8 == 0 && v_row_stride % 8 == 0 &&
             ((uintptr_t)k_new & 15) == 0 && ((uintptr_t)v_new & 15) == 0 && ((uintptr_t)A_k & 15) == 0 &&
             ((uintptr_t)A_v & 15) == 0) {
    int nkt = 0;
    for (int h = 0; h < L.n_kv_heads; ++h) nkt += (L.rank_k[h] + GN - 1) / GN;
    const int nvt = (L.rank_v + GN - 1) / GN;
    // The TMA + tcgen05 GEMM (append_gemm.cu) is the default for n_new >= 64; starkv_set_option(ctx, "append_tc5", 0) forces the
    // mma.sync kernel below (kept as the second implementation the tests compare, and for what the GEMM does not cover).
    const int g = ctx->append_tc5 ? sk_append_gemm(ctx, pool, table, max_pages, seq_ids, positions, n_new, k_new, k_row_stride,
                                                   k_head_stride, d_in_k, v_new, v_row_stride, d_in_v, A_k, A_v, z)
                                  : 0;
    if (g == 2) {   // projection, quantiser and paged write in one kernel
      ctx->last_launches = 1;
      return STARKV_OK;
    }
    if (!g) {
    ctx->last_append = "append_project_mma_kernel";
    SK_PREFER_SMEM(ctx, append_project_mma_kernel);
    append_project_mma_kernel<<<dim3(nkt + nvt, (n_new + GM - 1) / GM), 128, 0, ctx->stream>>>(
        L, n_new, nkt, (const __half*)k_new, k_row_stride, k_head_stride, d_in_k, (const __half*)v_new, v_row_stride, d_in_v,
        (const __half*)A_k, (const __half*)A_v, z);
    }
  } else {
  ctx->last_append = "append_project_kernel";
  dim3 g1(L.n_kv_heads + (L.rank_v + 127) / 128, (n_new + APP_TOK - 1) / APP_TOK);
  append_project_kernel<<<g1, 128, 0, ctx->stream>>>(L, n_new, (const __half*)k_new, k_row_stride, k_head_stride, d_in_k,
                                                     (const __half*)v_new, v_row_stride, d_in_v, (const __half*)A_k,
                                                     (const __half*)A_v, z);
  }
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  if (smem > 48 * 1024) SK_CUDA_CHECK(ctx, sk_need_smem(ctx, append_write_kernel, (int)smem));
  SK_PREFER_SMEM(ctx, append_write_kernel);
  sk_launch(ctx, append_write_kernel, dim3(n_new), dim3(AW_THREADS), smem, L, (const __half*)z, zp, n_part, n_new,
            seq_ids, positions, table, max_pages, (uint8_t*)pool);
  ctx->last_launches = 2;
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  return STARKV_OK;
}
