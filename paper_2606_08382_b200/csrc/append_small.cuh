// Compress-on-append for a handful of new tokens (decode: one per sequence), all of A1-A4 in ONE launch
// (section 3.2 L56-60 projection, Eq.12 L208 quantiser; A11, A15).
//
//   A1  z = X . A for <= 16 tokens: a GEMV-like problem whose cost is reading A once.  One CTA per (64 latent columns,
//       256-wide K chunk), all tokens at once: each warp keeps 32 rows of A in registers (coalesced half2 per lane and
//       row); the fp32 partial sums go to zp[k split][token][column].
//   A2-A4  The CTAs of one GROUP (a KV head's key columns, or the joint value columns) count their arrivals on a ticket;
//       the last one adds the K splits in a fixed order (deterministic), rounds once to fp16, takes the per-token
//       absmax of each precision block, quantises, packs and writes the page fields of its group for every new token.
//       4-bit value fields share a byte between two slots: set with atomicAnd/atomicOr on the containing word so that
//       concurrent appends to neighbouring slots cannot lose an update.
// The body is a device function so that the decode step can run it in the same launch as the query image
// (step_pre_tm_kernel, decode_tm.cu).
#pragma once
#include "common.cuh"

constexpr int APS_COLS = 64, APS_KCH = 256, APS_TOK = 16, APS_KS_MAX = 16;   // K splits = ceil(d_in / 256) <= 16
constexpr int APS_THREADS = 256;
constexpr int APS_SM_FLOATS = 8 * APS_TOK * APS_COLS;                        // 32 KB of shared memory
constexpr int APS_ZR_MAX = APS_SM_FLOATS * 2;                                // fp16 staging of a group's rows

struct AppendSmallArgs {
  int n_new, n_key_tiles, n_tiles, n_part;
  int x_vec;      // both inputs: 16-byte aligned rows and d_in % 8 == 0
  int fused;      // host side only: A1-A4 in this launch (else A1 here, then append_write_kernel reads the partials)
  const __half* k_new;
  long long k_row_stride, k_head_stride;
  int d_in_k;
  const __half* v_new;
  long long v_row_stride;
  int d_in_v;
  const __half* A_k;
  const __half* A_v;
  float* zp;
  const int32_t* seq_ids;
  const int32_t* positions;
  const int32_t* table;
  int max_pages;
  uint8_t* pool;
  int* tickets;   // n_kv_heads + 1 zeroed counters, reset by the last arriver
};

// page index (-1: the caller's ids are out of range, the token is skipped, never written wildly) and slot of new token j
__device__ __forceinline__ void aps_lookup(const StarkvLayout& L, const AppendSmallArgs& a, int j, int* pidx, int* slot) {
  const int P = L.page_tokens;
  const int pos = a.positions[j], sid = a.seq_ids[j];
  *pidx = -1;
  *slot = 0;
  if (pos < 0 || pos / P >= a.max_pages || sid < 0) return;
  *pidx = a.table[(size_t)sid * a.max_pages + pos / P];
  *slot = pos % P;
}
// the same from the table every CTA fills at its start (two dependent global loads hidden behind the projection instead
// of sitting in the last CTA's serial tail)
__device__ __forceinline__ uint8_t* aps_page_of(const StarkvLayout& L, const AppendSmallArgs& a, const int* s_pidx,
                                                const int* s_slot, int j, int* slot) {
  const int pidx = s_pidx[j];
  if (pidx < 0) return nullptr;
  *slot = s_slot[j];
  return a.pool + (size_t)pidx * L.page_bytes;
}

// bx = column tile (keys of head 0.., then values), by = K split.  `sm` = APS_SM_FLOATS floats of shared memory.
// FUSED = false stops after the partial sums (A1 only): a large group (many tokens x wide value rank x many K splits)
// is too much serial work for one last-arriving CTA, so append_write_kernel, one CTA per token, does A2-A4 instead.
template <bool FUSED>
__device__ __forceinline__ void append_small_body(const StarkvLayout& L, const AppendSmallArgs& a, int bx, int by, float* sm) {
  __shared__ int s_last;
  __shared__ float s_vsc[APS_TOK][2];
  __shared__ int s_pidx[APS_TOK], s_slot[APS_TOK];
  if (FUSED && threadIdx.x < a.n_new) aps_lookup(L, a, threadIdx.x, &s_pidx[threadIdx.x], &s_slot[threadIdx.x]);
  const int R = L.sum_rank_k + L.rank_v;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n_new = a.n_new;
  const __half* x0;
  long long xstride;
  int d_in, ncols, col_out0, lda, group, group_tiles;
  const __half* A;
  if (bx < a.n_key_tiles) {
    int h = 0, t = bx;
    while (t >= (L.rank_k[h] + APS_COLS - 1) / APS_COLS) { t -= (L.rank_k[h] + APS_COLS - 1) / APS_COLS; ++h; }
    const int c0 = t * APS_COLS;
    x0 = a.k_new + (long long)h * a.k_head_stride; xstride = a.k_row_stride; d_in = a.d_in_k;
    ncols = min(APS_COLS, L.rank_k[h] - c0); col_out0 = L.koff[h] + c0; A = a.A_k + L.koff[h] + c0; lda = L.sum_rank_k;
    group = h; group_tiles = (L.rank_k[h] + APS_COLS - 1) / APS_COLS;
  } else {
    const int c0 = (bx - a.n_key_tiles) * APS_COLS;
    x0 = a.v_new; xstride = a.v_row_stride; d_in = a.d_in_v;
    ncols = min(APS_COLS, L.rank_v - c0); col_out0 = L.sum_rank_k + c0; A = a.A_v + c0; lda = L.rank_v;
    group = L.n_kv_heads; group_tiles = a.n_tiles - a.n_key_tiles;
  }
  const int per = ((d_in + a.n_part - 1) / a.n_part + 31) / 32 * 32;
  const int k_begin = by * per, k_end = min(d_in, k_begin + per);
  float acc[APS_TOK][2];
#pragma unroll
  for (int t = 0; t < APS_TOK; ++t) acc[t][0] = acc[t][1] = 0.f;
  const bool col_ok = 2 * lane < ncols;
  for (int kc = k_begin; kc < k_end; kc += APS_KCH) {
    // this warp's 32 rows of A first (independent loads, all in flight), then the x chunk
    const int kw = kc + warp * 32;
    const int kn = col_ok ? max(0, min(32, k_end - kw)) : 0;
    uint32_t av[32];
    {
      const __half* ap = A + (size_t)kw * lda + 2 * lane;
#pragma unroll
      for (int kk = 0; kk < 32; ++kk) av[kk] = kk < kn ? *reinterpret_cast<const uint32_t*>(ap + (size_t)kk * lda) : 0u;
    }
    uint4 xv[2];
    if (a.x_vec) {   // 16-byte aligned rows, d_in a multiple of 8: two independent 16-byte loads per thread, in flight
                     // together with the factor rows (issued before the barrier that frees the shared-memory chunk)
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int i = tid + u * APS_THREADS, t = i >> 5, k8 = (i & 31) * 8;
        xv[u] = (t < n_new && kc + k8 < k_end) ? *reinterpret_cast<const uint4*>(x0 + (long long)t * xstride + kc + k8)
                                               : make_uint4(0u, 0u, 0u, 0u);
      }
    }
    __syncthreads();
    if (a.x_vec) {
#pragma unroll
      for (int u = 0; u < 2; ++u) {
        const int i = tid + u * APS_THREADS, t = i >> 5, k8 = (i & 31) * 8;
        const float2 f0 = __half22float2(*reinterpret_cast<const __half2*>(&xv[u].x)), f1 = __half22float2(*reinterpret_cast<const __half2*>(&xv[u].y)),
                     f2 = __half22float2(*reinterpret_cast<const __half2*>(&xv[u].z)), f3 = __half22float2(*reinterpret_cast<const __half2*>(&xv[u].w));
        float4* d = reinterpret_cast<float4*>(sm + t * APS_KCH + k8);
        d[0] = make_float4(f0.x, f0.y, f1.x, f1.y);
        d[1] = make_float4(f2.x, f2.y, f3.x, f3.y);
      }
    } else {
      for (int i = tid; i < APS_TOK * APS_KCH; i += APS_THREADS) {
        const int t = i / APS_KCH, k = i % APS_KCH;
        sm[i] = (t < n_new && kc + k < k_end) ? __half2float(x0[(long long)t * xstride + kc + k]) : 0.f;
      }
    }
    __syncthreads();
    if (kn > 0) {
      const float* xp = sm + warp * 32;
#pragma unroll
      for (int kk = 0; kk < 32; ++kk) {
        const float2 af = __half22float2(*reinterpret_cast<const __half2*>(&av[kk]));
#pragma unroll
        for (int t = 0; t < APS_TOK; ++t) {
          const float x = xp[t * APS_KCH + kk];
          acc[t][0] = fmaf(x, af.x, acc[t][0]);
          acc[t][1] = fmaf(x, af.y, acc[t][1]);
        }
      }
    }
  }
  __syncthreads();
#pragma unroll
  for (int t = 0; t < APS_TOK; ++t)
    *reinterpret_cast<float2*>(sm + (warp * APS_TOK + t) * APS_COLS + 2 * lane) = make_float2(acc[t][0], acc[t][1]);
  __syncthreads();
  for (int i = tid; i < APS_TOK * APS_COLS; i += APS_THREADS) {
    const int t = i / APS_COLS, c = i % APS_COLS;
    float s = 0.f;
#pragma unroll
    for (int w = 0; w < 8; ++w) s += sm[(w * APS_TOK + t) * APS_COLS + c];
    if (t < n_new && c < ncols) a.zp[((size_t)by * n_new + t) * R + col_out0 + c] = s;
  }

  if (!FUSED) return;
  // ---- ticket: the last CTA of the group quantises and writes the group's fields
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    const int t = atomicAdd(a.tickets + group, 1);
    const int last = t == group_tiles * a.n_part - 1;
    if (last) a.tickets[group] = 0;
    s_last = last;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();

  const bool quant = L.bits_hi != 16;
  const int P = L.page_tokens;
  const bool is_v = group == L.n_kv_heads;
  const int gcols = is_v ? L.rank_v : L.rank_k[group];
  const int gcol0 = is_v ? L.sum_rank_k : L.koff[group];
  __half* zr = reinterpret_cast<__half*>(sm);   // [token][gcols]
  for (int i = tid; i < n_new * gcols; i += APS_THREADS) {
    const int j = i / gcols, c = i - j * gcols;
    float v[APS_KS_MAX];   // all K splits in flight at once, then added in order
#pragma unroll
    for (int p = 0; p < APS_KS_MAX; ++p) v[p] = p < a.n_part ? __ldcg(a.zp + ((size_t)p * n_new + j) * R + gcol0 + c) : 0.f;
    float s = 0.f;
#pragma unroll
    for (int p = 0; p < APS_KS_MAX; ++p) s += v[p];
    zr[i] = __float2half_rn(s);
  }
  __syncthreads();

  if (!is_v) {
    // keys: one warp per (token, precision block), lanes over channels
    const int h = group;
    for (int u = warp; u < n_new * 2; u += APS_THREADS / 32) {
      const int j = u >> 1, blk = u & 1;
      int slot;
      uint8_t* pg = aps_page_of(L, a, s_pidx, s_slot, j, &slot);
      if (!pg) continue;
      const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
      if (!quant) {
        if (blk) continue;
        __half* row = reinterpret_cast<__half*>(pg + L.k_hi_off[h]) + (size_t)slot * n;
        for (int c = lane; c < n; c += 32) row[c] = zr[j * gcols + c];
        continue;
      }
      uint16_t* sc = reinterpret_cast<uint16_t*>(pg + L.k_scale_off) + (h * 2 + blk) * P + slot;
      if (n == 0) {
        if (lane == 0) *sc = 0;
        continue;
      }
      const __half* zz = zr + j * gcols + (blk ? L.k_hi_n[h] : 0);
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
    return;
  }

  // values: per-token scales first (a warp per (token, block)), then the channel-major fields
  if (quant) {
    for (int u = warp; u < n_new * 2; u += APS_THREADS / 32) {
      const int j = u >> 1, w = u & 1;
      const int n = w ? L.v_lo_n : L.v_hi_n;
      const int c0 = w ? L.v_hi_n : 0;
      float amax = 0.f;
      for (int c = lane; c < n; c += 32) amax = fmaxf(amax, fabsf(__half2float(zr[j * gcols + c0 + c])));
#pragma unroll
      for (int o = 16; o; o >>= 1) amax = fmaxf(amax, __shfl_xor_sync(0xffffffffu, amax, o));
      if (lane == 0) {
        const __half s16 = n ? sk_scale_of(amax, sk_qmax(w ? L.bits_lo : L.bits_hi)) : __float2half(0.f);
        s_vsc[j][w] = __half2float(s16);
        int slot;
        uint8_t* pg = aps_page_of(L, a, s_pidx, s_slot, j, &slot);
        if (pg) reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[w * P + slot] = sk_half_bits(s16);
      }
    }
    __syncthreads();
  }
  for (int i = tid; i < n_new * gcols; i += APS_THREADS) {
    const int j = i / gcols, c = i - j * gcols;
    int slot;
    uint8_t* pg = aps_page_of(L, a, s_pidx, s_slot, j, &slot);
    if (!pg) continue;
    const int blk = (quant && c >= L.v_hi_n) ? 1 : 0;
    const int idx = blk ? c - L.v_hi_n : c;
    const int bits = blk ? L.bits_lo : L.bits_hi;
    uint8_t* base = pg + (blk ? L.v_lo_off : L.v_hi_off);
    const __half zv = zr[i];
    if (bits == 16) {
      reinterpret_cast<__half*>(base)[(size_t)idx * P + slot] = zv;
    } else if (bits == 8) {
      base[(size_t)idx * P + slot] = (uint8_t)(sk_code_of(__half2float(zv), s_vsc[j][blk], 127) + 128);
    } else {
      const unsigned u = (unsigned)(sk_code_of(__half2float(zv), s_vsc[j][blk], 7) + 8);
      const size_t byte = (size_t)idx * (P / 2) + (slot >> 1);
      unsigned* word = reinterpret_cast<unsigned*>(base + (byte & ~(size_t)3));
      const int sh = 8 * (int)(byte & 3) + 4 * (slot & 1);
      atomicAnd(word, ~(0xFu << sh));
      atomicOr(word, u << sh);
    }
  }
}
