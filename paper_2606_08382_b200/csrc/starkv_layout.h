// Byte map of one latent-cache page, written from DESIGN.md "Cache page format v1".
// (The CPU oracle has its own, independent, restatement of the same text.)
#pragma once
#include <stdint.h>

#define STARKV_MAX_KV_HEADS 64
#define STARKV_MAX_Q_HEADS 128

// Everything the kernels need to find a field inside a page.  POD; passed by value / __grid_constant__.
struct StarkvLayout {
  int32_t n_q_heads, n_kv_heads, head_dim, group;
  int32_t bits_hi, bits_lo;      // 16/16 = fp16 mode
  int32_t page_tokens;           // P
  int32_t page_bytes;
  int32_t sum_rank_k;            // sum r_h
  int32_t rank_v, v_hi_n, v_lo_n;
  int32_t k_scale_off;           // byte offset of K_scales[H_kv][2][P] (-1 in fp16 mode)
  int32_t v_hi_off, v_lo_off;    // channel-major blocks
  int32_t v_scale_off;           // V_scales[2][P] (-1 in fp16 mode)
  int32_t n_scales;              // 2*H_kv + 2
  float sm_scale;
  int32_t rank_k[STARKV_MAX_KV_HEADS];   // r_h
  int32_t koff[STARKV_MAX_KV_HEADS];     // first latent column of head h
  int32_t k_hi_n[STARKV_MAX_KV_HEADS];   // channels in the leading block (r_h in fp16 mode)
  int32_t k_lo_n[STARKV_MAX_KV_HEADS];
  int32_t k_hi_off[STARKV_MAX_KV_HEADS]; // byte offsets, token-major blocks
  int32_t k_lo_off[STARKV_MAX_KV_HEADS];
};

static inline int32_t starkv_up(int64_t x, int32_t m) { return (int32_t)((x + m - 1) / m * m); }

// Returns 0 on success, -1 invalid, -2 unsupported.
static inline int starkv_build_layout(StarkvLayout* L, int n_q, int n_kv, int d_h, const int32_t* rk,
                                      const int32_t* rk_hi, int rv, int rv_hi, int bits_hi, int bits_lo,
                                      int P, float sm_scale) {
  if (n_q <= 0 || n_kv <= 0 || n_q % n_kv != 0 || n_kv > STARKV_MAX_KV_HEADS || n_q > STARKV_MAX_Q_HEADS) return -1;
  if (d_h <= 0 || d_h % 16 != 0 || d_h > 256) return -1;
  if (P <= 0 || P % 16 != 0) return -1;
  if (!((bits_hi == 16 && bits_lo == 16) || (bits_hi == 8 && bits_lo == 4) || (bits_hi == 8 && bits_lo == 8) ||
        (bits_hi == 4 && bits_lo == 4)))
    return -2;
  const bool q = bits_hi != 16;
  if (rv <= 0 || rv % 8 != 0 || rv > n_kv * d_h) return -1;
  if (q && (rv_hi <= 0 || rv_hi % 8 != 0 || rv_hi > rv)) return -1;
  L->n_q_heads = n_q; L->n_kv_heads = n_kv; L->head_dim = d_h; L->group = n_q / n_kv;
  L->bits_hi = bits_hi; L->bits_lo = bits_lo; L->page_tokens = P; L->rank_v = rv;
  L->sm_scale = sm_scale;
  int64_t off = 0;
  int32_t col = 0;
  for (int h = 0; h < n_kv; ++h) {
    const int r = rk[h];
    if (r <= 0 || r % 8 != 0 || r > d_h) return -1;
    int hi = r, lo = 0;
    if (q) {
      hi = rk_hi[h];
      if (hi <= 0 || hi % 8 != 0 || hi > r) return -1;
      lo = r - hi;
    }
    L->rank_k[h] = r; L->koff[h] = col; col += r;
    L->k_hi_n[h] = hi; L->k_lo_n[h] = lo;
    L->k_hi_off[h] = (int32_t)off; off += starkv_up((int64_t)P * hi * bits_hi / 8, 16);
    L->k_lo_off[h] = (int32_t)off; off += starkv_up((int64_t)P * lo * bits_lo / 8, 16);
  }
  for (int h = n_kv; h < STARKV_MAX_KV_HEADS; ++h) {
    L->rank_k[h] = L->koff[h] = L->k_hi_n[h] = L->k_lo_n[h] = L->k_hi_off[h] = L->k_lo_off[h] = 0;
  }
  L->sum_rank_k = col;
  L->k_scale_off = -1;
  if (q) { L->k_scale_off = (int32_t)off; off += starkv_up((int64_t)n_kv * 2 * P * 2, 16); }
  L->v_hi_n = q ? rv_hi : rv;
  L->v_lo_n = q ? rv - rv_hi : 0;
  L->v_hi_off = (int32_t)off; off += starkv_up((int64_t)L->v_hi_n * P * bits_hi / 8, 16);
  L->v_lo_off = (int32_t)off; off += starkv_up((int64_t)L->v_lo_n * P * bits_lo / 8, 16);
  L->v_scale_off = -1;
  if (q) { L->v_scale_off = (int32_t)off; off += starkv_up((int64_t)2 * P * 2, 16); }
  L->n_scales = 2 * n_kv + 2;
  off = starkv_up(off, 128);
  if (off > (int64_t)1 << 30) return -1;
  L->page_bytes = (int32_t)off;
  return 0;
}
