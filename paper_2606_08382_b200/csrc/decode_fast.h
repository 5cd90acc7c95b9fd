// Host-built plan of the tensor-core decode kernel (passed to the kernels by value).
#pragma once
#include <stdint.h>

#include "starkv_layout.h"

// One "q step" = one m16n8k16 MMA of the QK product for one KV head: 16 latent channels of one precision
// block (int4 blocks: a 32-channel chunk makes two steps).  The latent-space query image holds, per step
// and per 8-column tile, the B fragment of q~^T for all 32 lanes (uint2 per lane).
struct FastPlan {
  int32_t qstep_begin[STARKV_MAX_KV_HEADS + 1];  // first q step of KV head g
  int32_t qk_owner[STARKV_MAX_KV_HEADS];         // head-set (0..3) that scores KV head g
  int32_t n_qsteps;
  int32_t ntq;            // 8-column tiles per KV head = ceil(2*G/8)   (columns = (head, hi/lo))
  int32_t qimg_bytes;     // n_qsteps * ntq * 256
  int32_t nt;             // head tiles of 8 (PV N tiles) = ceil(H_q/8)
  int32_t v_tiles_hi;     // 16-channel M tiles in the leading value block
  int32_t v_tiles;        // total value M tiles
  int32_t it_pages;       // pages per iteration (1 or 2)
  int32_t nstage;         // ring depth
  int32_t stage_bytes;    // it_pages * page_bytes
  // shared-memory byte offsets
  int32_t off_stage, off_qimg, off_s, off_p, off_max, off_alpha, off_bar, smem_bytes;
};

// channel (inside its precision block) that k index `k` (0..15) of q step `m` of a chunk refers to
//   8/16-bit blocks: chunk = 16 channels, lane j loads channels 4j..4j+3:  k = 8*hi8 + 2j + e -> 4j + 2*hi8 + e
//   4-bit blocks   : chunk = 32 channels, lane j loads channels 8j..8j+7:  -> 8j + 2m + hi8 + 4e
static inline __host__ __device__ int fast_k_to_channel(int bits, int m, int k) {
  const int hi8 = k >> 3, j = (k & 7) >> 1, e = k & 1;
  return bits == 4 ? 8 * j + 2 * m + hi8 + 4 * e : 4 * j + 2 * hi8 + e;
}
