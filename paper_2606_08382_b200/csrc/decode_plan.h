// Host-built plan of the tensor-core decode kernel (decode_fast.cu); passed to the kernel by value.
#pragma once
#include <stdint.h>

#include "starkv_layout.h"

// A "quad" = 4 consecutive query heads = the 8 columns (head, hi/lo) of one QK accumulator tile.
// With G = H_q/H_kv in {1, 2, 4} a quad is fed by 4/G KV heads (block-diagonal in the columns).
// One "q step" = one m16n8k16 MMA of the QK product of one KV head: 16 latent channels of one
// precision block (a 32-channel int4 chunk makes two steps).  The latent-space query image holds, per
// step, the B fragment (q~^T, zero outside the KV head's own columns) for all 32 lanes (uint2 per lane).
struct DecodePlan {
  int32_t nq;                                     // quads = ceil(H_q / 4) <= 8; warp w of a group scores quad w
  int32_t kv_per_quad;                            // 4 / G
  int32_t qstep_begin[STARKV_MAX_KV_HEADS + 1];   // first q step of KV head g
  int32_t n_qsteps;
  int32_t qimg_bytes;                             // n_qsteps * 256
  int32_t nt;                                     // PV n-tiles (8 heads each): 1, 2 or 4
  int32_t mt;                                     // PV m-tiles (16 value channels) per warp: 1..4
  int32_t v_tiles_hi, v_tiles;                    // m-tiles in the leading value block / in total
  int32_t nstage;                                 // page ring depth
  int32_t ng;                                     // groups of 8 warps per CTA: 1 or 2
  // shared-memory carve-up (bytes from the 128-aligned base)
  int32_t off_stage;                              // [nstage][page_bytes]; reused for the final group merge
  int32_t off_qimg;                               // latent-space query image
  int32_t off_p;                                  // [groups][2][P_BUF_BYTES]; P exchange buffers
  int32_t off_alpha;                              // [groups][2][32] float
  int32_t off_flag;                               // [groups][2][8] bytes: "some head of quad w rescaled"
  int32_t off_bar;                                // full[nstage] + image mbarriers, done[nstage] tickets, issued[nstage]
  int32_t off_tbl;                                // block-table entries of the CTA's page range
  int32_t off_kcst;                               // = off_qimg + qimg_bytes: QK accumulator start values
                                                  // [H_kv][2 blocks][4 quad columns] fp32 (same bulk copy as the image)
  int32_t smem_bytes;
  // tcgen05 PV variant (decode_tc5_kernel, integer modes): value page dequantised into a K-major UMMA A operand
  int32_t um;                                     // 1 = use it
  int32_t deq_slice[8];                           // warp gw of a group dequantises item slice deq_slice[gw] (32 threads' worth):
                                                  // the warps with the most QK steps get the lightest slices
  int32_t um_mt;                                  // 128-channel M tiles = ceil(r_v / 128) <= 4
  int32_t um_cols;                                // TMEM columns to allocate (power of two >= 2 groups * um_mt * 32)
  int32_t off_a;                                  // [2 groups][um_mt][16 KB] A operand
};

// channel (inside its precision block) that k index `k` (0..15) of q step `m` of a chunk refers to
//   8/16-bit blocks: chunk = 16 channels, lane j loads channels 4j..4j+3:  k = 8*hi8 + 2j + e -> 4j + 2*hi8 + e
//   4-bit blocks   : chunk = 32 channels, lane j loads channels 8j..8j+7:  -> 8j + 2m + hi8 + 4e
static inline __host__ __device__ int sk_k_to_channel(int bits, int m, int k) {
  const int hi8 = k >> 3, j = (k & 7) >> 1, e = k & 1;
  return bits == 4 ? 8 * j + 2 * m + hi8 + 4 * e : 4 * j + 2 * hi8 + e;
}

// ---------------------------------------------------------------------------------------------
// Host-built plan of the TMEM-operand decode kernel (decode_tm.cu, integer modes).
//
// One iteration = 128 tokens (two 64-token pages) = the 128 TMEM lanes.  Both products run on tcgen05.mma with the
// A operand in tensor memory:
//   QK   S^T[token x (head, block, g)] = codes[token x channel] . Q^T   A = the token's key codes as fp16 subnormals
//        (thread = token = lane writes its own row), B = latent-space query image in shared memory, K = 16 latent
//        channels ("k-step" = two 8-channel octets, each octet inside one (KV head, precision block)), N = a 16-column
//        window of the score tile that covers the columns of the k-step's two octets.
//   PV   O^T[channel x head] += c[channel x token] . P~^T   A = the channel's value codes, exact in fp16 (thread =
//        channel = lane), B = P~ = p * value scale, one operand per precision block.
// ---------------------------------------------------------------------------------------------
#define SK_TM_MAX_TRIPS 10                    // the key-row warps convert four octets (two k-steps) per trip
#define SK_TM_MAX_OCT (4 * SK_TM_MAX_TRIPS)   // octet slots (320 latent channels including padding)
#define SK_TM_MAX_KS (2 * SK_TM_MAX_TRIPS)    // k-steps
struct TmPlan {
  int32_t ok;                       // this descriptor runs on the kernel
  // Octet slots: first every 8-bit octet in cache order (head by head, leading block then trailing block), padded to
  // a multiple of four, then every 4-bit octet likewise.  Grouping by width keeps the conversion loops branch-free.
  int32_t n_trips8, n_trips4;       // trips (four slots) of the two groups
  int32_t n_ks;                     // k-steps of 16 latent channels = 2 (n_trips8 + n_trips4)
  int32_t oct_off[SK_TM_MAX_OCT];   // page byte offset of token slot 0's eight codes (padding slots: 0, read as codes =
                                    // finite values against zero query rows)
  int32_t oct_rowb[SK_TM_MAX_OCT];  // bytes from one token slot to the next
  alignas(16) uint32_t oct_desc[SK_TM_MAX_OCT];   // the two packed for the key-row warps: offset | row bytes << 18
  int32_t blk_oct0[2 * STARKV_MAX_KV_HEADS];   // first octet slot of (KV head h, block b) at [2 h + b]
  int32_t blk_noct[2 * STARKV_MAX_KV_HEADS];   // its octets (consecutive slots)
  int32_t n_pad, pad_oct[8];        // padding slots
  int32_t win[SK_TM_MAX_KS];        // first score column of the k-step's 16-column window (multiple of 8)
  int32_t ds_cols;                  // score-tile columns (multiple of 16, covers every window); column of
                                    // (KV head h, block b, group member g) = (2 h + b) G + g
  // latent-space query image, per sequence: [constant tile: ds_cols x 16][k-step tiles: n_ks x (hi 512 B, lo 512 B)]
  // [scalars: float 2^(24 - e) per (KV head, block)], all B tiles K-major no-swizzle (LBO 128, SBO 256)
  int32_t img_ks_off, img_scal_off, img_bytes;
  // value side
  int32_t n_vt;                     // 128-channel A tiles = ceil(r_v / 128) <= 2
  int32_t n_dt;                     // accumulator tiles = (A tile, precision block) pairs that intersect
  int32_t dt_tile[4], dt_blk[4];
  // tensor memory columns
  int32_t col_do, col_av, col_ak, col_ds;
  int32_t ds_nbuf;                  // score tiles in tensor memory: 2 (double-buffered) where they fit, else 1
  // shared memory (bytes from the 1024-aligned base)
  int32_t k_bytes, ks_bytes, v_bytes, vs_bytes;   // the four parts of a page: key blocks, key scales, value blocks, value scales
  int32_t kstride, vstride, sstride;              // stage strides of the three rings (scales: key scales then value scales)
  int32_t n_kstage, n_vstage, n_sstage;           // ring depths
  int32_t off_kstage, off_vstage, off_sstage, off_img, off_p, off_misc, off_bar, off_tbl, smem_bytes;
};
