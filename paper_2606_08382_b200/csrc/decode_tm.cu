// Decode attention over the quantised latent cache with BOTH products on tcgen05.mma and their A operands in tensor
// memory (rows D1-D7 of the hot path, integer modes), sm_100a.
//
//   PAPER.md §3.3: scores in latent space  s_t = q~ . L_k[t]  (no RoPE on this path, A1) and the value
//   side reordered as (p L_v) B_v;  A.6 L627: p stacked over the heads so that p L_v is ONE GEMM;  Eq.12 L208 / A.6 L625:
//   the codes are dequantised in registers and never materialised in memory.
//
// The cache format decides the mapping: key blocks are token-major, value blocks channel-major, and a
// tcgen05.mma A operand in tensor memory is "lane = row".  So for the score product a THREAD IS A TOKEN (it reads its own
// key rows and writes them to its own TMEM lane) and for the value product a THREAD IS A VALUE CHANNEL (it reads its own
// channel rows).  One iteration = 128 tokens = two 64-token pages = the 128 lanes.
//
//   QK   S[token, col] = sum_c u_c Q_c:  A = the offset-binary code fields as fp16 SUBNORMALS (u 2^-24; the odd nibble of
//        a 4-bit byte as 16 u 2^-24, one LOP3 / PRMT per two fields), B = the latent-space query image (qproj_tm_kernel):
//        Q = q~ 2^e as an fp16 hi + lo pair (two MMAs into the same fp32 columns), 1/16 folded into the odd 4-bit
//        channels, e chosen per (KV head, precision block).  One column per (query head, precision block):
//        col = (2 h + blk) G + g, because the per-token scales differ per block.  K = 16 channels = two octets; every
//        k-step writes a 16-column window of the score tile (the B tile is zero outside the octets' own columns).  The
//        code offset 2^(b-1) is one more k-step whose A row is the constant (2^-14, 2^-14, 0...) and whose B tile holds
//        -2^(b-1) 2^-10 sum_c Q_c (hi, lo): it also initialises the tile (accumulate off, N = all columns).
//   softmax  thread = token reads its score columns (tcgen05.ld), applies the per-(token, head, block) key scales in
//        fp32, p' = 2^(s - m + 4) against a LAZY running maximum m, and folds the per-token VALUE scales into two fp16
//        operands P~_blk = p' a, a = 16 s_v / M_blk (M_blk = a running power of two above the scales seen, so the operand
//        cannot overflow), stored MN-major.  m and M_blk move only when p' or the product would near the fp16 limit
//        (a tile exceeding m by about 2^11.5): moving them means rescaling the TMEM accumulators, which drains the
//        pipeline (about 2.8 us), so the first references are the maximum over the range's first 32 tokens and the
//        update path stays out of the common case.
//   PV   O[channel, head] += c[channel, token] P~[token, head]:  A = exact signed codes (magic-number trick), B = P~ of
//        the channel's block; a 128-channel A tile that straddles the block boundary is multiplied with both operands
//        into two accumulator tiles and each lane keeps its own.
// Warp roles (24 warps, warpgroup-aligned so that setmaxnreg can move registers between them; the CTA owns 768 x 80
// registers and the budgets 8 x 64 + 8 x 112 + 4 x 88 + 4 x 40 add up to exactly that -- setmaxnreg.inc can only
// take what another warpgroup of the CTA released):
//   0-3 / 4-7 key rows -> TMEM for the first / second half of the k-steps, 8-11 / 12-15 softmax of the lower / upper
//   half of the query heads, 16-19 value rows -> TMEM, 20 page producer (cp.async.bulk ring), 21 QK MMA issue,
//   22 PV MMA issue, 23 TMEM allocation.
// All hand-offs are mbarriers; there is no CTA-wide barrier in the loop.  The value operand is handed over per page
// (two halves of the 128 tokens), so that the next tile's value rows are converted while the MMAs of this one run.
#include <string.h>

#include "append_small.cuh"
#include "decode_common.cuh"
#include "decode_plan.h"
#include "sk_ptx.cuh"

using namespace skptx;

namespace {

constexpr int PTOK = 64;              // tokens per page on this path
constexpr int TM_THREADS = 768;
constexpr int TM_TBL = 512;           // block-table entries of the CTA's range kept in shared memory
constexpr float P_OFFSET = 4.f;       // p' = 2^(s - m + 4)
constexpr float A_SHIFT = 16.f;       // ... and the value-scale factor carries the other 2^4: a = 16 s_v / M (same product as 2^8 and 1)
constexpr float P_CAP = 46000.f;      // update the references before p' or an operand p' a could exceed this (fp16 holds 65504)
constexpr float kLog2e = 1.4426950408889634f;
constexpr int BAR_SM = 1;             // named barrier of the softmax warps
constexpr int P_BLK_BYTES = 8192;     // P~ operand of one precision block: 128 tokens x 32 heads fp16
constexpr uint32_t TM_COLS = 512;     // the whole tensor memory (one CTA per SM)
// floats in the misc area
constexpr int MISC_MREF = 0, MISC_M = 32, MISC_INVM = 34, MISC_RED = 36, RED_STRIDE = 20, MISC_FLAG = 200, MISC_NEWM = 216;

// ---------------------------------------------------------------------------------------------
// D1: latent-space query image (see TmPlan).  One block per (KV head, precision block, sequence): its channels'
// q~ = sm_scale log2e q B_k^T (a warp per latent channel, B_k row coalesced), its own power-of-two scale, its columns of
// the constant tile and its octets' rows of the k-step tiles.
// ---------------------------------------------------------------------------------------------
constexpr int QP_THREADS = 256, QP_WARPS = 8, QP_U = 8;
struct QpShared {
  float qt[128][4];                   // q~[channel of the block][g]
  float wmax[QP_WARPS];
  float cst[4];
  __align__(16) __half qs[4 * 256];   // the KV head's query rows
};
__device__ __forceinline__ void qproj_tm_body(const StarkvLayout& L, const TmPlan& T, const __half* __restrict__ q,
                                              const __half* __restrict__ B_k, uint8_t* __restrict__ img_all, size_t img_stride,
                                              int hb, int b, QpShared& S) {
  float (&qt)[128][4] = S.qt;
  float (&wmax)[QP_WARPS] = S.wmax;
  float (&cst)[4] = S.cst;
  __half* qs = S.qs;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int h = hb >> 1, blk = hb & 1;
  const int G = L.group, dh = L.head_dim;
  const int nch = blk ? L.k_lo_n[h] : L.k_hi_n[h];
  const int bits = blk ? L.bits_lo : L.bits_hi;
  const int col0 = L.koff[h] + (blk ? L.k_hi_n[h] : 0);
  const bool act = lane * 8 < dh;
  const float qscale = L.sm_scale * kLog2e;
  uint8_t* img = img_all + (size_t)b * img_stride;
  {
    const uint4* src = reinterpret_cast<const uint4*>(q + ((size_t)b * L.n_q_heads + h * G) * dh);
    uint4* dst = reinterpret_cast<uint4*>(qs);
    for (int i = tid; i < G * dh / 8; i += QP_THREADS) dst[i] = src[i];
  }
  __syncthreads();
  float mx = 0.f;
  for (int c0 = 0; c0 < nch; c0 += QP_WARPS * QP_U) {
    uint4 bk[QP_U];
#pragma unroll
    for (int u = 0; u < QP_U; ++u) {
      const int c = c0 + warp + QP_WARPS * u;
      bk[u] = (c < nch && act) ? *reinterpret_cast<const uint4*>(B_k + (size_t)(col0 + c) * dh + lane * 8) : make_uint4(0, 0, 0, 0);
    }
    float a[QP_U][4];
#pragma unroll
    for (int u = 0; u < QP_U; ++u) {
      const float2 b0 = __half22float2(*reinterpret_cast<const __half2*>(&bk[u].x)), b1 = __half22float2(*reinterpret_cast<const __half2*>(&bk[u].y)),
                   b2 = __half22float2(*reinterpret_cast<const __half2*>(&bk[u].z)), b3 = __half22float2(*reinterpret_cast<const __half2*>(&bk[u].w));
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        uint4 y = make_uint4(0, 0, 0, 0);
        if (g < G && act) y = *reinterpret_cast<const uint4*>(qs + g * dh + lane * 8);
        const float2 q0 = __half22float2(*reinterpret_cast<const __half2*>(&y.x)), q1 = __half22float2(*reinterpret_cast<const __half2*>(&y.y)),
                     q2 = __half22float2(*reinterpret_cast<const __half2*>(&y.z)), q3 = __half22float2(*reinterpret_cast<const __half2*>(&y.w));
        float s = q0.x * b0.x;
        s = fmaf(q0.y, b0.y, s); s = fmaf(q1.x, b1.x, s); s = fmaf(q1.y, b1.y, s);
        s = fmaf(q2.x, b2.x, s); s = fmaf(q2.y, b2.y, s); s = fmaf(q3.x, b3.x, s);
        a[u][g] = fmaf(q3.y, b3.y, s);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1)
#pragma unroll
      for (int u = 0; u < QP_U; ++u)
#pragma unroll
        for (int g = 0; g < 4; ++g) a[u][g] += __shfl_xor_sync(0xffffffffu, a[u][g], o);
    if (lane == 0) {
#pragma unroll
      for (int u = 0; u < QP_U; ++u) {
        const int c = c0 + warp + QP_WARPS * u;
        if (c < nch) {
#pragma unroll
          for (int g = 0; g < 4; ++g) {
            const float v = a[u][g] * qscale;
            qt[c][g] = v;
            mx = fmaxf(mx, fabsf(v));
          }
        }
      }
    }
  }
  if (lane == 0) wmax[warp] = mx;
  __syncthreads();
  float m = 0.f;
#pragma unroll
  for (int i = 0; i < QP_WARPS; ++i) m = fmaxf(m, wmax[i]);
  // Q = q~ 2^e with max |Q| of the block in [2^5, 2^6): the hi + lo fp16 pair then keeps >= 2^-27 of the largest entry
  // even for the 1/16-scaled channels, and the constant step (-2^(b-1) 2^-10 sum Q) stays below 2^10
  int e = 0;
  if (m > 0.f && m < INFINITY) {
    e = 6 - (int)(((__float_as_uint(m) >> 23) & 0xff) - 126);
    e = e < -100 ? -100 : (e > 100 ? 100 : e);
  }
  const float scale = ldexpf(1.f, e);
  // ---- constant step: warp g sums the block's channels for group member g
  if (warp < G) {
    float sacc = 0.f;
    for (int c = lane; c < nch; c += 32) {
      const bool s16 = bits == 4 && (c & 1);
      const float av = qt[c][warp] * scale * (s16 ? 0.0625f : 1.f);
      const __half hi = __float2half_rn(av);
      const __half lo = __float2half_rn(av - __half2float(hi));
      sacc += (__half2float(hi) + __half2float(lo)) * (s16 ? 16.f : 1.f);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) sacc += __shfl_xor_sync(0xffffffffu, sacc, o);
    if (lane == 0) cst[warp] = -(float)(1 << (bits - 1)) * 0.0009765625f * sacc;
  }
  __syncthreads();
  // own columns of the constant tile (block 0 of head 0 also clears the columns past the last head)
  {
    const int n_first = hb * G, n_own = G;
    const int n_pad0 = 2 * L.n_kv_heads * G;
    const int n_extra = hb == 0 ? T.ds_cols - n_pad0 : 0;
    for (int w = tid; w < (n_own + n_extra) * 8; w += QP_THREADS) {
      const int ni = w >> 3, kp = w & 7;
      const int n = ni < n_own ? n_first + ni : n_pad0 + (ni - n_own);
      uint32_t word = 0;
      if (kp == 0 && ni < n_own) {
        const float C = cst[ni];
        const __half hi = __float2half_rn(C);
        const __half lo = __float2half_rn(C - __half2float(hi));
        word = (uint32_t)__half_as_ushort(hi) | ((uint32_t)__half_as_ushort(lo) << 16);
      }
      *reinterpret_cast<uint32_t*>(img + (n >> 3) * 256 + (n & 7) * 16 + (kp >> 2) * 128 + (kp & 3) * 4) = word;
    }
  }
  // own octets' rows of the k-step tiles (block 0 of head 0 also clears the padding slots)
  {
    const int o_first = T.blk_oct0[hb], n_own = T.blk_noct[hb];
    const int n_o = n_own + (hb == 0 ? T.n_pad : 0);
    for (int idx = tid; idx < n_o * 128; idx += QP_THREADS) {
      const int oi = idx >> 7, part = (idx >> 6) & 1, w = idx & 63;
      const bool own = oi < n_own;
      const int o = own ? o_first + oi : T.pad_oct[oi - n_own];
      const int ks = o >> 1, hf = o & 1;
      const int n = w >> 2, kp = 4 * hf + (w & 3);
      const int col = T.win[ks] + n;
      uint32_t word = 0;
      if (own && col >= hb * G && col < hb * G + G) {
        const int g = col - hb * G;
#pragma unroll
        for (int eo = 0; eo < 2; ++eo) {
          const int kk = 2 * (w & 3) + eo;
          const bool four = bits == 4;
          const int cin = four ? (kk >> 1) + 4 * (kk & 1) : kk;        // register order of the 4-bit dequantisation
          const bool s16 = four && ((kk >> 1) & 1);
          const float av = qt[8 * oi + cin][g] * scale * (s16 ? 0.0625f : 1.f);
          const __half hi = __float2half_rn(av);
          const __half v = part ? __float2half_rn(av - __half2float(hi)) : hi;
          word |= (uint32_t)__half_as_ushort(v) << (16 * eo);
        }
      }
      *reinterpret_cast<uint32_t*>(img + T.img_ks_off + ks * 1024 + part * 512 + (n >> 3) * 256 + (n & 7) * 16 + (kp >> 2) * 128 +
                                   (kp & 3) * 4) = word;
    }
  }
  if (tid == 0) reinterpret_cast<float*>(img + T.img_scal_off)[hb] = ldexpf(1.f, 24 - e);
}

__global__ void __launch_bounds__(QP_THREADS) qproj_tm_kernel(const __grid_constant__ StarkvLayout L, const __grid_constant__ TmPlan T,
                                                              const __half* __restrict__ q, const __half* __restrict__ B_k,
                                                              uint8_t* __restrict__ img_all, size_t img_stride) {
  __shared__ QpShared S;
  sk_pdl_enter();
  qproj_tm_body(L, T, q, B_k, img_all, img_stride, blockIdx.x, blockIdx.y, S);
}

// First launch of a fused decode step (starkv_decode_step): the query image and the compress-on-append of the step's new
// tokens do not depend on each other, so they share one grid: blocks [0, n_qp) build the image, the rest run the small
// append (append_small.cuh).  Both finish before the decode kernel's griddepcontrol.wait returns.
static_assert(QP_THREADS == APS_THREADS, "the two bodies share a block size");
template <bool FUSED>
__global__ void __launch_bounds__(QP_THREADS) step_pre_tm_kernel(const __grid_constant__ StarkvLayout L, const __grid_constant__ TmPlan T,
                                                                 const __half* __restrict__ q, const __half* __restrict__ B_k,
                                                                 uint8_t* __restrict__ img_all, size_t img_stride, int n_qp,
                                                                 const __grid_constant__ AppendSmallArgs a) {
  __shared__ __align__(16) float sm[APS_SM_FLOATS];
  static_assert(sizeof(QpShared) <= sizeof(float) * APS_SM_FLOATS, "query-image scratch fits the append's shared memory");
  sk_pdl_enter();
  const int i = blockIdx.x;
  if (i < n_qp) {
    const int nhb = 2 * L.n_kv_heads;
    qproj_tm_body(L, T, q, B_k, img_all, img_stride, i % nhb, i / nhb, *reinterpret_cast<QpShared*>(sm));
  } else {
    const int j = i - n_qp;
    append_small_body<FUSED>(L, a, j % a.n_tiles, j / a.n_tiles, sm);
  }
}

// ---------------------------------------------------------------------------------------------
// the decode kernel
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ int f_ordered(float v) {   // monotone map float -> int (its own inverse)
  const int k = __float_as_int(v);
  return k ^ ((k >> 31) & 0x7fffffff);
}
__device__ __forceinline__ float f_unordered(int k) { return __int_as_float(k ^ ((k >> 31) & 0x7fffffff)); }

// position of a consumer / producer in a ring of n stages: stage index and mbarrier phase parity, advanced without divisions
struct RingPos {
  int st, ph, n;
  __device__ __forceinline__ RingPos(int j0, int n_) : st(j0 % n_), ph((j0 / n_) & 1), n(n_) {}
  __device__ __forceinline__ void advance(int k) {   // k <= n
    st += k;
    if (st >= n) { st -= n; ph ^= 1; }
  }
};

// NHH = query heads per softmax warpgroup (the heads are split over NSPLIT warpgroups), G = H_q / H_kv
template <int NHH, int G, int NSPLIT>
__global__ void __launch_bounds__(TM_THREADS, 1) decode_tm_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ TmPlan T, const uint8_t* __restrict__ img_all,
    size_t img_stride, const uint8_t* __restrict__ pool, const int32_t* __restrict__ table, int max_pages,
    const int32_t* __restrict__ seq_lens, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // warp-uniform to the compiler
  const int split = blockIdx.x, b = blockIdx.y;
  sk_pdl_trigger();

  // Three page rings, each with full[] / empty[] mbarriers: a page is fetched as its key blocks, its value blocks and its
  // scales (key scales + value scales), because the three are consumed at different depths of the pipeline -- the key
  // rows a few tiles ahead of the value rows and of the softmax, which reads the scales.  One ring of whole pages
  // would have to hold every page for the whole pipeline depth.
  const int nK = T.n_kstage, nV = T.n_vstage, nS = T.n_sstage;
  const uint32_t fullK0 = smem_u32(smem + T.off_bar);
  const uint32_t emptyK0 = fullK0 + 8 * nK;
  const uint32_t fullV0 = emptyK0 + 8 * nK;
  const uint32_t emptyV0 = fullV0 + 8 * nV;
  const uint32_t fullS0 = emptyV0 + 8 * nV;
  const uint32_t emptyS0 = fullS0 + 8 * nS;
  const uint32_t imgbar = emptyS0 + 8 * nS;
  const uint32_t ak_full0 = imgbar + 8 /* [2]: per half of the k-steps */, qk_done0 = imgbar + 24 /* [2]: per score buffer */,
                 ds_free0 = imgbar + 40 /* [2]: per score buffer */, p_full0 = imgbar + 56 /* [2] */,
                 av_full0 = imgbar + 72 /* [2]: per page */, pv_done0 = imgbar + 88 /* [2]: per P~ buffer */,
                 pv_half = imgbar + 104 /* the value MMAs over the first page's tokens are complete */,
                 qk_half = imgbar + 112 /* the score MMAs over the first half of the k-steps are complete */;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + T.off_bar + 16 * (nK + nV + nS) + 128);
  // the score tile is double-buffered when tensor memory has room (T.ds_nbuf = 2): tile `it` uses buffer it % ds_nbuf, so the
  // score MMAs of the next tile run while the softmax warps still read this one
  const int ds_nbuf = T.ds_nbuf;
  int32_t* tbl_s = reinterpret_cast<int32_t*>(smem + T.off_tbl);
  float* misc = reinterpret_cast<float*>(smem + T.off_misc);
  uint8_t* kstage_base = smem + T.off_kstage;
  uint8_t* vstage_base = smem + T.off_vstage;
  uint8_t* sstage_base = smem + T.off_sstage;
  const uint32_t page_bytes = (uint32_t)L.page_bytes;

  if (tid == 0) {
    for (int s = 0; s < nK; ++s) { mbar_init(fullK0 + 8 * s, 1); mbar_init(emptyK0 + 8 * s, 4); }            // 2 + 2 key warps read a page
    for (int s = 0; s < nV; ++s) { mbar_init(fullV0 + 8 * s, 1); mbar_init(emptyV0 + 8 * s, 4); }            // 4 value warps
    for (int s = 0; s < nS; ++s) { mbar_init(fullS0 + 8 * s, 1); mbar_init(emptyS0 + 8 * s, 2 * NSPLIT); }   // softmax warps of the page
    mbar_init(imgbar, 1);
    mbar_init(ak_full0, 4);
    mbar_init(ak_full0 + 8, 4);
    mbar_init(qk_half, 1);
    mbar_init(qk_done0, 1);
    mbar_init(qk_done0 + 8, 1);
    mbar_init(ds_free0, 4 * NSPLIT);
    mbar_init(ds_free0 + 8, 4 * NSPLIT);
    mbar_init(p_full0, 4 * NSPLIT);
    mbar_init(p_full0 + 8, 4 * NSPLIT);
    mbar_init(av_full0, 4);
    mbar_init(av_full0 + 8, 4);
    mbar_init(pv_done0, 1);
    mbar_init(pv_done0 + 8, 1);
    mbar_init(pv_half, 1);
    fence_barrier_init();
  }
  if (warp == 23) tmem_alloc(smem_u32((const void*)tmem_slot), TM_COLS);
  if (tid < 36) misc[tid] = tid < 32 ? -P_OFFSET : (tid < 34 ? 0.f : A_SHIFT);   // reference m - P_OFFSET with m = 0, M = 0, a-factor A_SHIFT / 1 (all replaced by the first tile)

  sk_pdl_wait();   // seq_lens, block table, query image, pages: nothing global is read before this point
  const int len = seq_lens[b];
  int n_pages = len > 0 ? (len + PTOK - 1) / PTOK : 0;
  if (n_pages > max_pages) n_pages = max_pages;
  int p0, p1;
  sk_split_range(n_pages, n_splits, 2, split, &p0, &p1);
  const int n_pg = p1 - p0;                 // pages of this CTA
  const int n_it = (n_pg + 1) >> 1;         // 128-token iterations
  const size_t pstride = sk_part_stride(L.rank_v);
  float* my_parts = parts + ((size_t)b * n_splits + split) * L.n_q_heads * pstride;
  const int32_t* my_table = table + (size_t)b * max_pages + p0;
  for (int i = tid; i < min(n_pg, TM_TBL); i += TM_THREADS) tbl_s[i] = my_table[i];

  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tbase = *tmem_slot;

  if (n_pg <= 0) {   // empty range (CTA-uniform): neutral partial
    for (int i = tid; i < L.n_q_heads * (int)pstride; i += TM_THREADS) my_parts[i] = (i % (int)pstride) == 0 ? -INFINITY : 0.f;
  } else if (warp < 8) {
    // =============================== key rows -> A operand of the score product ===============================
    // warps 0-3 convert the first half of the k-steps, warps 4-7 the second half (each warp its own 32 tokens = lanes)
    setmaxnreg_dec<64>();
    const int wq = warp & 3, half = warp >> 2, tq = wq * 32 + lane, pgsel = tq >> 6, slot = tq & 63;
    const uint32_t tl = tbase + ((uint32_t)(wq * 32) << 16) + (uint32_t)T.col_ak;
    if (half == 0) {
      const uint32_t c[8] = {0x04000400u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};   // constant step: (2^-14, 2^-14, 0, ...)
      tmem_st8(tl, c);
    }
    const int n8 = T.n_trips8, nt = T.n_trips8 + T.n_trips4, nt0 = (nt + 1) >> 1;
    const int k_begin = half ? nt0 : 0, k_end = half ? nt : nt0;
    const uint4* desc4 = reinterpret_cast<const uint4*>(T.oct_desc);
    RingPos rk(pgsel, nK);
    const int dsh = ds_nbuf - 1;   // tile it uses score buffer it & dsh, for the (it >> dsh)-th time
    for (int it = 0; it < n_it; ++it, rk.advance(2)) {
      const int j = 2 * it + pgsel;
      const bool exists = j < n_pg;
      const int st = rk.st;
      uint4 dq = desc4[k_begin];
      if (exists) mbar_wait(fullK0 + 8 * st, (uint32_t)rk.ph);
      const uint8_t* row = kstage_base + (size_t)st * T.kstride;
      if (it > 0) {   // the previous tile's score MMAs over this half have read the operand
        if (half) mbar_wait(qk_done0 + 8 * ((it - 1) & dsh), (uint32_t)(((it - 1) >> dsh) & 1));
        else mbar_wait(qk_half, (uint32_t)((it - 1) & 1));
        tc_fence_after();
      }
      // Four octets (two k-steps) per trip: packed plan entries (page offset | row bytes << 18; the next trip's entry is
      // fetched a trip ahead), loads, conversions, one 16-column store.
#pragma unroll 2
      for (int k2 = k_begin; k2 < k_end; ++k2) {
        const uint32_t dsc[4] = {dq.x, dq.y, dq.z, dq.w};
        dq = desc4[k2 + 1 < SK_TM_MAX_TRIPS ? k2 + 1 : k2];
        const uint8_t* p[4];
#pragma unroll
        for (int oo = 0; oo < 4; ++oo) p[oo] = row + (dsc[oo] & 0x3ffffu) + slot * (dsc[oo] >> 18);
        uint32_t r[16];
        if (k2 < n8) {   // 8-bit fields: (u0, u1), (u2, u3), ... as fp16 subnormals u 2^-24
          uint2 x[4];
#pragma unroll
          for (int oo = 0; oo < 4; ++oo) x[oo] = *reinterpret_cast<const uint2*>(p[oo]);
#pragma unroll
          for (int oo = 0; oo < 4; ++oo) {
            r[4 * oo] = prmt(x[oo].x, 0u, 0x4140u);
            r[4 * oo + 1] = prmt(x[oo].x, 0u, 0x4342u);
            r[4 * oo + 2] = prmt(x[oo].y, 0u, 0x4140u);
            r[4 * oo + 3] = prmt(x[oo].y, 0u, 0x4342u);
          }
        } else {         // 4-bit fields: (u0, u4), 16 (u1, u5), (u2, u6), 16 (u3, u7); the 16 is taken out of the query image
          uint32_t w[4];
#pragma unroll
          for (int oo = 0; oo < 4; ++oo) w[oo] = *reinterpret_cast<const uint32_t*>(p[oo]);
#pragma unroll
          for (int oo = 0; oo < 4; ++oo) {
            const uint32_t w2 = w[oo] >> 8;
            r[4 * oo] = w[oo] & 0x000f000fu;
            r[4 * oo + 1] = w[oo] & 0x00f000f0u;
            r[4 * oo + 2] = w2 & 0x000f000fu;
            r[4 * oo + 3] = w2 & 0x00f000f0u;
          }
        }
        tmem_st16(tl + 8 + 16 * k2, r);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(ak_full0 + 8 * half);
        if (exists) mbar_arrive(emptyK0 + 8 * st);
      }
    }
  } else if (warp < 16) {
    // ========================================= softmax (thread = token) =========================================
    setmaxnreg_inc<112>();
    const int hh = (warp - 8) >> 2;   // which half of the query heads
    if (hh < NSPLIT) {
      const int wq = warp & 3, wr = warp - 8, tq = wq * 32 + lane, pgsel = tq >> 6, slot = tq & 63;
      const int hbase = hh * NHH;     // first query head of this warpgroup
      const uint32_t tlane = tbase + ((uint32_t)(wq * 32) << 16);
      float* mref_s = misc + MISC_MREF;   // running reference of every head, stored as m - 8: 2^(s - (m - 8)) = p'
      float* M_s = misc + MISC_M;
      float* invM_s = misc + MISC_INVM;
      int* red = reinterpret_cast<int*>(misc + MISC_RED);                                // [8 warps][RED_STRIDE], ordered ints
      volatile uint8_t* flag = reinterpret_cast<volatile uint8_t*>(misc + MISC_FLAG);   // [2][8 bytes]: one per warp
      float* mnew_s = misc + MISC_NEWM;
      const int Hq = L.n_q_heads, n_kv = L.n_kv_heads;
      constexpr int NBAR = 128 * NSPLIT;
      // position of this token along K of the value product, per precision block (4-bit rows are dequantised in the
      // order 0,4,1,5,2,6,3,7 inside every 8 slots)
      uint32_t paddr[2];
#pragma unroll
      for (int blk = 0; blk < 2; ++blk) {
        const int bits = blk ? L.bits_lo : L.bits_hi;
        const int i8 = slot & 7;
        const int kp = 64 * pgsel + (bits == 4 ? (slot & ~7) + (i8 < 4 ? 2 * i8 : 2 * (i8 - 4) + 1) : slot);
        paddr[blk] = (uint32_t)(blk * P_BLK_BYTES + (kp >> 3) * 128 + (kp & 7) * 16 + hh * (NHH / 8) * 2048);
      }
      float l_acc[NHH];
#pragma unroll
      for (int i = 0; i < NHH; ++i) l_acc[i] = 0.f;
      if (tq < 4 && hh == 0) reinterpret_cast<volatile uint32_t*>(misc + MISC_FLAG)[tq] = 0u;   // (unused warps' bytes stay 0)
      mbar_wait(imgbar, 0);
      const float* ce_s = reinterpret_cast<const float*>(smem + T.off_img + T.img_scal_off);   // 2^(24 - e) per (head, block)
      bar_sync(BAR_SM, NBAR);

      uint32_t d[2 * NHH];
      RingPos rs(pgsel, nS);
      const int dsh = ds_nbuf - 1;
      for (int it = 0; it < n_it; ++it, rs.advance(2)) {
        const int j = 2 * it + pgsel;
        const bool exists = j < n_pg;
        const int st = rs.st;
        const int buf = it & 1;
        const int sb = it & dsh;
        if (!(ds_nbuf == 2 && it > 0)) {   // (double-buffered score tiles: loaded ahead, at the end of the previous tile's arithmetic)
          mbar_wait(qk_done0 + 8 * sb, (uint32_t)((it >> dsh) & 1));
          tc_fence_after();
          tmem_ld<2 * NHH>(tlane + (uint32_t)(T.col_ds + sb * T.ds_cols + 2 * hbase), d);
        }
        if (exists) mbar_wait(fullS0 + 8 * st, (uint32_t)rs.ph);
        const uint8_t* sslot = sstage_base + (size_t)st * T.sstride;   // [key scales][value scales] of the page
        const uint16_t* ksc = reinterpret_cast<const uint16_t*>(sslot) + slot;
        const uint16_t* vsc = reinterpret_cast<const uint16_t*>(sslot + T.ks_bytes) + slot;
        const bool valid = exists && ((p0 + j) * PTOK + slot) < len;
        // unconditional loads (slots past the sequence end and heads past the last hold finite or junk bits that the
        // selects below discard): no divergent regions, one base address
        float sc[2 * (NHH / G)];
#pragma unroll
        for (int hl = 0; hl < NHH / G; ++hl) {
          const int kvh = min(hbase / G + hl, n_kv - 1);
          sc[2 * hl] = h_bits_to_f(ksc[(2 * kvh) * PTOK]) * ce_s[2 * kvh];
          sc[2 * hl + 1] = h_bits_to_f(ksc[(2 * kvh + 1) * PTOK]) * ce_s[2 * kvh + 1];
        }
        const float sv0 = valid ? h_bits_to_f(vsc[0]) : 0.f;
        const float sv1 = valid ? h_bits_to_f(vsc[PTOK]) : 0.f;
        tmem_wait_ld();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) mbar_arrive(ds_free0 + 8 * sb);
        float arg[NHH];
#pragma unroll
        for (int hl = 0; hl < NHH / G; ++hl)
#pragma unroll
          for (int g = 0; g < G; ++g)
            arg[hl * G + g] = fmaf(sc[2 * hl], __uint_as_float(d[2 * hl * G + g]), sc[2 * hl + 1] * __uint_as_float(d[2 * hl * G + G + g]));
        // (the references are subtracted after the scores are complete, not inside the multiply-adds: all sixteen of them
        // live next to the 32 score registers spill the softmax warps' 112 registers -- measured, C3 27.1 -> 31.8 us)
        if (it == 0) {
          // The references start from the range's first 32 tokens (warp 0 of each half; the first token is always inside
          // the sequence): per head the largest of their scores, and 2^8 times their largest value scales.  A later token
          // that exceeds them by the lazy bounds takes the update path below.  That path costs about 2.8 us per CTA
          // (three barriers, reductions, a rescale of the TMEM accumulators, all instruction-cache cold), so it has to be
          // rare: with the FIRST token's score as the reference it ran in most CTAs of the diffuse regime (any of the
          // range's tokens 2^6 above one arbitrary token triggers it), with the maximum of 32 it does not.
          if (wq == 0) {
#pragma unroll
            for (int i = 0; i < NHH; ++i) {
              const int k = __reduce_max_sync(0xffffffffu, f_ordered(valid ? arg[i] : -INFINITY));
              if (lane == 0) mref_s[hbase + i] = f_unordered(k) - P_OFFSET;
            }
            if (hh == 0) {
#pragma unroll
              for (int blk = 0; blk < 2; ++blk) {
                // (non-negative floats order as their bits)
                const float sv = __uint_as_float(__reduce_max_sync(0xffffffffu, __float_as_uint(blk ? sv1 : sv0)));
                unsigned eb = ((__float_as_uint(sv) >> 23) & 0xffu) + 8u;   // 2^8 of headroom
                if (eb > 254u) eb = 254u;
                const float M = sv > 0.f ? __uint_as_float(eb << 23) : 1.f;
                if (lane == 0) {
                  M_s[blk] = M;
                  invM_s[blk] = A_SHIFT / M;
                }
              }
            }
          }
          bar_sync(BAR_SM, NBAR);
        }
        const float M0 = M_s[0], M1 = M_s[1];
#pragma unroll
        for (int i = 0; i < NHH; ++i) arg[i] -= mref_s[hbase + i];
        // slots past the sequence end only exist in the last tile of a sequence's last split: mask there, not everywhere
        if ((p0 + 2 * it + 2) * PTOK > len) {
#pragma unroll
          for (int i = 0; i < NHH; ++i) arg[i] = valid ? arg[i] : -INFINITY;
        }
        float mxa = -INFINITY;
        if (hbase + NHH <= Hq) {   // (CTA-uniform) every head of this warpgroup exists
#pragma unroll
          for (int i = 0; i < NHH; ++i) mxa = fmaxf(mxa, arg[i]);
        } else {
#pragma unroll
          for (int i = 0; i < NHH; ++i)
            if (hbase + i < Hq) mxa = fmaxf(mxa, arg[i]);
        }
        if (ds_nbuf == 2 && it + 1 < n_it) {
          // the next tile's scores: its MMAs ran while this tile was being read, so the TMEM load's latency hides behind the
          // rest of this tile's work
          const int sn = (it + 1) & 1;
          mbar_wait(qk_done0 + 8 * sn, (uint32_t)(((it + 1) >> 1) & 1));
          tc_fence_after();
          tmem_ld<2 * NHH>(tlane + (uint32_t)(T.col_ds + sn * T.ds_cols + 2 * hbase), d);
        }
        // The fp16 operand is P~ = p' a with p' = 2^(s - m + 4) and a = 16 s_v / M, both fp16.  The references only have to
        // move when p' or the product nears the fp16 limit: the running maximum may lag the true one by 2^11.5 (2^6 with
        // the split 2^8 and 1 of the same product), which keeps the (costly) update path out of the way of heavy-tailed
        // scores.
        float a0 = sv0 * invM_s[0], a1 = sv1 * invM_s[1];
        const float pmax = ex2(mxa);
        const bool trig = valid && (pmax > P_CAP || pmax * fmaxf(a0, a1) > P_CAP || sv0 > M0 || sv1 > M1);
        const bool wany = __any_sync(0xffffffffu, trig);
        if (lane == 0) {
          flag[buf * 8 + wr] = wany ? 1 : 0;
          if (exists) mbar_arrive(emptyS0 + 8 * st);   // every scale of the page has been used: the slot may be refilled
        }
        bar_sync(BAR_SM, NBAR);
        const volatile uint32_t* flw = reinterpret_cast<const volatile uint32_t*>(flag + buf * 8);
        const bool upd = (flw[0] | flw[1]) != 0u;
        if (upd) {
          // ---- a maximum (or a value-scale bound) moves: new reference, rescale the running sums and the accumulators
#pragma unroll
          for (int i = 0; i < NHH; ++i) {
            const float v = valid ? arg[i] + mref_s[hbase + i] : -INFINITY;   // the score itself
            const int k = __reduce_max_sync(0xffffffffu, f_ordered(v));
            if (lane == 0) red[wr * RED_STRIDE + i] = k;
          }
          {
            const unsigned a0 = __reduce_max_sync(0xffffffffu, __float_as_uint(sv0));   // non-negative floats order as their bits
            const unsigned a1 = __reduce_max_sync(0xffffffffu, __float_as_uint(sv1));
            if (lane == 0) { red[wr * RED_STRIDE + 16] = (int)a0; red[wr * RED_STRIDE + 17] = (int)a1; }
          }
          bar_sync(BAR_SM, NBAR);
          const int* redh = red + 4 * hh * RED_STRIDE;   // the four warps of this half cover the tile's 128 tokens
          float fs[NHH];
#pragma unroll
          for (int i = 0; i < NHH; ++i) {
            const float mt = f_unordered(max(max(redh[i], redh[RED_STRIDE + i]), max(redh[2 * RED_STRIDE + i], redh[3 * RED_STRIDE + i])));
            const float m_old = mref_s[hbase + i];    // (references are stored as m - 8)
            // only a maximum that the tile exceeds moves (to the true maximum so far); the first tile sets it
            float m_new = fmaxf(mt - P_OFFSET, m_old);
            if (!(m_new > -INFINITY)) m_new = m_old;
            const float delta = m_old - m_new;       // <= 0 after the first tile
            fs[i] = ex2(delta);
            arg[i] += delta;
            l_acc[i] *= fs[i];
            mnew_s[hbase + i] = m_new;               // (every thread of the half computes and stores the same value)
          }
          float fM[2], Mn[2];
#pragma unroll
          for (int blk = 0; blk < 2; ++blk) {
            const float sm = __uint_as_float((unsigned)max(max(redh[16 + blk], redh[RED_STRIDE + 16 + blk]),
                                                           max(redh[2 * RED_STRIDE + 16 + blk], redh[3 * RED_STRIDE + 16 + blk])));
            const float M_old = M_s[blk];
            float M_new = M_old;
            if (sm > M_old) {   // a power of two 8-16 times above the largest scale seen: later tiles rarely exceed it
              unsigned eb = ((__float_as_uint(sm) >> 23) & 0xffu) + 4u;
              if (eb > 254u) eb = 254u;
              M_new = __uint_as_float(eb << 23);
            }
            if (M_new == 0.f) M_new = 1.f;
            Mn[blk] = M_new;
            fM[blk] = (M_old > 0.f) ? M_old / M_new : 1.f;
          }
          if (it > 0) {   // every value MMA issued so far is complete before the accumulators are touched
            mbar_wait(pv_done0 + 8 * ((it - 1) & 1), (uint32_t)(((it - 1) >> 1) & 1));
            tc_fence_after();
            for (int dt = 0; dt < T.n_dt; ++dt) {
              const float fb = fM[T.dt_blk[dt] ? 1 : 0];
              uint32_t v[NHH];
              tmem_ld<NHH>(tlane + (uint32_t)(T.col_do + 32 * dt + hbase), v);
              tmem_wait_ld();
#pragma unroll
              for (int i = 0; i < NHH; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * (fs[i] * fb));
              tmem_st<NHH>(tlane + (uint32_t)(T.col_do + 32 * dt + hbase), v);
            }
            tmem_wait_st();
            tc_fence_before();
          }
          bar_sync(BAR_SM, NBAR);   // every thread has read the old references
          if (tq < NHH) mref_s[hbase + tq] = mnew_s[hbase + tq];
          if (hh == 0 && tq == 0) {
            M_s[0] = Mn[0]; M_s[1] = Mn[1];
            invM_s[0] = A_SHIFT / Mn[0]; invM_s[1] = A_SHIFT / Mn[1];
          }
          bar_sync(BAR_SM, NBAR);
          a0 = sv0 * invM_s[0]; a1 = sv1 * invM_s[1];
        }
        // ---- p' and the two scaled operands
        const uint32_t a0h = pack_h2(a0, a0), a1h = pack_h2(a1, a1);
        if (it >= 2) mbar_wait(pv_done0 + 8 * buf, (uint32_t)(((it >> 1) - 1) & 1));   // the MMAs of tile it - 2 have read the buffer
        uint8_t* pb = smem + T.off_p + buf * 2 * P_BLK_BYTES;
#pragma unroll
        for (int oc = 0; oc < NHH / 8; ++oc) {
          float p[8];
#pragma unroll
          for (int k = 0; k < 8; ++k) {
            p[k] = ex2(arg[8 * oc + k]);   // -inf -> 0 for slots past the sequence end
            l_acc[8 * oc + k] += p[k];
          }
          // p' -> fp16 pairs once, then the two value-scale factors as packed fp16 multiplies (two roundings of 2^-11 on
          // a term of the value product; no flush to zero)
          const uint32_t q0 = pack_h2(p[0], p[1]), q1 = pack_h2(p[2], p[3]), q2 = pack_h2(p[4], p[5]), q3 = pack_h2(p[6], p[7]);
          uint4 x0, x1;
          x0.x = h2mul(q0, a0h); x0.y = h2mul(q1, a0h); x0.z = h2mul(q2, a0h); x0.w = h2mul(q3, a0h);
          x1.x = h2mul(q0, a1h); x1.y = h2mul(q1, a1h); x1.z = h2mul(q2, a1h); x1.w = h2mul(q3, a1h);
          *reinterpret_cast<uint4*>(pb + paddr[0] + oc * 2048) = x0;
          *reinterpret_cast<uint4*>(pb + paddr[1] + oc * 2048) = x1;
        }
        fence_proxy_async();   // generic-proxy stores -> visible to the tensor core's reads
        __syncwarp();
        if (lane == 0) mbar_arrive(p_full0 + 8 * buf);
      }
      // ---- split-K partial (D7): [m, l, 0, 0, acc[r_v]] per head
      {
        const int last = n_it - 1;
        mbar_wait(pv_done0 + 8 * (last & 1), (uint32_t)((last >> 1) & 1));
        tc_fence_after();
        for (int dt = 0; dt < T.n_dt; ++dt) {
          const int blk = T.dt_blk[dt] ? 1 : 0;
          const int ch = 128 * T.dt_tile[dt] + tq;
          uint32_t v[NHH];
          tmem_ld<NHH>(tlane + (uint32_t)(T.col_do + 32 * dt + hbase), v);
          tmem_wait_ld();
          const bool mine = ch < L.rank_v && ((ch >= L.v_hi_n) == (blk == 1));
          const float Mb = M_s[blk] * (1.f / A_SHIFT);   // O = sum c p' a = (16 / M) sum c p' s_v: back to the scale of l = sum p'
          if (mine) {
#pragma unroll
            for (int i = 0; i < NHH; ++i)
              if (hbase + i < Hq) my_parts[(size_t)(hbase + i) * pstride + SK_PART_ACC + ch] = __uint_as_float(v[i]) * Mb;
          }
        }
        float* redf = misc + MISC_RED;
#pragma unroll
        for (int i = 0; i < NHH; ++i) {
          float v = l_acc[i];
#pragma unroll
          for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
          if (lane == 0) redf[wr * RED_STRIDE + i] = v;
        }
        bar_sync(BAR_SM, NBAR);
        if (tq < NHH && hbase + tq < Hq) {
          const float* rh = redf + 4 * hh * RED_STRIDE;
          const float lsum = rh[tq] + rh[RED_STRIDE + tq] + rh[2 * RED_STRIDE + tq] + rh[3 * RED_STRIDE + tq];
          *reinterpret_cast<float4*>(my_parts + (size_t)(hbase + tq) * pstride) = make_float4(mref_s[hbase + tq] + P_OFFSET, lsum, 0.f, 0.f);
        }
      }
    }
  } else if (warp < 20) {
    // =============================== value rows -> A operand of the value product ===============================
    setmaxnreg_inc<88>();
    const int wq = warp - 16, tq = wq * 32 + lane;
    const uint32_t tl = tbase + ((uint32_t)(wq * 32) << 16) + (uint32_t)T.col_av;
    int roff[2];
    bool four[2], act[2];
#pragma unroll
    for (int m = 0; m < 2; ++m) {
      const int ch = 128 * m + tq;
      act[m] = m < T.n_vt && ch < L.rank_v;
      const bool lo = ch >= L.v_hi_n;
      const int bits = lo ? L.bits_lo : L.bits_hi;
      const int rowb = PTOK * bits / 8;
      four[m] = bits == 4;
      roff[m] = act[m] ? (lo ? L.v_lo_off + (ch - L.v_hi_n) * rowb : L.v_hi_off + ch * rowb) : 0;
    }
    RingPos rv(0, nV);
    for (int it = 0; it < n_it; ++it) {
#pragma unroll 1
      for (int pg = 0; pg < 2; ++pg, rv.advance(1)) {
        const int j = 2 * it + pg;
        const bool exists = j < n_pg;
        const int st = rv.st;
        if (exists) mbar_wait(fullV0 + 8 * st, (uint32_t)rv.ph);
        if (it > 0) {   // the previous tile's value MMAs over this half of the tokens have read the operand
          if (pg == 0) mbar_wait(pv_half, (uint32_t)((it - 1) & 1));
          else mbar_wait(pv_done0 + 8 * ((it - 1) & 1), (uint32_t)(((it - 1) >> 1) & 1));
          tc_fence_after();
        }
        const uint8_t* pagep = vstage_base + (size_t)st * T.vstride - L.v_hi_off;   // (row offsets are page-relative)
#pragma unroll
        for (int m = 0; m < 2; ++m) {
          if (m < T.n_vt) {
            const uint8_t* rowp = pagep + roff[m];
            uint32_t r[32];
            if (!act[m]) {
#pragma unroll
              for (int k = 0; k < 32; ++k) r[k] = 0u;
            } else if (four[m]) {
              const uint4 x0 = *reinterpret_cast<const uint4*>(rowp);
              const uint4 x1 = *reinterpret_cast<const uint4*>(rowp + 16);
              deq4_pairs(x0.x, r); deq4_pairs(x0.y, r + 4); deq4_pairs(x0.z, r + 8); deq4_pairs(x0.w, r + 12);
              deq4_pairs(x1.x, r + 16); deq4_pairs(x1.y, r + 20); deq4_pairs(x1.z, r + 24); deq4_pairs(x1.w, r + 28);
            } else {
#pragma unroll
              for (int c4 = 0; c4 < 4; ++c4) {
                const uint4 x = *reinterpret_cast<const uint4*>(rowp + 16 * c4);
                deq8_pairs(x.x, r[8 * c4], r[8 * c4 + 1]);
                deq8_pairs(x.y, r[8 * c4 + 2], r[8 * c4 + 3]);
                deq8_pairs(x.z, r[8 * c4 + 4], r[8 * c4 + 5]);
                deq8_pairs(x.w, r[8 * c4 + 6], r[8 * c4 + 7]);
              }
            }
            tmem_st32(tl + 64 * m + 32 * pg, r);
          }
        }
        tmem_wait_st();
        tc_fence_before();
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(av_full0 + 8 * pg);
          if (exists) mbar_arrive(emptyV0 + 8 * st);
        }
      }
    }
  } else {
    setmaxnreg_dec<40>();
    if (warp == 20) {
      // ================================== page producer (D2): key blocks ==================================
      if (elect_one()) {
        const uint64_t pol = l2_evict_first_policy();
        mbar_expect_tx(imgbar, (uint32_t)T.img_bytes);
        bulk_g2s(smem_u32(smem + T.off_img), img_all + (size_t)b * img_stride, (uint32_t)T.img_bytes, imgbar);
        RingPos rp(0, nK);
        for (int j = 0; j < n_pg; ++j, rp.advance(1)) {
          const int st = rp.st;
          if (j >= nK) mbar_wait(emptyK0 + 8 * st, (uint32_t)(rp.ph ^ 1));
          const int page = max(j < TM_TBL ? tbl_s[j] : my_table[j], 0);   // (a negative entry is a caller error: memory-safe)
          mbar_expect_tx(fullK0 + 8 * st, (uint32_t)T.k_bytes);
          bulk_g2s_stream(smem_u32(kstage_base + (size_t)st * T.kstride), pool + (size_t)page * page_bytes, (uint32_t)T.k_bytes,
                          fullK0 + 8 * st, pol);
        }
      }
      __syncwarp();
    } else if (warp == 23) {
      // ================================== page producer (D2): scales and value blocks ==================================
      if (elect_one()) {
        const uint64_t pol = l2_evict_first_policy();
        RingPos rs(0, nS), rv(0, nV);
        for (int j = 0; j < n_pg; ++j, rs.advance(1), rv.advance(1)) {
          const int page = max(j < TM_TBL ? tbl_s[j] : my_table[j], 0);   // (a negative entry is a caller error: memory-safe)
          const uint8_t* src = pool + (size_t)page * page_bytes;
          {
            const int st = rs.st;
            if (j >= nS) mbar_wait(emptyS0 + 8 * st, (uint32_t)(rs.ph ^ 1));
            const uint32_t dst = smem_u32(sstage_base + (size_t)st * T.sstride);
            mbar_expect_tx(fullS0 + 8 * st, (uint32_t)(T.ks_bytes + T.vs_bytes));
            bulk_g2s_stream(dst, src + L.k_scale_off, (uint32_t)T.ks_bytes, fullS0 + 8 * st, pol);
            bulk_g2s_stream(dst + (uint32_t)T.ks_bytes, src + L.v_scale_off, (uint32_t)T.vs_bytes, fullS0 + 8 * st, pol);
          }
          {
            const int st = rv.st;
            if (j >= nV) mbar_wait(emptyV0 + 8 * st, (uint32_t)(rv.ph ^ 1));
            mbar_expect_tx(fullV0 + 8 * st, (uint32_t)T.v_bytes);
            bulk_g2s_stream(smem_u32(vstage_base + (size_t)st * T.vstride), src + L.v_hi_off, (uint32_t)T.v_bytes, fullV0 + 8 * st, pol);
          }
        }
      }
      __syncwarp();
    } else if (warp == 21) {
      // ================================== score MMAs ==================================
      mbar_wait(imgbar, 0);
      const uint32_t img_s = smem_u32(smem + T.off_img);
      const uint64_t dconst = umma_desc(img_s, 128, 256);
      const uint64_t dks = umma_desc(img_s + (uint32_t)T.img_ks_off, 128, 256);
      const uint32_t id_const = umma_idesc_f16(T.ds_cols, false), id_win = umma_idesc_f16(16, false);
      const uint32_t t_ds = tbase + (uint32_t)T.col_ds, t_ak = tbase + (uint32_t)T.col_ak;
      const int n_ks = T.n_ks, ks_half = 2 * ((T.n_trips8 + T.n_trips4 + 1) >> 1);
      for (int it = 0; it < n_it; ++it) {
#pragma unroll 1
        for (int half = 0; half < 2; ++half) {
          const int sb = it & (ds_nbuf - 1);
          const uint32_t t_dsb = t_ds + (uint32_t)(sb * T.ds_cols);
          mbar_wait(ak_full0 + 8 * half, (uint32_t)(it & 1));
          if (half == 0 && it >= ds_nbuf) mbar_wait(ds_free0 + 8 * sb, (uint32_t)(((it >> (ds_nbuf - 1)) - 1) & 1));   // tile it - ds_nbuf has been read
          tc_fence_after();
          if (elect_one()) {
            if (half == 0) umma_ts_f16(t_dsb, t_ak, dconst, id_const, 0u);
            const int ks_end = half ? n_ks : ks_half;
#pragma unroll 2
            for (int ks = half ? ks_half : 0; ks < ks_end; ++ks) {
              const uint32_t dcol = t_dsb + (uint32_t)T.win[ks];
              umma_ts_f16(dcol, t_ak + 8 + 8 * ks, dks + (uint64_t)(ks * 64), id_win, 1u);
              umma_ts_f16(dcol, t_ak + 8 + 8 * ks, dks + (uint64_t)(ks * 64 + 32), id_win, 1u);
            }
            umma_commit(half ? qk_done0 + 8 * sb : qk_half);
          }
          __syncwarp();
        }
      }
    } else if (warp == 22) {
      // ================================== value MMAs ==================================
      const uint32_t id_pv = umma_idesc_f16(32, true);
      const uint32_t t_do = tbase + (uint32_t)T.col_do, t_av = tbase + (uint32_t)T.col_av;
      const uint32_t p_s = smem_u32(smem + T.off_p);
      const int n_dt = T.n_dt;
      uint32_t ta[4], pofs[4];
#pragma unroll
      for (int dt = 0; dt < 4; ++dt) {
        ta[dt] = t_av + (uint32_t)(64 * T.dt_tile[dt]);
        pofs[dt] = T.dt_blk[dt] ? (uint32_t)P_BLK_BYTES : 0u;
      }
      for (int it = 0; it < n_it; ++it) {
        const int buf = it & 1;
        mbar_wait(p_full0 + 8 * buf, (uint32_t)((it >> 1) & 1));
        const uint32_t pbuf = p_s + (uint32_t)(buf * 2 * P_BLK_BYTES);
#pragma unroll
        for (int pg = 0; pg < 2; ++pg) {
          mbar_wait(av_full0 + 8 * pg, (uint32_t)(it & 1));
          tc_fence_after();
          if (elect_one()) {
#pragma unroll
            for (int dt = 0; dt < 4; ++dt) {
              if (dt < n_dt) {
                const uint64_t dp = umma_desc(pbuf + pofs[dt], 128, 2048);
#pragma unroll
                for (int k4 = 0; k4 < 4; ++k4) {
                  const int ks = 4 * pg + k4;
                  umma_ts_f16(t_do + 32 * dt, ta[dt] + 8 * ks, dp + (uint64_t)(ks * 16), id_pv, (it > 0 || ks > 0) ? 1u : 0u);
                }
              }
            }
            umma_commit(pg == 0 ? pv_half : pv_done0 + 8 * buf);
          }
          __syncwarp();
        }
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 23) tmem_dealloc(tbase, TM_COLS);
}

typedef void (*TmKernel)(const StarkvLayout, const TmPlan, const uint8_t*, size_t, const uint8_t*, const int32_t*, int,
                         const int32_t*, float*, int);

TmKernel tm_kernel_for(int n_q_heads, int G) {
  const bool small = n_q_heads <= 8;   // 8 heads on one softmax warpgroup; up to 32 as two halves of 16
  switch (G) {
    case 1: return small ? decode_tm_kernel<8, 1, 1> : decode_tm_kernel<16, 1, 2>;
    case 2: return small ? decode_tm_kernel<8, 2, 1> : decode_tm_kernel<16, 2, 2>;
    case 4: return small ? decode_tm_kernel<8, 4, 1> : decode_tm_kernel<16, 4, 2>;
  }
  return nullptr;
}

int round_up(int x, int m) { return (x + m - 1) / m * m; }

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: plan, launch
// ---------------------------------------------------------------------------------------------
int sk_tm_plan(starkv_ctx* ctx) {
  const StarkvLayout& L = ctx->L;
  TmPlan& T = ctx->tm;
  memset(&T, 0, sizeof(T));
  const int G = L.group;
  if (L.bits_hi == 16 || L.page_tokens != PTOK || L.n_q_heads > 32 || !(G == 1 || G == 2 || G == 4)) return 0;
  if (L.rank_v > 256 || L.n_kv_heads > 32) return 0;
  // octet slots: the 8-bit octets in cache order, padded to a multiple of four, then the 4-bit octets likewise
  int slot_hb[SK_TM_MAX_OCT];
  for (int o = 0; o < SK_TM_MAX_OCT; ++o) slot_hb[o] = -1;
  int no = 0;
  for (int pass = 0; pass < 2; ++pass) {
    const int want_bits = pass == 0 ? 8 : 4;
    for (int h = 0; h < L.n_kv_heads; ++h)
      for (int blk = 0; blk < 2; ++blk) {
        const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
        const int bits = blk ? L.bits_lo : L.bits_hi;
        if (bits != want_bits) continue;
        if (n > 128) return 0;
        const int rowb = n * bits / 8;
        const int hb = 2 * h + blk;
        // an octet must share its k-step's 16-column window with its partner: if the previous (even) slot's columns are
        // too far away (a head with an empty block lies between), leave the odd slot empty
        if (n > 0 && (no & 1) && slot_hb[no - 1] >= 0) {
          const int ca = slot_hb[no - 1] * G, cb = hb * G;
          if (cb + G > (ca & ~7) + 16) {
            if (no >= SK_TM_MAX_OCT || T.n_pad >= 8) return 0;
            T.pad_oct[T.n_pad++] = no;
            ++no;
          }
        }
        T.blk_oct0[hb] = no;
        T.blk_noct[hb] = n / 8;
        for (int oc = 0; oc < n / 8; ++oc) {
          if (no >= SK_TM_MAX_OCT) return 0;
          T.oct_off[no] = (blk ? L.k_lo_off[h] : L.k_hi_off[h]) + oc * bits;   // 8 codes = `bits` bytes
          T.oct_rowb[no] = rowb;
          slot_hb[no] = hb;
          ++no;
        }
      }
    while (no & 3) {   // padding slot: offset 0, stride 0 (finite codes against zero query rows)
      if (no >= SK_TM_MAX_OCT || T.n_pad >= 8) return 0;
      T.pad_oct[T.n_pad++] = no;
      ++no;
    }
    if (pass == 0) T.n_trips8 = no / 4;
    else T.n_trips4 = no / 4 - T.n_trips8;
  }
  T.n_ks = no / 2;
  for (int o = 0; o < SK_TM_MAX_OCT; ++o) {
    if (T.oct_off[o] >= (1 << 18) || T.oct_rowb[o] >= (1 << 14)) return 0;
    T.oct_desc[o] = (uint32_t)T.oct_off[o] | ((uint32_t)T.oct_rowb[o] << 18);
  }
  const int base_cols = 2 * (L.n_q_heads <= 8 ? 8 : 32);   // every score column the softmax warps load is initialised by the
                                                           // constant step; no window reaches past them
  for (int ks = 0; ks < T.n_ks; ++ks) {
    int ha = slot_hb[2 * ks], hbb = slot_hb[2 * ks + 1];
    if (ha < 0) ha = hbb;
    if (hbb < 0) hbb = ha;
    if (ha < 0) { T.win[ks] = 0; continue; }   // two padding slots
    const int ca = ha * G, cb = hbb * G;
    const int lo = ca < cb ? ca : cb, hi = (ca > cb ? ca : cb) + G;
    int win = lo & ~7;
    if (win + 16 > base_cols) win = base_cols - 16;
    T.win[ks] = win;
    if (lo < win || hi > win + 16) return 0;
  }
  const int need = base_cols;
  T.ds_cols = round_up(need, 16);
  if (T.ds_cols > 64) return 0;
  T.img_ks_off = T.ds_cols / 8 * 256;
  T.img_scal_off = T.img_ks_off + T.n_ks * 1024;
  T.img_bytes = T.img_scal_off + 2 * 32 * 4;
  T.n_vt = (L.rank_v + 127) / 128;
  T.n_dt = 0;
  for (int t = 0; t < T.n_vt; ++t) {
    const int c0 = 128 * t, c1 = (c0 + 128 < L.rank_v) ? c0 + 128 : L.rank_v;
    if (c0 < L.v_hi_n) { T.dt_tile[T.n_dt] = t; T.dt_blk[T.n_dt] = 0; ++T.n_dt; }
    if (c1 > L.v_hi_n) { T.dt_tile[T.n_dt] = t; T.dt_blk[T.n_dt] = 1; ++T.n_dt; }
  }
  // tensor memory: accumulators (32 columns per tile), value operand (64 per 128-channel tile), key operand (constant step +
  // 8 per k-step), score tile(s)
  T.col_do = 0;
  T.col_av = 32 * T.n_dt;
  T.col_ak = T.col_av + 64 * T.n_vt;
  T.col_ds = T.col_ak + 8 + 8 * T.n_ks;
  T.ds_nbuf = (T.col_ds + 2 * T.ds_cols <= 512) ? 2 : 1;
  if (T.col_ds + T.ds_nbuf * T.ds_cols > 512) return 0;
  // page parts (every block of the format is padded to 16 bytes, so the parts are bulk-copy aligned)
  T.k_bytes = L.k_scale_off;
  T.ks_bytes = L.v_hi_off - L.k_scale_off;
  T.v_bytes = L.v_scale_off - L.v_hi_off;
  T.vs_bytes = round_up(2 * PTOK * 2, 16);
  T.kstride = round_up(T.k_bytes, 128);
  T.vstride = round_up(T.v_bytes, 128);
  T.sstride = round_up(T.ks_bytes + T.vs_bytes, 128);
  int off = 0;
  const int fixed = round_up(T.img_bytes, 128) + 2 * 2 * P_BLK_BYTES + 1024 /* misc */ + 1024 /* barriers */ + 4 * TM_TBL +
                    1024 /* base alignment */;
  const int avail = ctx->smem_optin - fixed;
  // the key rows are consumed first (a few stages cover the memory latency); values and scales wait for the softmax
  // and the value MMAs, about three tiles deeper
  int nk = 5;
  int nv = (avail - nk * T.kstride) / (T.vstride + T.sstride);
  if (nv > 14) nv = 14;
  if (nv < 4) { nk = 3; nv = (avail - nk * T.kstride) / (T.vstride + T.sstride); }
  if (nv < 4) return 0;
  T.n_kstage = nk; T.n_vstage = nv; T.n_sstage = nv;
  T.off_kstage = off; off += nk * T.kstride;
  T.off_vstage = off; off += nv * T.vstride;
  T.off_sstage = off; off += nv * T.sstride;
  off = round_up(off, 128);
  T.off_img = off; off += round_up(T.img_bytes, 128);
  T.off_p = off; off += 2 * 2 * P_BLK_BYTES;
  T.off_misc = off; off += 1024;
  T.off_bar = off; off += 1024;
  T.off_tbl = off; off += 4 * TM_TBL;
  T.smem_bytes = round_up(off, 128);
  if (T.smem_bytes > ctx->smem_optin) return 0;
  TmKernel k = tm_kernel_for(L.n_q_heads, G);
  if (!k) return 0;
  if (sk_need_smem(ctx, k, T.smem_bytes) != cudaSuccess) { cudaGetLastError(); return 0; }
  if (sk_prefer_smem(ctx, qproj_tm_kernel) != cudaSuccess) cudaGetLastError();
  T.ok = 1;
  return 1;
}

int sk_decode_tm(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                 const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes, void* out,
                 const AppendSmallArgs* app) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (!ctx->tm.ok) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  uint8_t* img = (uint8_t*)ws + w.qimg_off;
  if (app) {
    const int n_qp = 2 * L.n_kv_heads * batch;
    if (app->fused) {
      SK_PREFER_SMEM(ctx, step_pre_tm_kernel<true>);
      SK_CUDA_CHECK(ctx, sk_launch(ctx, step_pre_tm_kernel<true>, dim3(n_qp + app->n_tiles * app->n_part), dim3(QP_THREADS), 0, L,
                                   ctx->tm, (const __half*)q, (const __half*)B_k, img, w.qimg_stride, n_qp, *app));
    } else {   // projection partials with the query image, then the quantiser / paged write as a launch of its own
      SK_PREFER_SMEM(ctx, step_pre_tm_kernel<false>);
      SK_CUDA_CHECK(ctx, sk_launch(ctx, step_pre_tm_kernel<false>, dim3(n_qp + app->n_tiles * app->n_part), dim3(QP_THREADS), 0, L,
                                   ctx->tm, (const __half*)q, (const __half*)B_k, img, w.qimg_stride, n_qp, *app));
      const int rw = sk_append_small_write(ctx, app);
      if (rw) return rw;
    }
  } else {
    SK_CUDA_CHECK(ctx, sk_launch(ctx, qproj_tm_kernel, dim3(2 * L.n_kv_heads, batch), dim3(QP_THREADS), 0, L, ctx->tm,
                                 (const __half*)q, (const __half*)B_k, img, w.qimg_stride));
  }
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  TmKernel k = tm_kernel_for(L.n_q_heads, L.group);
  SK_CUDA_CHECK(ctx, sk_launch(ctx, k, dim3(w.n_splits, batch), dim3(TM_THREADS), (size_t)ctx->tm.smem_bytes, L, ctx->tm,
                               (const uint8_t*)img, w.qimg_stride, (const uint8_t*)pool, table, max_pages, seq_lens, parts,
                               w.n_splits));
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out, reinterpret_cast<float*>((uint8_t*)ws + w.slice_off));
  ctx->last_launches = 3 + ((app && !app->fused) ? 1 : 0);
  return rc;
}
