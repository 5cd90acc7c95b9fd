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
//        channels.  One column per (query head, precision block): col = (2 h + blk) G + g, because the per-token scales
//        differ per block.  K = 16 channels = two octets; every k-step writes a 16-column window of the score tile (the
//        B tile is zero outside the octets' own columns).  The code offset 2^(b-1) is one more k-step whose A row is the
//        constant (2^-14, 2^-14, 0...) and whose B tile holds -2^(b-1) 2^-10 sum_c Q_c (hi, lo): it also initialises
//        the tile (accumulate off, N = all columns).
//   softmax  thread = token reads its 2 H_q score columns (tcgen05.ld), applies the per-(token, head, block) key scales
//        in fp32, p' = 2^(s - m + 8) against a LAZY running maximum m (moved only when a tile exceeds it by 2^6, so that
//        P <= 2^14 in fp16), folds the per-token VALUE scales into two fp16 operands P~_blk = p' s_v / M_blk (M_blk = a
//        running power of two >= the scales seen, so the operand cannot overflow) and stores them MN-major.  When a
//        maximum or M_blk moves (rare), the four softmax warps rescale the TMEM accumulators and their running sums.
//   PV   O[channel, head] += c[channel, token] P~[token, head]:  A = exact signed codes (magic-number trick), B = P~ of
//        the channel's block; a 128-channel A tile that straddles the block boundary is multiplied with both operands
//        into two accumulator tiles and each lane keeps its own.
// Warp roles (16 warps, warpgroup-aligned so that setmaxnreg can move registers to the softmax warps):
//   0-3 key rows -> TMEM, 4-7 softmax, 8-11 value rows -> TMEM, 12 page producer (cp.async.bulk ring),
//   13 QK MMA issue, 14 PV MMA issue, 15 TMEM allocation.  All hand-offs are mbarriers; no CTA-wide barrier in the loop.
#include <string.h>

#include "decode_common.cuh"
#include "decode_plan.h"
#include "sk_ptx.cuh"

using namespace skptx;

namespace {

constexpr int PTOK = 64;              // tokens per page on this path
constexpr int TM_THREADS = 512;
constexpr int TM_TBL = 512;           // block-table entries of the CTA's range kept in shared memory
constexpr float P_OFFSET = 8.f;       // p' = 2^(s - m + 8)
constexpr float TAU = 6.f;            // the running maximum may lag the true one by 2^TAU: p' <= 2^14
constexpr float kLog2e = 1.4426950408889634f;
constexpr int BAR_SM = 1;             // named barrier of the four softmax warps
constexpr int P_BLK_BYTES = 8192;     // P~ operand of one precision block: 128 tokens x 32 heads fp16
constexpr uint32_t TM_COLS = 512;     // the whole tensor memory (one CTA per SM)
constexpr int MISC_MREF = 0, MISC_M = 32, MISC_INVM = 34, MISC_RED = 36, MISC_FLAG = 192, MISC_NEWM = 200;   // floats in the misc area
constexpr int RED_STRIDE = 36;

// ---------------------------------------------------------------------------------------------
// D1: latent-space query image of one sequence (see TmPlan).  One block per sequence, 16 warps, a warp per latent
// channel at a time (B_k row coalesced, 8 halves per lane).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(512) qproj_tm_kernel(const __grid_constant__ StarkvLayout L, const __grid_constant__ TmPlan T,
                                                       const __half* __restrict__ q, const __half* __restrict__ B_k,
                                                       uint8_t* __restrict__ img_all, size_t img_stride) {
  __shared__ float qt[SK_TM_MAX_KS * 16][4];   // q~[latent column][g]
  __shared__ float wmax[16];
  __shared__ float cst[128];                   // constant-step value of each score column
  sk_pdl_enter();
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int G = L.group, dh = L.head_dim, sumr = L.sum_rank_k;
  const bool act = lane * 8 < dh;
  const float qscale = L.sm_scale * kLog2e;
  float mx = 0.f;
  for (int c = warp; c < sumr; c += 16) {
    const int h = sk_head_of_col(L, c);
    uint4 x = make_uint4(0, 0, 0, 0);
    if (act) x = *reinterpret_cast<const uint4*>(B_k + (size_t)c * dh + lane * 8);
    const float2 b0 = __half22float2(*reinterpret_cast<const __half2*>(&x.x)), b1 = __half22float2(*reinterpret_cast<const __half2*>(&x.y)),
                 b2 = __half22float2(*reinterpret_cast<const __half2*>(&x.z)), b3 = __half22float2(*reinterpret_cast<const __half2*>(&x.w));
    float a[4];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
      uint4 y = make_uint4(0, 0, 0, 0);
      if (g < G && act) y = *reinterpret_cast<const uint4*>(q + ((size_t)b * L.n_q_heads + h * G + g) * dh + lane * 8);
      const float2 q0 = __half22float2(*reinterpret_cast<const __half2*>(&y.x)), q1 = __half22float2(*reinterpret_cast<const __half2*>(&y.y)),
                   q2 = __half22float2(*reinterpret_cast<const __half2*>(&y.z)), q3 = __half22float2(*reinterpret_cast<const __half2*>(&y.w));
      float s = q0.x * b0.x;
      s = fmaf(q0.y, b0.y, s); s = fmaf(q1.x, b1.x, s); s = fmaf(q1.y, b1.y, s);
      s = fmaf(q2.x, b2.x, s); s = fmaf(q2.y, b2.y, s); s = fmaf(q3.x, b3.x, s);
      a[g] = fmaf(q3.y, b3.y, s);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1)
#pragma unroll
      for (int g = 0; g < 4; ++g) a[g] += __shfl_xor_sync(0xffffffffu, a[g], o);
    if (lane == 0) {
#pragma unroll
      for (int g = 0; g < 4; ++g) {
        const float v = a[g] * qscale;
        qt[c][g] = v;
        mx = fmaxf(mx, fabsf(v));
      }
    }
  }
  if (lane == 0) wmax[warp] = mx;
  __syncthreads();
  float m = 0.f;
#pragma unroll
  for (int i = 0; i < 16; ++i) m = fmaxf(m, wmax[i]);
  // Q = q~ 2^e with max |Q| in [2^5, 2^6): the hi + lo fp16 pair then keeps >= 2^-27 of the largest entry even for the
  // 1/16-scaled channels, and the constant step (-2^(b-1) 2^-10 sum Q) stays below 2^10
  int e = 0;
  if (m > 0.f && m < INFINITY) {
    e = 6 - (int)(((__float_as_uint(m) >> 23) & 0xff) - 126);
    e = e < -100 ? -100 : (e > 100 ? 100 : e);
  }
  const float scale = ldexpf(1.f, e);
  uint8_t* img = img_all + (size_t)b * img_stride;
  // ---- constant step
  if (tid < T.ds_cols) {
    const int hb = tid / G, g = tid % G, h = hb >> 1, blk = hb & 1;
    float C = 0.f;
    if (h < L.n_kv_heads) {
      const int bits = blk ? L.bits_lo : L.bits_hi;
      const int nch = blk ? L.k_lo_n[h] : L.k_hi_n[h];
      const int col0 = L.koff[h] + (blk ? L.k_hi_n[h] : 0);
      float s = 0.f;
      for (int c = 0; c < nch; ++c) {
        const bool s16 = bits == 4 && (c & 1);
        const float a = qt[col0 + c][g] * scale * (s16 ? 0.0625f : 1.f);
        const __half hi = __float2half_rn(a);
        const __half lo = __float2half_rn(a - __half2float(hi));
        s += (__half2float(hi) + __half2float(lo)) * (s16 ? 16.f : 1.f);
      }
      C = -(float)(1 << (bits - 1)) * 0.0009765625f * s;
    }
    cst[tid] = C;
  }
  __syncthreads();
  for (int w = tid; w < T.ds_cols * 8; w += 512) {
    const int n = w >> 3, kp = w & 7;
    uint32_t word = 0;
    if (kp == 0) {
      const float C = cst[n];
      const __half hi = __float2half_rn(C);
      const __half lo = __float2half_rn(C - __half2float(hi));
      word = (uint32_t)__half_as_ushort(hi) | ((uint32_t)__half_as_ushort(lo) << 16);
    }
    *reinterpret_cast<uint32_t*>(img + (n >> 3) * 256 + (n & 7) * 16 + (kp >> 2) * 128 + (kp & 3) * 4) = word;
  }
  // ---- k-step tiles
  for (int idx = tid; idx < T.n_ks * 256; idx += 512) {
    const int ks = idx >> 8, part = (idx >> 7) & 1, w = idx & 127;
    const int n = w >> 3, kp = w & 7;
    const int col = T.win[ks] + n, hb = col / G, g = col % G;
    uint32_t word = 0;
#pragma unroll
    for (int eo = 0; eo < 2; ++eo) {
      const int k = 2 * kp + eo, o = 2 * ks + (k >> 3), kk = k & 7;
      if (T.oct_off[o] < 0 || hb != 2 * T.oct_head[o] + T.oct_blk[o]) continue;
      const bool four = T.oct_bits[o] == 4;
      const int cin = four ? (kk >> 1) + 4 * (kk & 1) : kk;        // register order of the 4-bit dequantisation
      const bool s16 = four && ((kk >> 1) & 1);
      const float a = qt[T.oct_col[o] + cin][g] * scale * (s16 ? 0.0625f : 1.f);
      const __half hi = __float2half_rn(a);
      const __half v = part ? __float2half_rn(a - __half2float(hi)) : hi;
      word |= (uint32_t)__half_as_ushort(v) << (16 * eo);
    }
    *reinterpret_cast<uint32_t*>(img + T.img_ks_off + ks * 1024 + part * 512 + (n >> 3) * 256 + (n & 7) * 16 + (kp >> 2) * 128 +
                                 (kp & 3) * 4) = word;
  }
  if (tid == 0) *reinterpret_cast<float*>(img + T.img_scal_off) = ldexpf(1.f, 24 - e);
}

// ---------------------------------------------------------------------------------------------
// the decode kernel
// ---------------------------------------------------------------------------------------------
struct TmShared {   // addresses every role needs
  uint8_t* smem;
  uint32_t full0, empty0, imgbar, ak_full, qk_done, ds_free, p_full0, av_full, pv_done0;
};

template <int NH, int G>
__global__ void __launch_bounds__(TM_THREADS, 1) decode_tm_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ TmPlan T, const uint8_t* __restrict__ img_all,
    size_t img_stride, const uint8_t* __restrict__ pool, const int32_t* __restrict__ table, int max_pages,
    const int32_t* __restrict__ seq_lens, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(1024) uint8_t smem[];
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);   // warp-uniform to the compiler
  const int split = blockIdx.x, b = blockIdx.y;
  sk_pdl_trigger();

  // barrier area: full[nstage], empty[nstage], then the single barriers
  const int nstage = T.nstage;
  const uint32_t full0 = smem_u32(smem + T.off_bar);
  const uint32_t empty0 = full0 + 8 * nstage;
  const uint32_t imgbar = empty0 + 8 * nstage;
  const uint32_t ak_full = imgbar + 8, qk_done = imgbar + 16, ds_free = imgbar + 24, p_full0 = imgbar + 32 /* [2] */,
                 av_full = imgbar + 48, pv_done0 = imgbar + 56 /* [2] */;
  volatile uint32_t* tmem_slot = reinterpret_cast<volatile uint32_t*>(smem + T.off_bar + 8 * (2 * nstage) + 72);
  int32_t* tbl_s = reinterpret_cast<int32_t*>(smem + T.off_tbl);
  float* misc = reinterpret_cast<float*>(smem + T.off_misc);
  uint8_t* stage_base = smem + T.off_stage;
  const uint32_t page_bytes = (uint32_t)L.page_bytes;

  if (tid == 0) {
    for (int s = 0; s < nstage; ++s) {
      mbar_init(full0 + 8 * s, 1);
      mbar_init(empty0 + 8 * s, 8);   // 2 key warps + 2 softmax warps + 4 value warps read a page
    }
    mbar_init(imgbar, 1);
    mbar_init(ak_full, 4);
    mbar_init(qk_done, 1);
    mbar_init(ds_free, 4);
    mbar_init(p_full0, 4);
    mbar_init(p_full0 + 8, 4);
    mbar_init(av_full, 4);
    mbar_init(pv_done0, 1);
    mbar_init(pv_done0 + 8, 1);
    fence_barrier_init();
  }
  if (warp == 15) tmem_alloc(smem_u32((const void*)tmem_slot), TM_COLS);
  if (tid < 36) misc[tid] = tid < 32 ? 0.f : (tid < 34 ? 0.f : 1.f);   // m = 0, M = 0 (forces the first update), 1/M = 1

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
  } else if (warp < 4) {
    // =============================== key rows -> A operand of the score product ===============================
    setmaxnreg_dec<80>();
    const int wq = warp, tq = wq * 32 + lane, pgsel = tq >> 6, slot = tq & 63;
    const uint32_t tl = tbase + ((uint32_t)(wq * 32) << 16) + (uint32_t)T.col_ak;
    {
      const uint32_t c[8] = {0x04000400u, 0u, 0u, 0u, 0u, 0u, 0u, 0u};   // constant step: (2^-14, 2^-14, 0, ...)
      tmem_st8(tl, c);
    }
    for (int it = 0; it < n_it; ++it) {
      const int j = 2 * it + pgsel;
      const bool exists = j < n_pg;
      const int st = j % nstage;
      if (exists) mbar_wait(full0 + 8 * st, (uint32_t)((j / nstage) & 1));
      if (it > 0) {   // the previous tile's score MMAs have read the operand
        mbar_wait(qk_done, (uint32_t)((it - 1) & 1));
        tc_fence_after();
      }
      const uint8_t* row = stage_base + (size_t)st * page_bytes;
      for (int ks = 0; ks < T.n_ks; ++ks) {
        uint32_t r[8];
#pragma unroll
        for (int hf = 0; hf < 2; ++hf) {
          const int o = 2 * ks + hf;
          const int off = T.oct_off[o];
          if (off < 0) {
            r[4 * hf] = r[4 * hf + 1] = r[4 * hf + 2] = r[4 * hf + 3] = 0u;
          } else {
            const uint8_t* p = row + off + slot * T.oct_rowb[o];
            if (T.oct_bits[o] == 8) {
              const uint2 x = *reinterpret_cast<const uint2*>(p);
              r[4 * hf] = prmt(x.x, 0u, 0x4140u);       // (u0, u1) as fp16 subnormals u 2^-24
              r[4 * hf + 1] = prmt(x.x, 0u, 0x4342u);
              r[4 * hf + 2] = prmt(x.y, 0u, 0x4140u);
              r[4 * hf + 3] = prmt(x.y, 0u, 0x4342u);
            } else {
              const uint32_t w = *reinterpret_cast<const uint32_t*>(p);
              const uint32_t w2 = w >> 8;
              r[4 * hf] = w & 0x000f000fu;              // (u0, u4)
              r[4 * hf + 1] = w & 0x00f000f0u;          // 16 (u1, u5): the 16 is taken out of the query image
              r[4 * hf + 2] = w2 & 0x000f000fu;         // (u2, u6)
              r[4 * hf + 3] = w2 & 0x00f000f0u;         // 16 (u3, u7)
            }
          }
        }
        tmem_st8(tl + 8 + 8 * ks, r);
      }
      tmem_wait_st();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(ak_full);
        if (exists) mbar_arrive(empty0 + 8 * st);
      }
    }
  } else if (warp < 8) {
    // ========================================= softmax (thread = token) =========================================
    setmaxnreg_inc<216>();
    const int wq = warp - 4, tq = wq * 32 + lane, pgsel = tq >> 6, slot = tq & 63;
    const uint32_t tlane = tbase + ((uint32_t)(wq * 32) << 16);
    float* mref_s = misc + MISC_MREF;
    float* M_s = misc + MISC_M;
    float* invM_s = misc + MISC_INVM;
    float* red = misc + MISC_RED;
    volatile int* flag = reinterpret_cast<volatile int*>(misc + MISC_FLAG);   // [2][4]
    float* mnew_s = misc + MISC_NEWM;
    const int Hq = L.n_q_heads, n_kv = L.n_kv_heads;
    // position of this token along K of the value product, per precision block (4-bit rows are dequantised in the
    // order 0,4,1,5,2,6,3,7 inside every 8 slots)
    uint32_t paddr[2];
#pragma unroll
    for (int blk = 0; blk < 2; ++blk) {
      const int bits = blk ? L.bits_lo : L.bits_hi;
      const int i8 = slot & 7;
      const int kp = 64 * pgsel + (bits == 4 ? (slot & ~7) + (i8 < 4 ? 2 * i8 : 2 * (i8 - 4) + 1) : slot);
      paddr[blk] = (uint32_t)(blk * P_BLK_BYTES + (kp >> 3) * 128 + (kp & 7) * 16);
    }
    float l_acc[NH];
#pragma unroll
    for (int i = 0; i < NH; ++i) l_acc[i] = 0.f;
    mbar_wait(imgbar, 0);
    const float c_e = *reinterpret_cast<const float*>(smem + T.off_img + T.img_scal_off);

    for (int it = 0; it < n_it; ++it) {
      const int j = 2 * it + pgsel;
      const bool exists = j < n_pg;
      const int st = j % nstage;
      const int buf = it & 1;
      mbar_wait(qk_done, (uint32_t)(it & 1));
      tc_fence_after();
      uint32_t d[2 * NH];
      tmem_ld<2 * NH>(tlane + (uint32_t)T.col_ds, d);
      tmem_wait_ld();
      tc_fence_before();
      __syncwarp();
      if (lane == 0) mbar_arrive(ds_free);
      if (exists) mbar_wait(full0 + 8 * st, (uint32_t)((j / nstage) & 1));
      const uint8_t* page = stage_base + (size_t)st * page_bytes;
      const uint16_t* ksc = reinterpret_cast<const uint16_t*>(page + L.k_scale_off) + slot;
      const uint16_t* vsc = reinterpret_cast<const uint16_t*>(page + L.v_scale_off) + slot;
      const bool valid = exists && ((p0 + j) * PTOK + slot) < len;
      float arg[NH];
#pragma unroll
      for (int h = 0; h < NH / G; ++h) {
        float shi = 0.f, slo = 0.f;
        if (h < n_kv && valid) {
          shi = h_bits_to_f(ksc[(2 * h) * PTOK]) * c_e;
          slo = h_bits_to_f(ksc[(2 * h + 1) * PTOK]) * c_e;
        }
#pragma unroll
        for (int g = 0; g < G; ++g) {
          const int i = h * G + g;
          const float s = fmaf(shi, __uint_as_float(d[2 * h * G + g]), slo * __uint_as_float(d[2 * h * G + G + g]));
          arg[i] = valid ? s - mref_s[i] : -INFINITY;
        }
      }
      float sv0 = 0.f, sv1 = 0.f;
      if (valid) {
        sv0 = h_bits_to_f(vsc[0]);
        sv1 = h_bits_to_f(vsc[PTOK]);
      }
      float mxa = -INFINITY;
#pragma unroll
      for (int i = 0; i < NH; ++i)
        if (i < Hq) mxa = fmaxf(mxa, arg[i]);
      bool trig = valid && (mxa > TAU || sv0 > M_s[0] || sv1 > M_s[1]);
      if (it == 0) trig = true;
      const bool wany = __any_sync(0xffffffffu, trig);
      if (lane == 0) flag[buf * 4 + wq] = wany ? 1 : 0;
      bar_sync(BAR_SM, 128);
      const bool upd = (flag[buf * 4] | flag[buf * 4 + 1] | flag[buf * 4 + 2] | flag[buf * 4 + 3]) != 0;
      if (upd) {
        // ---- a maximum (or a value-scale bound) moves: new reference, rescale the running sums and the accumulators
#pragma unroll
        for (int i = 0; i < NH; ++i) {
          float v = valid ? arg[i] + mref_s[i] : -INFINITY;   // the score itself
#pragma unroll
          for (int o = 16; o; o >>= 1) v = fmaxf(v, __shfl_xor_sync(0xffffffffu, v, o));
          if (lane == 0) red[wq * RED_STRIDE + i] = v;
        }
        {
          float a0 = sv0, a1 = sv1;
#pragma unroll
          for (int o = 16; o; o >>= 1) {
            a0 = fmaxf(a0, __shfl_xor_sync(0xffffffffu, a0, o));
            a1 = fmaxf(a1, __shfl_xor_sync(0xffffffffu, a1, o));
          }
          if (lane == 0) { red[wq * RED_STRIDE + 32] = a0; red[wq * RED_STRIDE + 33] = a1; }
        }
        bar_sync(BAR_SM, 128);
        float fs[NH];
#pragma unroll
        for (int i = 0; i < NH; ++i) {
          const float mt = fmaxf(fmaxf(red[i], red[RED_STRIDE + i]), fmaxf(red[2 * RED_STRIDE + i], red[3 * RED_STRIDE + i]));
          const float m_old = mref_s[i];
          // only a maximum that the tile exceeds moves (to the true maximum so far); the first tile sets it
          float m_new = (it == 0) ? mt : (mt > m_old ? mt : m_old);
          if (m_new == -INFINITY) m_new = m_old;   // (no valid token in the tile: cannot happen for it == 0)
          const float delta = m_old - m_new;       // <= 0
          fs[i] = ex2(delta);
          arg[i] += delta;
          l_acc[i] *= fs[i];
          mnew_s[i] = m_new;                       // (every thread computes and stores the same value)
        }
        float fM[2], Mn[2];
#pragma unroll
        for (int blk = 0; blk < 2; ++blk) {
          const float sm = fmaxf(fmaxf(red[32 + blk], red[RED_STRIDE + 32 + blk]),
                                 fmaxf(red[2 * RED_STRIDE + 32 + blk], red[3 * RED_STRIDE + 32 + blk]));
          const float M_old = M_s[blk];
          float M_new = M_old;
          if (sm > M_old) {   // next power of two above the largest scale seen
            const uint32_t eb = (__float_as_uint(sm) >> 23) & 0xffu;
            M_new = eb >= 254u ? sm : __uint_as_float((eb + 1u) << 23);
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
            uint32_t v[NH];
            tmem_ld<NH>(tlane + (uint32_t)(T.col_do + 32 * dt), v);
            tmem_wait_ld();
#pragma unroll
            for (int i = 0; i < NH; ++i) v[i] = __float_as_uint(__uint_as_float(v[i]) * (fs[i] * fb));
            tmem_st<NH>(tlane + (uint32_t)(T.col_do + 32 * dt), v);
          }
          tmem_wait_st();
          tc_fence_before();
        }
        bar_sync(BAR_SM, 128);   // every thread has read the old references
        if (tq < NH) mref_s[tq] = mnew_s[tq];
        if (tq == 0) {
          M_s[0] = Mn[0]; M_s[1] = Mn[1];
          invM_s[0] = 1.f / Mn[0]; invM_s[1] = 1.f / Mn[1];
        }
        bar_sync(BAR_SM, 128);
      }
      // ---- p' and the two scaled operands
      const float a0 = sv0 * invM_s[0], a1 = sv1 * invM_s[1];
      if (it >= 2) mbar_wait(pv_done0 + 8 * buf, (uint32_t)(((it >> 1) - 1) & 1));   // the MMAs of tile it - 2 have read the buffer
      uint8_t* pb = smem + T.off_p + buf * 2 * P_BLK_BYTES;
#pragma unroll
      for (int oc = 0; oc < NH / 8; ++oc) {
        float p[8];
#pragma unroll
        for (int k = 0; k < 8; ++k) {
          p[k] = ex2(arg[8 * oc + k] + P_OFFSET);   // -inf -> 0 for slots past the sequence end
          l_acc[8 * oc + k] += p[k];
        }
        uint4 x0, x1;
        x0.x = pack_h2(p[0] * a0, p[1] * a0); x0.y = pack_h2(p[2] * a0, p[3] * a0);
        x0.z = pack_h2(p[4] * a0, p[5] * a0); x0.w = pack_h2(p[6] * a0, p[7] * a0);
        x1.x = pack_h2(p[0] * a1, p[1] * a1); x1.y = pack_h2(p[2] * a1, p[3] * a1);
        x1.z = pack_h2(p[4] * a1, p[5] * a1); x1.w = pack_h2(p[6] * a1, p[7] * a1);
        *reinterpret_cast<uint4*>(pb + paddr[0] + oc * 2048) = x0;
        *reinterpret_cast<uint4*>(pb + paddr[1] + oc * 2048) = x1;
      }
      fence_proxy_async();   // generic-proxy stores -> visible to the tensor core's reads
      __syncwarp();
      if (lane == 0) {
        mbar_arrive(p_full0 + 8 * buf);
        if (exists) mbar_arrive(empty0 + 8 * st);
      }
    }
    // ---- split-K partial (D7): [m, l, 0, 0, acc[r_v]] per head
    {
      const int last = n_it - 1;
      mbar_wait(pv_done0 + 8 * (last & 1), (uint32_t)((last >> 1) & 1));
      tc_fence_after();
      for (int dt = 0; dt < T.n_dt; ++dt) {
        const int blk = T.dt_blk[dt] ? 1 : 0;
        const int ch = 128 * T.dt_tile[dt] + tq;
        uint32_t v[NH];
        tmem_ld<NH>(tlane + (uint32_t)(T.col_do + 32 * dt), v);
        tmem_wait_ld();
        const bool mine = ch < L.rank_v && ((ch >= L.v_hi_n) == (blk == 1));
        const float Mb = M_s[blk];
        if (mine) {
#pragma unroll
          for (int i = 0; i < NH; ++i)
            if (i < Hq) my_parts[(size_t)i * pstride + SK_PART_ACC + ch] = __uint_as_float(v[i]) * Mb;
        }
      }
#pragma unroll
      for (int i = 0; i < NH; ++i) {
        float v = l_acc[i];
#pragma unroll
        for (int o = 16; o; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
        if (lane == 0) red[wq * RED_STRIDE + i] = v;
      }
      bar_sync(BAR_SM, 128);
      if (tq < Hq) {
        const float lsum = red[tq] + red[RED_STRIDE + tq] + red[2 * RED_STRIDE + tq] + red[3 * RED_STRIDE + tq];
        *reinterpret_cast<float4*>(my_parts + (size_t)tq * pstride) = make_float4(mref_s[tq], lsum, 0.f, 0.f);
      }
    }
  } else if (warp < 12) {
    // =============================== value rows -> A operand of the value product ===============================
    setmaxnreg_inc<136>();
    const int wq = warp - 8, tq = wq * 32 + lane;
    const uint32_t tl = tbase + ((uint32_t)(wq * 32) << 16) + (uint32_t)T.col_av;
    const int BH = L.bits_hi, BL = L.bits_lo;
    for (int it = 0; it < n_it; ++it) {
      const int jA = 2 * it;
      const bool existsB = jA + 1 < n_pg;
      const int stA = jA % nstage, stB = (jA + 1) % nstage;
      mbar_wait(full0 + 8 * stA, (uint32_t)((jA / nstage) & 1));
      if (existsB) mbar_wait(full0 + 8 * stB, (uint32_t)(((jA + 1) / nstage) & 1));
      if (it > 0) {   // the previous tile's value MMAs have read the operand
        mbar_wait(pv_done0 + 8 * ((it - 1) & 1), (uint32_t)(((it - 1) >> 1) & 1));
        tc_fence_after();
      }
      for (int m = 0; m < T.n_vt; ++m) {
        const int ch = 128 * m + tq;
        const bool act = ch < L.rank_v;
        const bool lo = ch >= L.v_hi_n;
        const int bits = lo ? BL : BH;
        const int rowb = PTOK * bits / 8;
        const int roff = lo ? L.v_lo_off + (ch - L.v_hi_n) * rowb : L.v_hi_off + ch * rowb;
#pragma unroll
        for (int pg = 0; pg < 2; ++pg) {
          const uint8_t* rowp = stage_base + (size_t)(pg ? stB : stA) * page_bytes + roff;
          uint32_t r[32];
          if (!act) {
#pragma unroll
            for (int k = 0; k < 32; ++k) r[k] = 0u;
          } else if (bits == 4) {
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
        mbar_arrive(av_full);
        mbar_arrive(empty0 + 8 * stA);
        if (existsB) mbar_arrive(empty0 + 8 * stB);
      }
    }
  } else {
    setmaxnreg_dec<64>();
    if (warp == 12) {
      // ================================== page producer (D2) ==================================
      if (elect_one()) {
        const uint64_t pol = l2_evict_first_policy();
        mbar_expect_tx(imgbar, (uint32_t)T.img_bytes);
        bulk_g2s(smem_u32(smem + T.off_img), img_all + (size_t)b * img_stride, (uint32_t)T.img_bytes, imgbar);
        for (int j = 0; j < n_pg; ++j) {
          const int st = j % nstage;
          if (j >= nstage) mbar_wait(empty0 + 8 * st, (uint32_t)(((j / nstage) - 1) & 1));
          const int page = j < TM_TBL ? tbl_s[j] : my_table[j];
          mbar_expect_tx(full0 + 8 * st, page_bytes);
          bulk_g2s_stream(smem_u32(stage_base + (size_t)st * page_bytes), pool + (size_t)page * page_bytes, page_bytes,
                          full0 + 8 * st, pol);
        }
      }
      __syncwarp();
    } else if (warp == 13) {
      // ================================== score MMAs ==================================
      mbar_wait(imgbar, 0);
      const uint32_t img_s = smem_u32(smem + T.off_img);
      const uint64_t dconst = umma_desc(img_s, 128, 256);
      const uint64_t dks = umma_desc(img_s + (uint32_t)T.img_ks_off, 128, 256);
      const uint32_t id_const = umma_idesc_f16(T.ds_cols, false), id_win = umma_idesc_f16(16, false);
      const uint32_t t_ds = tbase + (uint32_t)T.col_ds, t_ak = tbase + (uint32_t)T.col_ak;
      for (int it = 0; it < n_it; ++it) {
        mbar_wait(ak_full, (uint32_t)(it & 1));
        if (it > 0) mbar_wait(ds_free, (uint32_t)((it - 1) & 1));
        tc_fence_after();
        if (elect_one()) {
          umma_ts_f16(t_ds, t_ak, dconst, id_const, 0u);
          for (int ks = 0; ks < T.n_ks; ++ks) {
            const uint32_t dcol = t_ds + (uint32_t)T.win[ks];
            const uint64_t db = dks + (uint64_t)(ks * 64);
            umma_ts_f16(dcol, t_ak + 8 + 8 * ks, db, id_win, 1u);
            umma_ts_f16(dcol, t_ak + 8 + 8 * ks, db + 32, id_win, 1u);
          }
          umma_commit(qk_done);
        }
        __syncwarp();
      }
    } else if (warp == 14) {
      // ================================== value MMAs ==================================
      const uint32_t id_pv = umma_idesc_f16(32, true);
      const uint32_t t_do = tbase + (uint32_t)T.col_do, t_av = tbase + (uint32_t)T.col_av;
      const uint32_t p_s = smem_u32(smem + T.off_p);
      for (int it = 0; it < n_it; ++it) {
        const int buf = it & 1;
        mbar_wait(p_full0 + 8 * buf, (uint32_t)((it >> 1) & 1));
        mbar_wait(av_full, (uint32_t)(it & 1));
        tc_fence_after();
        if (elect_one()) {
          for (int dt = 0; dt < T.n_dt; ++dt) {
            const uint64_t dp = umma_desc(p_s + (uint32_t)(buf * 2 * P_BLK_BYTES + (T.dt_blk[dt] ? P_BLK_BYTES : 0)), 128, 2048);
            const uint32_t ta = t_av + (uint32_t)(64 * T.dt_tile[dt]);
            const uint32_t td = t_do + (uint32_t)(32 * dt);
#pragma unroll
            for (int ks = 0; ks < 8; ++ks) umma_ts_f16(td, ta + 8 * ks, dp + (uint64_t)(ks * 16), id_pv, (it > 0 || ks > 0) ? 1u : 0u);
          }
          umma_commit(pv_done0 + 8 * buf);
        }
        __syncwarp();
      }
    }
  }

  tc_fence_before();
  __syncthreads();
  if (warp == 15) tmem_dealloc(tbase, TM_COLS);
}

typedef void (*TmKernel)(const StarkvLayout, const TmPlan, const uint8_t*, size_t, const uint8_t*, const int32_t*, int,
                         const int32_t*, float*, int);

TmKernel tm_kernel_for(int n_q_heads, int G) {
  const bool small = n_q_heads <= 8;
  switch (G) {
    case 1: return small ? decode_tm_kernel<8, 1> : decode_tm_kernel<32, 1>;
    case 2: return small ? decode_tm_kernel<8, 2> : decode_tm_kernel<32, 2>;
    case 4: return small ? decode_tm_kernel<8, 4> : decode_tm_kernel<32, 4>;
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
  if (L.rank_v > 256) return 0;
  // octets in cache order: head by head, leading block then trailing block
  int no = 0;
  for (int h = 0; h < L.n_kv_heads; ++h)
    for (int blk = 0; blk < 2; ++blk) {
      const int n = blk ? L.k_lo_n[h] : L.k_hi_n[h];
      const int bits = blk ? L.bits_lo : L.bits_hi;
      const int rowb = n * bits / 8;
      for (int oc = 0; oc < n / 8; ++oc) {
        if (no >= SK_TM_MAX_OCT) return 0;
        T.oct_off[no] = (blk ? L.k_lo_off[h] : L.k_hi_off[h]) + oc * bits;   // 8 codes = `bits` bytes
        T.oct_rowb[no] = rowb;
        T.oct_bits[no] = bits;
        T.oct_head[no] = h;
        T.oct_blk[no] = blk;
        T.oct_col[no] = L.koff[h] + (blk ? L.k_hi_n[h] : 0) + 8 * oc;
        ++no;
      }
    }
  T.n_ks = (no + 1) / 2;
  for (int o = no; o < SK_TM_MAX_OCT; ++o) { T.oct_off[o] = -1; T.oct_bits[o] = 8; }
  int need = 2 * (L.n_q_heads <= 8 ? 8 : 32);   // every score column the softmax warps load is initialised by the constant step
  for (int ks = 0; ks < T.n_ks; ++ks) {
    const int oa = 2 * ks, ob = (2 * ks + 1 < no) ? 2 * ks + 1 : oa;
    const int ca = (2 * T.oct_head[oa] + T.oct_blk[oa]) * G, cb = (2 * T.oct_head[ob] + T.oct_blk[ob]) * G;
    const int lo = ca < cb ? ca : cb, hi = (ca > cb ? ca : cb) + G;
    T.win[ks] = lo & ~7;
    if (hi > T.win[ks] + 16) return 0;
    if (T.win[ks] + 16 > need) need = T.win[ks] + 16;
  }
  T.ds_cols = round_up(need, 16);
  if (T.ds_cols > 112) return 0;
  T.img_ks_off = T.ds_cols / 8 * 256;
  T.img_scal_off = T.img_ks_off + T.n_ks * 1024;
  T.img_bytes = T.img_scal_off + 16;
  T.n_vt = (L.rank_v + 127) / 128;
  T.n_dt = 0;
  for (int t = 0; t < T.n_vt; ++t) {
    const int c0 = 128 * t, c1 = (c0 + 128 < L.rank_v) ? c0 + 128 : L.rank_v;
    if (c0 < L.v_hi_n) { T.dt_tile[T.n_dt] = t; T.dt_blk[T.n_dt] = 0; ++T.n_dt; }
    if (c1 > L.v_hi_n) { T.dt_tile[T.n_dt] = t; T.dt_blk[T.n_dt] = 1; ++T.n_dt; }
  }
  T.col_do = 0; T.col_av = 128; T.col_ak = 256; T.col_ds = 400;
  int off = 0;
  const int fixed = round_up(T.img_bytes, 128) + 2 * 2 * P_BLK_BYTES + 1024 /* misc */ + 512 /* barriers */ + 4 * TM_TBL +
                    1024 /* base alignment */;
  int ns = (ctx->smem_optin - fixed) / L.page_bytes;
  if (ns > 12) ns = 12;
  if (ns < 4) return 0;
  T.nstage = ns;
  T.off_stage = off; off += ns * L.page_bytes;
  off = round_up(off, 128);
  T.off_img = off; off += round_up(T.img_bytes, 128);
  T.off_p = off; off += 2 * 2 * P_BLK_BYTES;
  T.off_misc = off; off += 1024;
  T.off_bar = off; off += 512;
  T.off_tbl = off; off += 4 * TM_TBL;
  T.smem_bytes = round_up(off, 128);
  if (T.smem_bytes > ctx->smem_optin) return 0;
  TmKernel k = tm_kernel_for(L.n_q_heads, G);
  if (!k) return 0;
  // attributes are per device: set for the device this context was created on, every time a context is created
  if (cudaFuncSetAttribute(k, cudaFuncAttributeMaxDynamicSharedMemorySize, T.smem_bytes) != cudaSuccess) { cudaGetLastError(); return 0; }
  cudaFuncSetAttribute(qproj_tm_kernel, cudaFuncAttributePreferredSharedMemoryCarveout, (int)cudaSharedmemCarveoutMaxShared);
  cudaGetLastError();
  T.ok = 1;
  return 1;
}

int sk_decode_tm(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                 const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes, void* out) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (!ctx->tm.ok) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  uint8_t* img = (uint8_t*)ws + w.qimg_off;
  SK_CUDA_CHECK(ctx, sk_launch(ctx, qproj_tm_kernel, dim3(batch), dim3(512), 0, L, ctx->tm, (const __half*)q, (const __half*)B_k,
                               img, w.qimg_stride));
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  TmKernel k = tm_kernel_for(L.n_q_heads, L.group);
  SK_CUDA_CHECK(ctx, sk_launch(ctx, k, dim3(w.n_splits, batch), dim3(TM_THREADS), (size_t)ctx->tm.smem_bytes, L, ctx->tm,
                               (const uint8_t*)img, w.qimg_stride, (const uint8_t*)pool, table, max_pages, seq_lens, parts,
                               w.n_splits));
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out);
  ctx->last_launches = 3;
  return rc;
}
