// Compress-on-append for many new tokens (prefill), rows A1-A4 in ONE kernel on the 5th-generation tensor cores:
// z = X . A by TMA + tcgen05.mma with the fp32 accumulator in tensor memory, and the quantiser + paged write as the
// TMEM epilogue.
//   PAPER.md section 3.2 L58 (K' = x (Sigma V)_K per head, V' = x (Sigma V)_V joint), section 4.4 L204-210 / Eq.12
//   (leading channels at bits_hi, trailing at bits_lo, per token); A11 (quantiser), A15 (dense-KV and
//   hidden-state input modes are one strided GEMM), "Cache page format v1".
// One CTA computes a 128-token x N-column tile (N <= 512 = the whole tensor memory):
//   warp 0      TMA producer: cp.async.bulk.tensor (128-byte swizzle) of the X tile [128 tokens x 64 k] and of the factor
//               tile as [64 k x 64 columns] boxes into a ring of stages, completion counted on the stage's `full` mbarrier
//   warp 1      tcgen05.mma issue (cta_group::1, kind::f16, M = 128, N <= 256 per instruction, two column halves when
//               N > 256, K = 16; X is the K-major A operand, the factor is the MN-major B operand: it is [d_in, columns]
//               row-major, i.e. column-contiguous, so no transpose is ever materialised); tcgen05.commit releases a stage
//               (`empty`) and, after the last k block, signals the epilogue
//   warps 2-5   epilogue, thread = token (TMEM lane): per (head, precision block) segment of the tile, one pass of
//               tcgen05.ld for the row's absmax (after the single rounding to fp16), the fp16 scale, a second pass for
//               the RNE codes, packed and stored straight into the token's page: key rows token-major (whole words),
//               value fields channel-major (consecutive lanes = consecutive slots, so a warp's stores to a channel row
//               coalesce; two 4-bit slots share a byte: paired through a shuffle when the neighbouring lane is the
//               neighbouring slot, atomicAnd/atomicOr otherwise).  No intermediate z in HBM, no second kernel.
// Tiles are made of whole heads (key columns of one or several KV heads; the joint value columns are one tile), so a
// per-token scale never needs another CTA's columns.  When the value rank exceeds 512 columns, the unfused variant
// writes z = fp16(X . A) to the workspace and append_write_kernel (codec.cu) quantises it.
// K tails and partial tiles are handled by the tensor maps' zero fill of out-of-range boxes (factor rows >= d_in read
// as zero, so X columns past a head's own d_in contribute nothing).
#include <cuda.h>
#include <string.h>

#include "common.cuh"
#include "ctx.h"
#include "sk_ptx.cuh"

using namespace skptx;

namespace {

constexpr int GM = 128, GK = 64;
constexpr int GA_BYTES = GM * GK * 2;            // 16 KB: 128 rows of 128 bytes
constexpr int GB_BOX = GK * 64 * 2;              // 8 KB: 64 k rows of 128 bytes (64 columns)
constexpr int G_THREADS = 64 + 4 * 3 * 32;   // producer, MMA issue, 12 epilogue warps (GE = 3 per TMEM lane quarter)
constexpr int G_MAX_TILES = 72;

struct GemmTile {
  int16_t src;       // 0 = keys (X_k, A_k), 1 = values (X_v, A_v)
  int16_t h0, nh;    // fused key tile: first KV head and number of heads; value tile: h0 = precision block
  int16_t ncols;     // valid columns (multiple of 8)
  int32_t x_col0;    // first X column of the tile's K range
  int32_t w_col0;    // first factor column (= first z column for keys; sum_rank_k + it for values)
  int32_t d_in;
};
struct GemmPlan {
  int32_t n_tiles, n_new, R;
  int32_t stage_bytes, n_stages, tmem_cols, n_seg_max;
  const int32_t* seq_ids;
  const int32_t* positions;
  const int32_t* table;
  int32_t max_pages;
  uint8_t* pool;
  GemmTile t[G_MAX_TILES];
};

// shared-memory matrix descriptors, 128-byte swizzle (layout type 2 at bit 61), version 1 at bit 46
__device__ __forceinline__ uint64_t desc_sw128(uint32_t saddr, uint32_t lbo, uint32_t sbo) {
  return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(lbo >> 4) << 16) | ((uint64_t)(sbo >> 4) << 32) | ((uint64_t)1 << 46) |
         ((uint64_t)2 << 61);
}
__device__ __forceinline__ void umma_ss_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ void tma_load_2d(uint32_t dst, const CUtensorMap* map, int c0, int c1, uint32_t bar) {
  asm volatile("cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst),
               "l"(map), "r"(c0), "r"(c1), "r"(bar)
               : "memory");
}

// eight accumulator columns of this thread's row, rounded once to fp16 (the latent the quantiser sees)
__device__ __forceinline__ void ld8_h(uint32_t taddr, __half (&h)[8]) {
  uint32_t v[8];
  tmem_ld8(taddr, v);
  tmem_wait_ld();
#pragma unroll
  for (int k = 0; k < 8; ++k) h[k] = __float2half_rn(__uint_as_float(v[k]));
}

// Epilogue work split: GE warps share each TMEM lane quarter (a warp may read the lanes [32 (w % 4), +32)); the 8-column
// chunks of a segment go round-robin to the quarter's warps, the per-token absmax of a segment is combined through a
// shared-memory table (atomicMax on the bits of a non-negative float), one named barrier between the two passes.
constexpr int GE = 3;
constexpr int G_EPI_THREADS = 4 * GE * 32;

// segment i of a tile: a (head, precision block) of a key tile, or the tile's value block
struct Seg { int c0, n, bits, h, blk; };
__device__ __forceinline__ Seg seg_of(const StarkvLayout& L, const GemmTile& T, int i) {
  Seg s;
  if (T.src) {
    s.h = 0; s.blk = T.h0; s.c0 = 0; s.n = T.ncols; s.bits = T.h0 ? L.bits_lo : L.bits_hi;
  } else if (L.bits_hi == 16) {
    s.h = T.h0 + i; s.blk = 0; s.c0 = L.koff[s.h] - L.koff[T.h0]; s.n = L.k_hi_n[s.h]; s.bits = 16;
  } else {
    s.h = T.h0 + (i >> 1); s.blk = i & 1;
    s.c0 = L.koff[s.h] - L.koff[T.h0] + (s.blk ? L.k_hi_n[s.h] : 0);
    s.n = s.blk ? L.k_lo_n[s.h] : L.k_hi_n[s.h];
    s.bits = s.blk ? L.bits_lo : L.bits_hi;
  }
  return s;
}

// codes of 8 columns of a key row -> the row's bytes (row = nullptr: the token is not written)
__device__ __forceinline__ void key_chunk(const __half (&h)[8], int c, int bits, float sf, uint8_t* row) {
  if (bits == 16) {
    if (row) *reinterpret_cast<uint4*>(row + 2 * c) = *reinterpret_cast<const uint4*>(h);
  } else if (bits == 8) {
    uint32_t w[2] = {0u, 0u};
#pragma unroll
    for (int k = 0; k < 8; ++k) w[k >> 2] |= (uint32_t)(sk_code_of(__half2float(h[k]), sf, 127) + 128) << (8 * (k & 3));
    if (row) *reinterpret_cast<uint2*>(row + c) = make_uint2(w[0], w[1]);
  } else {
    uint32_t w = 0u;
#pragma unroll
    for (int k = 0; k < 8; ++k) w |= (uint32_t)(sk_code_of(__half2float(h[k]), sf, 7) + 8) << (4 * k);
    if (row) *reinterpret_cast<uint32_t*>(row + (c >> 1)) = w;
  }
}

// codes of 8 channels of a value block -> channel-major rows of P slots (base = nullptr: the token is not written)
__device__ __forceinline__ void value_chunk(const __half (&h)[8], int c, int bits, float sf, int P, uint8_t* base, int slot,
                                            bool paired) {
  const bool wr = base != nullptr;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int idx = c + k;
    if (bits == 16) {
      if (wr) reinterpret_cast<__half*>(base)[(size_t)idx * P + slot] = h[k];
    } else if (bits == 8) {
      if (wr) base[(size_t)idx * P + slot] = (uint8_t)(sk_code_of(__half2float(h[k]), sf, 127) + 128);
    } else {
      const unsigned u = (unsigned)(sk_code_of(__half2float(h[k]), sf, 7) + 8);
      const unsigned up = __shfl_xor_sync(0xffffffffu, u, 1);   // the neighbouring lane's field
      if (wr) {
        const size_t byte = (size_t)idx * (P / 2) + (slot >> 1);
        if (paired) {
          if (!(slot & 1)) base[byte] = (uint8_t)(u | (up << 4));
        } else {
          unsigned* word = reinterpret_cast<unsigned*>(base + (byte & ~(size_t)3));
          const int sh = 8 * (int)(byte & 3) + 4 * (slot & 1);
          atomicAnd(word, ~(0xFu << sh));
          atomicOr(word, u << sh);
        }
      }
    }
  }
}

template <bool FUSED>
__global__ void __launch_bounds__(G_THREADS) append_gemm_kernel(const __grid_constant__ StarkvLayout L,
                                                                const __grid_constant__ GemmPlan P,
                                                                const __grid_constant__ CUtensorMap map_xk,
                                                                const __grid_constant__ CUtensorMap map_xv,
                                                                const __grid_constant__ CUtensorMap map_wk,
                                                                const __grid_constant__ CUtensorMap map_wv,
                                                                __half* __restrict__ z) {
  extern __shared__ uint8_t gsm_raw[];
  __shared__ uint32_t tmem_slot;
  const uint32_t sbase = (smem_u32(gsm_raw) + 1023u) & ~1023u;   // 128-byte swizzle atoms are 1024-byte aligned
  const int n_st = P.n_stages;
  const uint32_t stage_bytes = (uint32_t)P.stage_bytes;
  const uint32_t full0 = sbase + n_st * stage_bytes, empty0 = full0 + 8 * n_st, accbar = empty0 + 8 * n_st;
  uint32_t* amax_tab = reinterpret_cast<uint32_t*>(gsm_raw + (sbase - smem_u32(gsm_raw)) + n_st * stage_bytes + 256);   // [segment][token row]
  const int tid = threadIdx.x, lane = tid & 31;
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const GemmTile& T = P.t[blockIdx.x];
  const int m0 = blockIdx.y * GM;
  const int n_mma = (T.ncols + 15) & ~15;
  const int n_box = (n_mma + 63) >> 6;
  const int nkb = (T.d_in + GK - 1) / GK;
  const CUtensorMap* mx = T.src ? &map_xv : &map_xk;
  const CUtensorMap* mw = T.src ? &map_wv : &map_wk;

  if (tid == 0) {
    for (int s = 0; s < n_st; ++s) { mbar_init(full0 + 8 * s, 1); mbar_init(empty0 + 8 * s, 1); }
    mbar_init(accbar, 1);
    fence_barrier_init();
  }
  if (warp == 1) tmem_alloc(smem_u32(&tmem_slot), (uint32_t)P.tmem_cols);
  if (FUSED)
    for (int i = tid; i < P.n_seg_max * GM; i += G_THREADS) amax_tab[i] = 0u;
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  const uint32_t tmem_d = tmem_slot;

  if (warp == 0) {
    if (elect_one()) {
      const uint32_t bytes = (uint32_t)(GA_BYTES + n_box * GB_BOX);
      int s = 0, u = 0;   // stage, use count of the stage
      for (int kb = 0; kb < nkb; ++kb) {
        if (u > 0) mbar_wait(empty0 + 8 * s, (uint32_t)((u - 1) & 1));
        const uint32_t sa = sbase + s * stage_bytes, sb = sa + GA_BYTES;
        mbar_expect_tx(full0 + 8 * s, bytes);
        tma_load_2d(sa, mx, T.x_col0 + kb * GK, m0, full0 + 8 * s);
        for (int j = 0; j < n_box; ++j) tma_load_2d(sb + j * GB_BOX, mw, T.w_col0 + 64 * j, kb * GK, full0 + 8 * s);
        if (++s == n_st) { s = 0; ++u; }
      }
    }
    __syncwarp();
  } else if (warp == 1) {
    // instruction descriptors: D fp32, A and B fp16, A K-major, B MN-major, M = 128
    const int n0 = n_mma < 256 ? n_mma : 256, n1 = n_mma - n0;
    const uint32_t idesc0 = umma_idesc_f16(n0, true), idesc1 = umma_idesc_f16(n1 > 0 ? n1 : 16, true);
    int s = 0, u = 0;
    for (int kb = 0; kb < nkb; ++kb) {
      mbar_wait(full0 + 8 * s, (uint32_t)(u & 1));
      tc_fence_after();
      if (elect_one()) {
        const uint32_t sa = sbase + s * stage_bytes, sb = sa + GA_BYTES;
#pragma unroll
        for (int k = 0; k < GK / 16; ++k) {
          // X tile, K-major: 8-row groups 1024 bytes apart (SBO); 16 k = 32 bytes inside the swizzle atom
          const uint64_t da = desc_sw128(sa + k * 32, 16, 1024);
          // factor tile, MN-major: 64-column atoms 8 KB apart (LBO), 8-k-row groups 1024 bytes apart (SBO); 16 k = 2 groups
          const uint64_t db = desc_sw128(sb + k * 2048, GB_BOX, 1024);
          const uint32_t acc = (kb > 0 || k > 0) ? 1u : 0u;
          umma_ss_f16(tmem_d, da, db, idesc0, acc);
          if (n1 > 0) umma_ss_f16(tmem_d + 256, da, desc_sw128(sb + 4 * GB_BOX + k * 2048, GB_BOX, 1024), idesc1, acc);
        }
        umma_commit(empty0 + 8 * s);
        if (kb == nkb - 1) umma_commit(accbar);
      }
      __syncwarp();
      if (++s == n_st) { s = 0; ++u; }
    }
  } else {
    // epilogue: warp w may read TMEM lanes [32 (w % 4), +32) = token rows; GE warps per quarter share the columns
    const int q = warp & 3, e = (warp - 2) >> 2;
    const int rl = q * 32 + lane;
    const int row = m0 + rl;
    const uint32_t tl = tmem_d + ((uint32_t)(q * 32) << 16);
    if (!FUSED) {
      mbar_wait(accbar, 0);
      tc_fence_after();
      __half* dst = z + (size_t)row * P.R + T.w_col0 + (T.src ? L.sum_rank_k : 0);
      for (int cb = 8 * e; cb < T.ncols; cb += 8 * GE) {   // ncols is a multiple of 8
        __half h[8];
        ld8_h(tl + cb, h);
        if (row < P.n_new) *reinterpret_cast<uint4*>(dst + cb) = *reinterpret_cast<const uint4*>(h);
      }
    } else {
      // the token's page and slot (looked up while the main loop runs)
      const int Pt = L.page_tokens;
      uint8_t* pg = nullptr;
      int slot = 0;
      if (row < P.n_new) {
        const int pos = P.positions[row], sid = P.seq_ids[row];
        if (pos >= 0 && pos / Pt < P.max_pages && sid >= 0) {   // caller error otherwise: skip the token, never write wildly
          const int pidx = P.table[(size_t)sid * P.max_pages + pos / Pt];
          if (pidx >= 0) { pg = P.pool + (size_t)pidx * L.page_bytes; slot = pos % Pt; }
        }
      }
      const bool quant = L.bits_hi != 16;
      const int nseg = T.src ? 1 : (quant ? 2 * T.nh : T.nh);
      // two 4-bit slots of a value row share a byte: the lanes of a pair (2i, 2i+1) write it together when they are the
      // two slots of one byte
      const unsigned long long me = pg ? (unsigned long long)(uintptr_t)pg : ~0ull;
      const unsigned long long other = __shfl_xor_sync(0xffffffffu, me, 1);
      const int oslot = __shfl_xor_sync(0xffffffffu, slot, 1);
      const bool paired = pg && other == me && oslot == (slot ^ 1);
      mbar_wait(accbar, 0);
      tc_fence_after();
      if (quant) {   // pass 1: per-token absmax of every segment (after the single rounding to fp16)
        for (int i = 0; i < nseg; ++i) {
          const Seg sg = seg_of(L, T, i);
          float amax = 0.f;
          for (int c = 8 * e; c < sg.n; c += 8 * GE) {
            __half h[8];
            ld8_h(tl + sg.c0 + c, h);
#pragma unroll
            for (int k = 0; k < 8; ++k) amax = fmaxf(amax, fabsf(__half2float(h[k])));
          }
          if (8 * e < sg.n) atomicMax(amax_tab + i * GM + rl, __float_as_uint(amax));
        }
        bar_sync(1, G_EPI_THREADS);
      }
      for (int i = 0; i < nseg; ++i) {   // pass 2: scales, codes, stores
        const Seg sg = seg_of(L, T, i);
        float sf = 0.f;
        if (quant) {
          const __half s16 = sg.n ? sk_scale_of(__uint_as_float(amax_tab[i * GM + rl]), sk_qmax(sg.bits)) : __float2half(0.f);
          sf = __half2float(s16);
          if (pg && e == i % GE) {
            uint16_t* sc = T.src ? reinterpret_cast<uint16_t*>(pg + L.v_scale_off) + sg.blk * Pt + slot
                                 : reinterpret_cast<uint16_t*>(pg + L.k_scale_off) + (sg.h * 2 + sg.blk) * Pt + slot;
            *sc = sk_half_bits(s16);
          }
        }
        uint8_t* dstp = nullptr;
        if (pg) {
          if (T.src) dstp = pg + (sg.blk ? L.v_lo_off : L.v_hi_off);
          else dstp = pg + (sg.blk ? L.k_lo_off[sg.h] : L.k_hi_off[sg.h]) + (size_t)slot * (sg.n * sg.bits / 8);
        }
        for (int c = 8 * e; c < sg.n; c += 8 * GE) {
          __half h[8];
          ld8_h(tl + sg.c0 + c, h);
          if (T.src) value_chunk(h, c, sg.bits, sf, Pt, dstp, slot, paired);
          else key_chunk(h, c, sg.bits, sf, dstp);
        }
      }
    }
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) tmem_dealloc(tmem_d, (uint32_t)P.tmem_cols);
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

EncodeTiledFn encode_fn() {
  static EncodeTiledFn fn = nullptr;   // (process-wide: the driver entry point does not depend on the device)
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
      fn = (EncodeTiledFn)p;
    else
      cudaGetLastError();
  }
  return fn;
}

// fp16 matrix [rows][cols] with `ld` elements between rows; box = 64 columns x box_rows
bool make_map(CUtensorMap* m, const void* base, uint64_t cols, uint64_t rows, uint64_t ld, uint32_t box_rows) {
  EncodeTiledFn fn = encode_fn();
  if (!fn) return false;
  const cuuint64_t dim[2] = {cols, rows};
  const cuuint64_t stride[1] = {ld * 2};
  const cuuint32_t box[2] = {64, box_rows};
  const cuuint32_t es[2] = {1, 1};
  return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT16, 2, const_cast<void*>(base), dim, stride, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace

// 2 = launched with the quantiser and the paged write fused (nothing else to do), 1 = launched, z holds fp16(X . A),
// 0 = this call is not covered (alignment, tile count, no driver entry point): the caller falls back
int sk_append_gemm(starkv_ctx* ctx, void* pool, const int32_t* table, int max_pages, const int32_t* seq_ids,
                   const int32_t* positions, int n_new, const void* k_new, int64_t k_row_stride, int64_t k_head_stride, int d_in_k,
                   const void* v_new, int64_t v_row_stride, int d_in_v, const void* A_k, const void* A_v, void* z) {
  const StarkvLayout& L = ctx->L;
  if (n_new < 64) return 0;
  if ((k_row_stride & 7) || (v_row_stride & 7) || (k_head_stride & 7) || (L.sum_rank_k & 7) || (L.rank_v & 7)) return 0;
  if (((uintptr_t)k_new | (uintptr_t)v_new | (uintptr_t)A_k | (uintptr_t)A_v | (uintptr_t)z) & 15) return 0;
  if (k_head_stride < 0 || k_row_stride <= 0 || v_row_stride <= 0) return 0;
  const bool fused = L.v_hi_n <= 512 && L.v_lo_n <= 512;   // a value block is one tile: its columns fit the tensor memory
  GemmPlan P;
  memset(&P, 0, sizeof(P));
  P.n_new = n_new;
  P.R = L.sum_rank_k + L.rank_v;
  P.seq_ids = seq_ids; P.positions = positions; P.table = table; P.max_pages = max_pages; P.pool = (uint8_t*)pool;
  int nt = 0, widest = 0;
  auto push = [&](int src, int h0, int nh, int ncols, int x_col0, int w_col0, int d_in) {
    if (nt >= G_MAX_TILES) return false;
    P.t[nt++] = GemmTile{(int16_t)src, (int16_t)h0, (int16_t)nh, (int16_t)ncols, x_col0, w_col0, d_in};
    widest = ncols > widest ? ncols : widest;
    return true;
  };
  // value tiles first (the longest K loops start first): one per precision block when fused, else 256 columns at a time
  int n_seg_max = 1;
  if (fused) {
    if (!push(1, 0, 0, L.v_hi_n, 0, 0, d_in_v)) return 0;
    if (L.v_lo_n > 0 && !push(1, 1, 0, L.v_lo_n, 0, L.v_hi_n, d_in_v)) return 0;
  } else {
    for (int c0 = 0; c0 < L.rank_v; c0 += 256)
      if (!push(1, 0, 0, L.rank_v - c0 < 256 ? L.rank_v - c0 : 256, 0, c0, d_in_v)) return 0;
  }
  // key tiles: whole heads (rank_k <= head_dim <= 256), several per tile where the heads share X (hidden-state mode)
  for (int h = 0; h < L.n_kv_heads;) {
    int nh = 1, cols = L.rank_k[h];
    if (k_head_stride == 0)
      while (h + nh < L.n_kv_heads && cols + L.rank_k[h + nh] <= 256) cols += L.rank_k[h + nh++];
    if (!push(0, h, nh, cols, (int)(h * k_head_stride), L.koff[h], d_in_k)) return 0;
    n_seg_max = 2 * nh > n_seg_max ? 2 * nh : n_seg_max;
    h += nh;
  }
  P.n_tiles = nt;
  const int n_box_max = (((widest + 15) & ~15) + 63) >> 6;
  P.stage_bytes = GA_BYTES + n_box_max * GB_BOX;
  P.tmem_cols = widest > 256 ? 512 : 256;
  P.n_seg_max = fused ? n_seg_max : 0;
  const int tab_bytes = P.n_seg_max * GM * 4;
  const int room = ctx->smem_optin - 1024 /* alignment slack */ - 256 /* barriers */ - 64 /* static */ - tab_bytes;
  P.n_stages = room / P.stage_bytes;
  if (P.n_stages > 6) P.n_stages = 6;
  if (P.n_stages < 2) return 0;
  const int smem = P.n_stages * P.stage_bytes + 1024 + 256 + tab_bytes;
  const uint64_t xk_cols = (uint64_t)(k_head_stride ? (L.n_kv_heads - 1) * k_head_stride + d_in_k : d_in_k);
  if (xk_cols > (uint64_t)k_row_stride || (uint64_t)d_in_v > (uint64_t)v_row_stride) return 0;
  CUtensorMap mxk, mxv, mwk, mwv;
  if (!make_map(&mxk, k_new, xk_cols, (uint64_t)n_new, (uint64_t)k_row_stride, GM) ||
      !make_map(&mxv, v_new, (uint64_t)d_in_v, (uint64_t)n_new, (uint64_t)v_row_stride, GM) ||
      !make_map(&mwk, A_k, (uint64_t)L.sum_rank_k, (uint64_t)d_in_k, (uint64_t)L.sum_rank_k, GK) ||
      !make_map(&mwv, A_v, (uint64_t)L.rank_v, (uint64_t)d_in_v, (uint64_t)L.rank_v, GK))
    return 0;
  const dim3 grid(nt, (n_new + GM - 1) / GM);
  if (fused) {
    if (sk_need_smem(ctx, append_gemm_kernel<true>, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    append_gemm_kernel<true><<<grid, G_THREADS, smem, ctx->stream>>>(L, P, mxk, mxv, mwk, mwv, (__half*)z);
  } else {
    if (sk_need_smem(ctx, append_gemm_kernel<false>, smem) != cudaSuccess) { cudaGetLastError(); return 0; }
    append_gemm_kernel<false><<<grid, G_THREADS, smem, ctx->stream>>>(L, P, mxk, mxv, mwk, mwv, (__half*)z);
  }
  if (cudaGetLastError() != cudaSuccess) return 0;
  ctx->last_append = "append_gemm_kernel";
  return fused ? 2 : 1;
}
