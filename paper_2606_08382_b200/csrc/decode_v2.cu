// Tensor-core decode attention over the latent cache (rows D1-D7 of the hot path), sm_100a.
//
//   PAPER.md §3.3: scores in latent space  s_t = q~ . L_k[t],  q~ = sm_scale q B_k^T  (no RoPE on
//   this path, A1), and the value side reordered as (p L_v) B_v  ("(p V') U_V").
//   PAPER.md A.6 L627: stack p over heads so that p L_v is ONE GEMM  P[H_q x T] . L_v[T x r_v]  -> tensor cores.
//   PAPER.md Eq.12 L208 / A.6 L625: latents are dequantised in registers, never materialised.
//
// One CTA (8 warps) walks a contiguous page range of one sequence (split-K), one 64-token page per
// iteration, ONE block barrier per page.  Pages arrive in a shared-memory ring by cp.async.bulk +
// mbarrier (a page is one contiguous byte range by construction of the format).  Per page:
//   QK       warp w scores "quad" w (4 query heads) against all 64 tokens on mma.sync m16n8k16:
//            S^T[tokens x (head, hi/lo)] = L_k[tokens x ch] . q~^T.  The latent query is an fp16 hi+lo pair in
//            two MMA columns per head, so hi+lo meets in one thread and the score keeps fp32 accuracy;
//            int4/int8 fields go to fp16 by the magic-number lop3/prmt trick (exact); per-token scales
//            multiply the fp32 sums.  With G < 4 several KV heads feed one quad (zero columns elsewhere).
//   softmax  in registers: page maximum by 3 shuffles, running (m, l) per thread, P -> fp16 with a 2^8
//            offset; an 8x8 movmatrix transpose turns the accumulator layout into the B fragments of the PV
//            product, which go to a double-buffered 4 KB exchange area (the only cross-warp traffic).
//   PV       after the barrier, warp w owns value channels [16(w+8a), +16): O^T[ch x heads] += L_v^T[ch x tok] . P^T,
//            L_v channel-major so that a 32-bit word holds consecutive tokens of one channel = the A
//            fragment's k pairs; value scales are applied element-wise in fp16 (c*s, one rounding).
//   The row of the QK tile that holds token t is chosen so that the transposed P lands in the token order
//   the dequantised value words produce (no shuffles on the value side).
// The partial (m, l, acc[H_q x r_v]) goes to the workspace; combine_kernel merges and up-projects.
#include <string.h>

#include "decode_common.cuh"
#include "decode_v2.h"

namespace {

constexpr int NWARPS = 8;
constexpr int NTHREADS = NWARPS * 32;
constexpr int PTOK = 64;         // tokens per page on this path
constexpr float P_OFFSET = 8.f;  // P is stored as 2^(s - m + 8) in fp16 (keeps small weights normal)
constexpr float kLog2e = 1.4426950408889634f;
constexpr int P_BUF_BYTES = 2 * 4 * 32 * 16;   // [k-step pair][n-tile][lane] uint4

// ---- PTX wrappers ---------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(bar),
      "r"(parity)
      : "memory");
}
// 1-D bulk copy global -> shared, completion counted on an mbarrier (SASS: UBLKCP)
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
               "l"(src), "r"(bytes), "r"(bar)
               : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }

__device__ __forceinline__ void mma16816(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                         uint32_t b1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
      : "+f"(d[0]), "+f"(d[1]), "+f"(d[2]), "+f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
// 8x8 b16 transpose across the warp: lane (R, j) holds M[R][2j..2j+1] and receives M[2j..2j+1][R]
__device__ __forceinline__ uint32_t movmatrix_trans(uint32_t x) {
  uint32_t r;
  asm volatile("movmatrix.sync.aligned.m8n8.trans.b16 %0, %1;" : "=r"(r) : "r"(x));
  return r;
}
__device__ __forceinline__ uint32_t lop3_and_or(uint32_t x, uint32_t m, uint32_t o) {
  uint32_t r;
  asm("lop3.b32 %0, %1, %2, %3, 0xea;" : "=r"(r) : "r"(x), "r"(m), "r"(o));  // (x & m) | o
  return r;
}
__device__ __forceinline__ uint32_t prmt(uint32_t a, uint32_t b, uint32_t sel) {
  uint32_t r;
  asm("prmt.b32 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(sel));
  return r;
}
__device__ __forceinline__ uint32_t h2sub(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("sub.f16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t h2mul(uint32_t a, uint32_t b) {
  uint32_t r;
  asm("mul.f16x2 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(b));
  return r;
}
__device__ __forceinline__ uint32_t h2fma(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t r;
  asm("fma.rn.f16x2 %0, %1, %2, %3;" : "=r"(r) : "r"(a), "r"(b), "r"(c));
  return r;
}
__device__ __forceinline__ uint32_t pack_h2(float lo, float hi) {
  uint32_t r;
  asm("cvt.rn.f16x2.f32 %0, %1, %2;" : "=r"(r) : "f"(hi), "f"(lo));  // first source -> upper half
  return r;
}
__device__ __forceinline__ float2 h2_to_f2(uint32_t h) {
  return __half22float2(*reinterpret_cast<const __half2*>(&h));
}

// ---- exact integer field -> fp16 (DESIGN.md format v1: offset-binary fields) ------------------
// int8 word (4 fields b0..b3) -> (c0,c1), (c2,c3)
__device__ __forceinline__ void deq8_pairs(uint32_t w, uint32_t& p01, uint32_t& p23) {
  p01 = h2sub(prmt(w, 0x64646464u, 0x4140u), 0x64806480u);  // 1024+u - 1152
  p23 = h2sub(prmt(w, 0x64646464u, 0x4342u), 0x64806480u);
}
// int4 word (8 fields n0..n7) -> (c0,c4), (c1,c5), (c2,c6), (c3,c7)
__device__ __forceinline__ void deq4_pairs(uint32_t w, uint32_t (&h)[4]) {
  const uint32_t w2 = w >> 8;
  h[0] = h2sub(lop3_and_or(w, 0x000f000fu, 0x64006400u), 0x64086408u);                 // 1024+u - 1032
  h[1] = h2fma(lop3_and_or(w, 0x00f000f0u, 0x64006400u), 0x2c002c00u, 0xd480d480u);    // (1024+16u)/16 - 72
  h[2] = h2sub(lop3_and_or(w2, 0x000f000fu, 0x64006400u), 0x64086408u);
  h[3] = h2fma(lop3_and_or(w2, 0x00f000f0u, 0x64006400u), 0x2c002c00u, 0xd480d480u);
}

// ---------------------------------------------------------------------------------------------
// D1: latent-space query image.  q~ = sm_scale * log2e * q B_k^T in fp32, split into an fp16 hi+lo pair
// and laid out as the B fragments of the QK MMAs (see V2Plan).  grid (H_kv, batch), 128 threads.
// KV head g's G query heads sit in columns 2*((g*G + i) mod 4) + {hi, lo}; the other columns are zero.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(128) qproj_kernel(const __grid_constant__ StarkvLayout L,
                                                    const __grid_constant__ V2Plan PL,
                                                    const __half* __restrict__ q, const __half* __restrict__ B_k,
                                                    uint32_t* __restrict__ qimg_all, size_t qimg_stride_words) {
  __shared__ float qs[4][256];   // the G (<= 4) query rows of this KV head
  __shared__ float qt[4][256];   // q~[i][ch]
  const int g = blockIdx.x, b = blockIdx.y;
  const int G = L.group, dh = L.head_dim, r = L.rank_k[g];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  for (int i = tid; i < 4 * dh; i += 128) {
    const int h = i / dh, d = i % dh;
    qs[h][d] = h < G ? __half2float(q[((size_t)b * L.n_q_heads + g * G + h) * dh + d]) : 0.f;
  }
  __syncthreads();
  for (int ch = warp; ch < r; ch += 4) {
    const __half* brow = B_k + (size_t)(L.koff[g] + ch) * dh;
    float a[4] = {0.f, 0.f, 0.f, 0.f};
    for (int d = lane; d < dh; d += 32) {
      const float bv = __half2float(brow[d]);
#pragma unroll
      for (int i = 0; i < 4; ++i) a[i] = fmaf(qs[i][d], bv, a[i]);
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
#pragma unroll
      for (int o = 16; o; o >>= 1) a[i] += __shfl_xor_sync(0xffffffffu, a[i], o);
    }
    if (lane == 0) {
#pragma unroll
      for (int i = 0; i < 4; ++i) qt[i][ch] = a[i] * (L.sm_scale * kLog2e);
    }
  }
  __syncthreads();
  const int n_hi = L.k_hi_n[g], n_lo = L.k_lo_n[g];
  const int mh = L.bits_hi == 4 ? 2 * ((n_hi + 31) >> 5) : (n_hi + 15) >> 4;
  const int s0 = PL.qstep_begin[g], steps = PL.qstep_begin[g + 1] - s0;
  uint32_t* dst = qimg_all + (size_t)b * qimg_stride_words + (size_t)s0 * 64;
  for (int wi = tid; wi < steps * 64; wi += 128) {
    const int reg = wi & 1, ln = (wi >> 1) & 31;
    int local = wi >> 6;
    int blk = 0;
    if (local >= mh) { blk = 1; local -= mh; }
    const int bits = blk ? L.bits_lo : L.bits_hi;
    const int n = blk ? n_lo : n_hi;
    const int chunk = bits == 4 ? local >> 1 : local, m = bits == 4 ? local & 1 : 0;
    const int col = ln >> 2, j = ln & 3;
    const int i = (col >> 1) - ((g * G) & 3), hilo = col & 1;
    uint32_t word = 0;
    if (i >= 0 && i < G) {
#pragma unroll
      for (int e = 0; e < 2; ++e) {
        const int k = 2 * j + e + 8 * reg;
        const int ch = chunk * (bits == 4 ? 32 : 16) + v2_k_to_channel(bits, m, k);
        if (ch >= n) continue;
        const float a = qt[i][(blk ? n_hi : 0) + ch];
        const __half hi = __float2half_rn(a);
        const __half v = hilo ? __float2half_rn(a - __half2float(hi)) : hi;
        word |= (uint32_t)__half_as_ushort(v) << (16 * e);
      }
    }
    dst[wi] = word;
  }
}

// ---------------------------------------------------------------------------------------------
// QK of one precision block of one KV head for the warp's 64 tokens (4 m-tiles of 16 rows).
// Row r of m-tile s holds token  tb(r & 7) + s*TS + 8*(r >> 3)  with tb / TS chosen per mode so that the
// movmatrix transpose of P yields the k order of the PV A fragments (see the header comment):
//   quantised: tb(R) = 16(R>>1) + 4(R&1), TS = 1     fp16: tb(R) = 16(R>>1) + (R&1), TS = 2
// ---------------------------------------------------------------------------------------------
template <bool QUANT>
__device__ __forceinline__ int tok_base(int R) { return QUANT ? 16 * (R >> 1) + 4 * (R & 1) : 16 * (R >> 1) + (R & 1); }

template <bool QUANT>
__device__ __forceinline__ void qk_block(float (&acc)[4][4], const uint8_t* __restrict__ pg, int block_off, int n, int bits,
                                         const uint2* __restrict__ qimg_lane, int& step, int R, int j) {
  constexpr int TS = QUANT ? 1 : 2;
  const int tb = tok_base<QUANT>(R);
  if (!QUANT) {
    const int rowbytes = 2 * n;
    const uint8_t* r0 = pg + block_off + tb * rowbytes + 8 * j;
    const int nchunks = (n + 15) >> 4;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf = qimg_lane[step * 32];
      ++step;
      const bool valid = c * 16 + 4 * j < n;
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const uint8_t* p = r0 + (s * TS) * rowbytes + c * 32;
        uint2 x0 = make_uint2(0, 0), x1 = make_uint2(0, 0);
        if (valid) {
          x0 = *reinterpret_cast<const uint2*>(p);
          x1 = *reinterpret_cast<const uint2*>(p + 8 * rowbytes);
        }
        mma16816(acc[s], x0.x, x1.x, x0.y, x1.y, bf.x, bf.y);
      }
    }
  } else if (bits == 8) {
    const int rowbytes = n;
    const uint8_t* r0 = pg + block_off + tb * rowbytes + 4 * j;
    const int nchunks = (n + 15) >> 4;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf = qimg_lane[step * 32];
      ++step;
      const bool valid = c * 16 + 4 * j < n;
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const uint8_t* p = r0 + s * rowbytes + c * 16;
        const uint32_t w0 = valid ? *reinterpret_cast<const uint32_t*>(p) : 0x80808080u;
        const uint32_t w1 = valid ? *reinterpret_cast<const uint32_t*>(p + 8 * rowbytes) : 0x80808080u;
        uint32_t a0, a1, a2, a3;
        deq8_pairs(w0, a0, a2);
        deq8_pairs(w1, a1, a3);
        mma16816(acc[s], a0, a1, a2, a3, bf.x, bf.y);
      }
    }
  } else {
    const int rowbytes = n >> 1;
    const uint8_t* r0 = pg + block_off + tb * rowbytes + 4 * j;
    const int nchunks = (n + 31) >> 5;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf0 = qimg_lane[step * 32];
      const uint2 bf1 = qimg_lane[(step + 1) * 32];
      step += 2;
      const bool valid = c * 32 + 8 * j < n;
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        const uint8_t* p = r0 + s * rowbytes + c * 16;
        const uint32_t w0 = valid ? *reinterpret_cast<const uint32_t*>(p) : 0x88888888u;
        const uint32_t w1 = valid ? *reinterpret_cast<const uint32_t*>(p + 8 * rowbytes) : 0x88888888u;
        uint32_t h0[4], h1[4];
        deq4_pairs(w0, h0);
        deq4_pairs(w1, h1);
        mma16816(acc[s], h0[0], h1[0], h0[1], h1[1], bf0.x, bf0.y);
        mma16816(acc[s], h0[2], h1[2], h0[3], h1[3], bf1.x, bf1.y);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// PV of one 16-channel m-tile over the page's 64 tokens (4 k-steps) against all NT head tiles.
//   vrow0/vrow1: this thread's two channel rows (R, R+8) of the value block, already clamped
//   sc0/sc2    : value scales as (t, t+4) fp16 pairs of this thread's 16 tokens (quantised modes)
//   pf         : P^T B fragments  [k-step pair][head tile] = (b0, b1 of step 2sp, b0, b1 of step 2sp+1)
// ---------------------------------------------------------------------------------------------
template <bool QUANT, int NT>
__device__ __forceinline__ void pv_tile(float (&acc)[NT][4], const uint8_t* __restrict__ vrow0,
                                        const uint8_t* __restrict__ vrow1, int bits, bool dead0, bool dead1,
                                        const uint32_t (&sc0)[4], const uint32_t (&sc2)[4], const uint4 (&pf)[2][NT],
                                        int j) {
  uint32_t A0[4], A1[4], A2[4], A3[4];
  if (QUANT) {
    if (bits == 4) {
      const uint2 x0 = *reinterpret_cast<const uint2*>(vrow0 + 8 * j);
      const uint2 x1 = *reinterpret_cast<const uint2*>(vrow1 + 8 * j);
      uint32_t h[4];
      deq4_pairs(x0.x, h);
#pragma unroll
      for (int s = 0; s < 4; ++s) A0[s] = h2mul(h[s], sc0[s]);
      deq4_pairs(x0.y, h);
#pragma unroll
      for (int s = 0; s < 4; ++s) A2[s] = h2mul(h[s], sc2[s]);
      deq4_pairs(x1.x, h);
#pragma unroll
      for (int s = 0; s < 4; ++s) A1[s] = h2mul(h[s], sc0[s]);
      deq4_pairs(x1.y, h);
#pragma unroll
      for (int s = 0; s < 4; ++s) A3[s] = h2mul(h[s], sc2[s]);
    } else {
      const uint4 x0 = *reinterpret_cast<const uint4*>(vrow0 + 16 * j);
      const uint4 x1 = *reinterpret_cast<const uint4*>(vrow1 + 16 * j);
      auto deq8v = [&](uint32_t wa, uint32_t wb, const uint32_t (&sc)[4], uint32_t (&out)[4]) {
        const uint32_t ta = prmt(wa, wb, 0x5140u), tb = prmt(wa, wb, 0x7362u);   // (t0,t4,t1,t5), (t2,t6,t3,t7)
        out[0] = h2mul(h2sub(prmt(ta, 0x64646464u, 0x4140u), 0x64806480u), sc[0]);
        out[1] = h2mul(h2sub(prmt(ta, 0x64646464u, 0x4342u), 0x64806480u), sc[1]);
        out[2] = h2mul(h2sub(prmt(tb, 0x64646464u, 0x4140u), 0x64806480u), sc[2]);
        out[3] = h2mul(h2sub(prmt(tb, 0x64646464u, 0x4342u), 0x64806480u), sc[3]);
      };
      deq8v(x0.x, x0.y, sc0, A0);
      deq8v(x0.z, x0.w, sc2, A2);
      deq8v(x1.x, x1.y, sc0, A1);
      deq8v(x1.z, x1.w, sc2, A3);
    }
  } else {
    const uint4* r0 = reinterpret_cast<const uint4*>(vrow0 + 32 * j);
    const uint4* r1 = reinterpret_cast<const uint4*>(vrow1 + 32 * j);
    const uint4 x0 = r0[0], y0 = r0[1], x1 = r1[0], y1 = r1[1];
    A0[0] = x0.x; A0[1] = x0.y; A0[2] = x0.z; A0[3] = x0.w;
    A2[0] = y0.x; A2[1] = y0.y; A2[2] = y0.z; A2[3] = y0.w;
    A1[0] = x1.x; A1[1] = x1.y; A1[2] = x1.z; A1[3] = x1.w;
    A3[0] = y1.x; A3[1] = y1.y; A3[2] = y1.z; A3[3] = y1.w;
  }
  if (dead0 || dead1) {   // ragged last tile of a block: rows past the block contribute nothing
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      if (dead0) { A0[s] = 0; A2[s] = 0; }
      if (dead1) { A1[s] = 0; A3[s] = 0; }
    }
  }
#pragma unroll
  for (int s = 0; s < 4; ++s)
#pragma unroll
    for (int c = 0; c < NT; ++c) {
      const uint4 f = pf[s >> 1][c];
      mma16816(acc[c], A0[s], A1[s], A2[s], A3[s], (s & 1) ? f.z : f.x, (s & 1) ? f.w : f.y);
    }
}

// ---------------------------------------------------------------------------------------------
// Main kernel.  grid (n_splits, batch), 256 threads.
//   QUANT  integer latents (else fp16)   NT  head tiles of 8   MT  value m-tiles (16 channels) per warp
// ---------------------------------------------------------------------------------------------
template <bool QUANT, int NT, int MT, int MINB>
__global__ void __launch_bounds__(NTHREADS, MINB) decode_v2_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ V2Plan PL, const uint8_t* __restrict__ pool,
    const int32_t* __restrict__ table, int max_pages, const int32_t* __restrict__ seq_lens,
    const uint8_t* __restrict__ qimg_all, size_t qimg_stride, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int TS = QUANT ? 1 : 2;

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int j = lane & 3, R = lane >> 2;
  const int split = blockIdx.x, b = blockIdx.y;
  const int len = seq_lens[b];
  const int n_pages = (len + PTOK - 1) / PTOK;
  int p0, p1;
  sk_split_range(n_pages, n_splits, 1, split, &p0, &p1);
  const int n_it = p1 - p0;
  const size_t pstride = sk_part_stride(L.rank_v);
  float* my_parts = parts + ((size_t)b * n_splits + split) * L.n_q_heads * pstride;

  if (n_it <= 0) {   // empty range: neutral partial
    for (int i = tid; i < L.n_q_heads * (int)pstride; i += NTHREADS) {
      const int c = i % (int)pstride;
      my_parts[i] = c == 0 ? -INFINITY : 0.f;
    }
    return;
  }

  uint8_t* stage_base = smem + PL.off_stage;
  const uint2* qimg_lane = reinterpret_cast<const uint2*>(smem + PL.off_qimg) + lane;
  uint8_t* Pm = smem + PL.off_p;                                       // [2][P_BUF_BYTES]
  float* alpha_s = reinterpret_cast<float*>(smem + PL.off_alpha);      // [2][32]
  const uint32_t bar0 = smem_u32(smem + PL.off_bar);                   // full[nstage], then qbar
  const uint32_t qbar = bar0 + 8 * PL.nstage;
  const int32_t* my_table = table + (size_t)b * max_pages;
  const int nstage = PL.nstage;
  const uint32_t page_bytes = (uint32_t)L.page_bytes;

  auto issue = [&](int it) {   // thread 0 only
    const int st = it % nstage;
    const uint32_t bar = bar0 + 8 * st;
    mbar_expect_tx(bar, page_bytes);
    bulk_g2s(smem_u32(stage_base + (size_t)st * page_bytes), pool + (size_t)my_table[p0 + it] * page_bytes, page_bytes, bar);
  };

  if (tid == 0) {
    for (int s = 0; s < nstage; ++s) mbar_init(bar0 + 8 * s, 1);
    mbar_init(qbar, 1);
    fence_barrier_init();
    mbar_expect_tx(qbar, (uint32_t)PL.qimg_bytes);
    bulk_g2s(smem_u32(smem + PL.off_qimg), qimg_all + (size_t)b * qimg_stride, (uint32_t)PL.qimg_bytes, qbar);
    for (int it = 0; it < min(nstage, n_it); ++it) issue(it);
  }
  for (int i = tid; i < 2 * P_BUF_BYTES / 16; i += NTHREADS) reinterpret_cast<uint4*>(Pm)[i] = make_uint4(0, 0, 0, 0);
  if (tid < 64) alpha_s[tid] = 1.f;
  __syncthreads();

  // this warp's quad (QK + softmax) and where its transposed P words go
  const bool has_quad = warp < PL.nq;
  const int kv0 = warp * PL.kv_per_quad;
  const int kv1 = min(kv0 + PL.kv_per_quad, L.n_kv_heads);
  const int tb = tok_base<QUANT>(R);
  // after the transpose lane (R' = 2j'' + e', j) holds the b-register of head j'' for k-step 2u + e';
  // its consumer is lane (4*(quad&1) + j'', j) of head tile quad>>1
  const int p_thr_off = (((warp >> 1) * 32 + (4 * (warp & 1) + (R >> 1)) * 4 + j) << 4) + ((R & 1) << 3);
  float m_run = -INFINITY, l_run = 0.f;

  float acc[MT][NT][4];
#pragma unroll
  for (int a = 0; a < MT; ++a)
#pragma unroll
    for (int c = 0; c < NT; ++c)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[a][c][e] = 0.f;

  mbar_wait(qbar, 0);

  for (int it = 0; it < n_it; ++it) {
    const int st = it % nstage;
    uint8_t* pg = stage_base + (size_t)st * page_bytes;
    const int tok0 = (p0 + it) * PTOK;
    mbar_wait(bar0 + 8 * st, (uint32_t)((it / nstage) & 1));
    const int nvalid = len - tok0;          // >= 1
    const bool tail = nvalid < PTOK;
    uint8_t* Pb = Pm + (it & 1) * P_BUF_BYTES;
    float* al = alpha_s + (it & 1) * 32;

    if (tail) {   // neutralise value data of slots past the sequence end (they may hold any bits);
                  // ordered before the PV reads by the page barrier below
      if (QUANT) {
        if (tid < 2 * PTOK && (tid & (PTOK - 1)) >= nvalid) reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[tid] = 0;
      } else {
        const int nbad = PTOK - nvalid;
        for (int i = tid; i < L.rank_v * nbad; i += NTHREADS)
          reinterpret_cast<uint16_t*>(pg + L.v_hi_off)[(i / nbad) * PTOK + nvalid + i % nbad] = 0;
      }
    }

    // ================= QK + softmax for this warp's quad =================
    if (has_quad) {
      float sc[4][2];
#pragma unroll
      for (int s = 0; s < 4; ++s) sc[s][0] = sc[s][1] = 0.f;
      for (int g = kv0; g < kv1; ++g) {
        float chi[4][4];
#pragma unroll
        for (int s = 0; s < 4; ++s)
#pragma unroll
          for (int e = 0; e < 4; ++e) chi[s][e] = 0.f;
        int step = PL.qstep_begin[g];
        qk_block<QUANT>(chi, pg, L.k_hi_off[g], L.k_hi_n[g], L.bits_hi, qimg_lane, step, R, j);
        if (QUANT) {
          const __half* ksc = reinterpret_cast<const __half*>(pg + L.k_scale_off) + (g * 2) * PTOK + tb;
          {
            const uint2 h0 = *reinterpret_cast<const uint2*>(ksc), h1 = *reinterpret_cast<const uint2*>(ksc + 8);
            const float2 a01 = h2_to_f2(h0.x), a23 = h2_to_f2(h0.y), b01 = h2_to_f2(h1.x), b23 = h2_to_f2(h1.y);
            sc[0][0] = fmaf(chi[0][0] + chi[0][1], a01.x, sc[0][0]); sc[0][1] = fmaf(chi[0][2] + chi[0][3], b01.x, sc[0][1]);
            sc[1][0] = fmaf(chi[1][0] + chi[1][1], a01.y, sc[1][0]); sc[1][1] = fmaf(chi[1][2] + chi[1][3], b01.y, sc[1][1]);
            sc[2][0] = fmaf(chi[2][0] + chi[2][1], a23.x, sc[2][0]); sc[2][1] = fmaf(chi[2][2] + chi[2][3], b23.x, sc[2][1]);
            sc[3][0] = fmaf(chi[3][0] + chi[3][1], a23.y, sc[3][0]); sc[3][1] = fmaf(chi[3][2] + chi[3][3], b23.y, sc[3][1]);
          }
          if (L.k_lo_n[g] > 0) {
#pragma unroll
            for (int s = 0; s < 4; ++s)
#pragma unroll
              for (int e = 0; e < 4; ++e) chi[s][e] = 0.f;
            qk_block<QUANT>(chi, pg, L.k_lo_off[g], L.k_lo_n[g], L.bits_lo, qimg_lane, step, R, j);
            const uint2 h0 = *reinterpret_cast<const uint2*>(ksc + PTOK), h1 = *reinterpret_cast<const uint2*>(ksc + PTOK + 8);
            const float2 a01 = h2_to_f2(h0.x), a23 = h2_to_f2(h0.y), b01 = h2_to_f2(h1.x), b23 = h2_to_f2(h1.y);
            sc[0][0] = fmaf(chi[0][0] + chi[0][1], a01.x, sc[0][0]); sc[0][1] = fmaf(chi[0][2] + chi[0][3], b01.x, sc[0][1]);
            sc[1][0] = fmaf(chi[1][0] + chi[1][1], a01.y, sc[1][0]); sc[1][1] = fmaf(chi[1][2] + chi[1][3], b01.y, sc[1][1]);
            sc[2][0] = fmaf(chi[2][0] + chi[2][1], a23.x, sc[2][0]); sc[2][1] = fmaf(chi[2][2] + chi[2][3], b23.x, sc[2][1]);
            sc[3][0] = fmaf(chi[3][0] + chi[3][1], a23.y, sc[3][0]); sc[3][1] = fmaf(chi[3][2] + chi[3][3], b23.y, sc[3][1]);
          }
        } else {
#pragma unroll
          for (int s = 0; s < 4; ++s) {
            sc[s][0] += chi[s][0] + chi[s][1];
            sc[s][1] += chi[s][2] + chi[s][3];
          }
        }
      }
      if (tail) {
#pragma unroll
        for (int s = 0; s < 4; ++s) {
          if (tb + s * TS >= nvalid) sc[s][0] = -INFINITY;
          if (tb + s * TS + 8 >= nvalid) sc[s][1] = -INFINITY;
        }
      }
      float mx = fmaxf(fmaxf(fmaxf(sc[0][0], sc[0][1]), fmaxf(sc[1][0], sc[1][1])),
                       fmaxf(fmaxf(sc[2][0], sc[2][1]), fmaxf(sc[3][0], sc[3][1])));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
      mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
      const float m_new = fmaxf(m_run, mx);        // finite: slot 0 of every page in range is valid
      const float alpha = exp2f(m_run - m_new);    // 0 on the first page
      const float sh = P_OFFSET - m_new;
      float sum = 0.f;
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        sc[s][0] = exp2f(sc[s][0] + sh);   // -inf -> 0
        sc[s][1] = exp2f(sc[s][1] + sh);
        sum += sc[s][0] + sc[s][1];
      }
      l_run = fmaf(l_run, alpha, sum);
      m_run = m_new;
#pragma unroll
      for (int u = 0; u < 2; ++u)
#pragma unroll
        for (int be = 0; be < 2; ++be) {
          const uint32_t y = movmatrix_trans(pack_h2(sc[2 * u][be], sc[2 * u + 1][be]));
          *reinterpret_cast<uint32_t*>(Pb + p_thr_off + u * (4 * 32 * 16) + be * 4) = y;
        }
      if (R == 0) al[4 * warp + j] = alpha;
    }
    __syncthreads();   // P and alpha of this page complete; every warp is done with page it-1
    if (tid == 0 && it >= 1 && it - 1 + nstage < n_it) issue(it - 1 + nstage);

    // ================= PV: O^T += L_v^T . P^T =================
    {
      bool changed = false;
      float2 alv[NT];
#pragma unroll
      for (int c = 0; c < NT; ++c) {
        alv[c] = *reinterpret_cast<const float2*>(al + 8 * c + 2 * j);
        changed |= (alv[c].x != 1.f) | (alv[c].y != 1.f);
      }
      if (__any_sync(0xffffffffu, changed)) {
#pragma unroll
        for (int c = 0; c < NT; ++c)
#pragma unroll
          for (int a = 0; a < MT; ++a) {
            acc[a][c][0] *= alv[c].x; acc[a][c][1] *= alv[c].y; acc[a][c][2] *= alv[c].x; acc[a][c][3] *= alv[c].y;
          }
      }
    }
    uint4 pf[2][NT];   // [k-step pair][head tile]
#pragma unroll
    for (int sp = 0; sp < 2; ++sp)
#pragma unroll
      for (int c = 0; c < NT; ++c) pf[sp][c] = *reinterpret_cast<const uint4*>(Pb + (((sp * 4 + c) * 32 + lane) << 4));
    int cur_blk = -1;
    uint32_t sc0[4] = {0, 0, 0, 0}, sc2[4] = {0, 0, 0, 0};
#pragma unroll
    for (int a = 0; a < MT; ++a) {
      const int tile = warp + NWARPS * a;
      if (tile >= PL.v_tiles) break;
      const int blk = tile >= PL.v_tiles_hi ? 1 : 0;
      const int ch0 = 16 * (tile - (blk ? PL.v_tiles_hi : 0));
      const int n = blk ? L.v_lo_n : L.v_hi_n;
      const int bits = blk ? L.bits_lo : L.bits_hi;
      const int c0 = min(ch0 + R, n - 1), c1 = min(ch0 + R + 8, n - 1);   // clamped; dead rows zeroed in pv_tile
      const uint8_t* vb = pg + (blk ? L.v_lo_off : L.v_hi_off);
      const int rowb = PTOK * bits / 8;
      if (QUANT && blk != cur_blk) {
        cur_blk = blk;
        const uint4* sp4 = reinterpret_cast<const uint4*>(pg + L.v_scale_off + (blk * PTOK + 16 * j) * 2);
        const uint4 u = sp4[0], v = sp4[1];
        sc0[0] = prmt(u.x, u.z, 0x5410u); sc0[1] = prmt(u.x, u.z, 0x7632u);
        sc0[2] = prmt(u.y, u.w, 0x5410u); sc0[3] = prmt(u.y, u.w, 0x7632u);
        sc2[0] = prmt(v.x, v.z, 0x5410u); sc2[1] = prmt(v.x, v.z, 0x7632u);
        sc2[2] = prmt(v.y, v.w, 0x5410u); sc2[3] = prmt(v.y, v.w, 0x7632u);
      }
      pv_tile<QUANT, NT>(acc[a], vb + c0 * rowb, vb + c1 * rowb, bits, ch0 + R >= n, ch0 + R + 8 >= n, sc0, sc2, pf, j);
    }
  }

  // ================= D7: write the split-K partial =================
  if (has_quad) {
    float lsum = l_run;
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 4);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 8);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 16);
    const int head = 4 * warp + j;
    if (R == 0 && head < L.n_q_heads) {
      my_parts[head * pstride + 0] = m_run;
      my_parts[head * pstride + 1] = lsum;
    }
  }
#pragma unroll
  for (int a = 0; a < MT; ++a) {
    const int tile = warp + NWARPS * a;
    if (tile >= PL.v_tiles) break;
    const int blk = tile >= PL.v_tiles_hi ? 1 : 0;
    const int ch0 = 16 * (tile - (blk ? PL.v_tiles_hi : 0));
    const int n = blk ? L.v_lo_n : L.v_hi_n;
    const int cg = blk ? L.v_hi_n : 0;
#pragma unroll
    for (int c = 0; c < NT; ++c) {
      const int h0 = 8 * c + 2 * j;
#pragma unroll
      for (int e = 0; e < 4; ++e) {
        const int head = h0 + (e & 1), ch = ch0 + R + 8 * (e >> 1);
        if (head < L.n_q_heads && ch < n) my_parts[head * pstride + 2 + cg + ch] = acc[a][c][e];
      }
    }
  }
}

template <bool QUANT, int NT, int MT>
cudaError_t launch_v2(const starkv_ctx* ctx, dim3 grid, const uint8_t* pool, const int32_t* table, int max_pages,
                      const int32_t* seq_lens, const uint8_t* qimg, size_t qimg_stride, float* parts, int n_splits) {
  auto kern = decode_v2_kernel<QUANT, NT, MT, (MT <= 2 ? 2 : 1)>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->plan.smem_bytes);
  if (e != cudaSuccess) return e;
  kern<<<grid, NTHREADS, ctx->plan.smem_bytes, ctx->stream>>>(ctx->L, ctx->plan, pool, table, max_pages, seq_lens, qimg,
                                                              qimg_stride, parts, n_splits);
  return cudaGetLastError();
}

template <bool QUANT>
cudaError_t dispatch_v2(const starkv_ctx* ctx, dim3 grid, const uint8_t* pool, const int32_t* table, int max_pages,
                        const int32_t* seq_lens, const uint8_t* qimg, size_t qimg_stride, float* parts, int n_splits) {
  const int nt = ctx->plan.nt, mt = ctx->plan.mt;
#define SK_V2(NTv, MTv) \
  if (nt == NTv && mt == MTv) \
    return launch_v2<QUANT, NTv, MTv>(ctx, grid, pool, table, max_pages, seq_lens, qimg, qimg_stride, parts, n_splits)
  SK_V2(1, 1); SK_V2(1, 2); SK_V2(1, 3); SK_V2(1, 4);
  SK_V2(2, 1); SK_V2(2, 2); SK_V2(2, 3); SK_V2(2, 4);
  SK_V2(4, 1); SK_V2(4, 2); SK_V2(4, 3); SK_V2(4, 4);
#undef SK_V2
  return cudaErrorInvalidValue;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: plan, workspace, launch
// ---------------------------------------------------------------------------------------------
static int round_up(int x, int m) { return (x + m - 1) / m * m; }

int sk_fast_plan(starkv_ctx* ctx) {
  const StarkvLayout& L = ctx->L;
  V2Plan& P = ctx->plan;
  memset(&P, 0, sizeof(P));
  ctx->fast_ok = 0;
  const int G = L.group;
  if (L.page_tokens != PTOK || L.n_q_heads > 32 || !(G == 1 || G == 2 || G == 4)) return 0;
  const bool quant = L.bits_hi != 16;
  int steps = 0;
  for (int g = 0; g < L.n_kv_heads; ++g) {
    P.qstep_begin[g] = steps;
    const int mh = L.bits_hi == 4 ? 2 * ((L.k_hi_n[g] + 31) / 32) : (L.k_hi_n[g] + 15) / 16;
    const int ml = !quant ? 0 : (L.bits_lo == 4 ? 2 * ((L.k_lo_n[g] + 31) / 32) : (L.k_lo_n[g] + 15) / 16);
    steps += mh + ml;
  }
  for (int g = L.n_kv_heads; g <= STARKV_MAX_KV_HEADS; ++g) P.qstep_begin[g] = steps;
  P.n_qsteps = steps;
  P.qimg_bytes = steps * 256;
  P.nq = (L.n_q_heads + 3) / 4;
  P.kv_per_quad = 4 / G;
  P.nt = L.n_q_heads <= 8 ? 1 : (L.n_q_heads <= 16 ? 2 : 4);
  P.v_tiles_hi = (L.v_hi_n + 15) / 16;
  P.v_tiles = P.v_tiles_hi + (L.v_lo_n + 15) / 16;
  P.mt = (P.v_tiles + NWARPS - 1) / NWARPS;
  if (P.mt > 4) return 0;
  const int fixed = round_up(P.qimg_bytes, 128) + 2 * P_BUF_BYTES + 2 * 32 * 4 + 128 /* barriers */ + 128 /* base align */;
  const int max_one = ctx->smem_optin;                       // 227 KB on sm_100a
  const int max_two = (ctx->smem_per_sm - 2 * 1024) / 2;     // two resident CTAs (1 KB reserved each)
  int ctas = 1, nstage = 0;
  if (P.mt <= 2) {
    int ns = (max_two - fixed) / L.page_bytes;
    if (ns > 4) ns = 4;
    if (ns >= 3) { ctas = 2; nstage = ns; }
  }
  if (nstage == 0) {
    int ns = (max_one - fixed) / L.page_bytes;
    if (ns > 4) ns = 4;
    if (ns < 2) return 0;
    nstage = ns;
  }
  P.ctas_per_sm = ctas;
  P.nstage = nstage;
  int off = 0;
  P.off_stage = off; off += nstage * L.page_bytes;           // page_bytes is a multiple of 128
  P.off_qimg = off; off += round_up(P.qimg_bytes, 128);
  P.off_p = off; off += 2 * P_BUF_BYTES;
  P.off_alpha = off; off += 2 * 32 * 4;
  P.off_bar = off; off += 8 * (nstage + 1);
  P.smem_bytes = round_up(off, 128);
  ctx->fast_ok = 1;
  return 1;
}

int sk_fast_supported(const starkv_ctx* ctx) { return ctx->fast_ok; }

void sk_plan_workspace(const starkv_ctx* ctx, int batch, int max_pages, SkWorkspace* w) {
  const StarkvLayout& L = ctx->L;
  const int slots = ctx->n_sm * (ctx->fast_ok ? ctx->plan.ctas_per_sm : 1);
  int ns = ctx->n_splits_override > 0 ? ctx->n_splits_override : slots / (batch > 0 ? batch : 1);
  if (ns > max_pages) ns = max_pages;
  if (ns < 1) ns = 1;
  w->n_splits = ns;
  size_t off = 0;
  w->qimg_stride = (size_t)round_up(ctx->fast_ok ? ctx->plan.qimg_bytes : 0, 256);
  w->qimg_off = off; off += w->qimg_stride * batch;
  w->part_off = off; off += ((size_t)batch * ns * L.n_q_heads * sk_part_stride(L.rank_v) * 4 + 255) / 256 * 256;
  w->host_off = off;
  const size_t qb = ((size_t)batch * L.n_q_heads * L.head_dim * 2 + 255) / 256 * 256;
  off += 2 * qb + ((size_t)batch * 4 + 255) / 256 * 256;
  w->total = off;
}

int sk_decode_fast(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                   const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                   void* out) {
  const StarkvLayout& L = ctx->L;
  const V2Plan& P = ctx->plan;
  ctx->last_launches = 0;
  if (!ctx->fast_ok) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  uint8_t* qimg = (uint8_t*)ws + w.qimg_off;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  qproj_kernel<<<dim3(L.n_kv_heads, batch), 128, 0, ctx->stream>>>(L, P, (const __half*)q, (const __half*)B_k,
                                                                   (uint32_t*)qimg, w.qimg_stride / 4);
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  const dim3 grid(w.n_splits, batch);
  const uint8_t* pl = (const uint8_t*)pool;
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  const cudaError_t e = L.bits_hi != 16
      ? dispatch_v2<true>(ctx, grid, pl, table, max_pages, seq_lens, qimg, w.qimg_stride, parts, w.n_splits)
      : dispatch_v2<false>(ctx, grid, pl, table, max_pages, seq_lens, qimg, w.qimg_stride, parts, w.n_splits);
  SK_CUDA_CHECK(ctx, e);
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out);
  ctx->last_launches = 3;
  return rc;
}
