// Tensor-core decode attention over the latent cache (rows D1-D7 of the hot path), sm_100a.
//
//   PAPER.md §3.3: scores in latent space  s_t = q~ . L_k[t],  q~ = sm_scale q B_k^T  (no RoPE on
//   this path, A1), and the value side reordered as (p L_v) B_v  ("(p V') U_V").
//   PAPER.md A.6 L627: stack p over heads so that p L_v is ONE GEMM  P[H_q x T] . L_v[T x r_v]  -> tensor cores.
//   PAPER.md Eq.12 L208 / A.6 L625: latents are dequantised in registers, never materialised.
//
// One CTA (8 warps) walks a contiguous page range of one sequence (split-K).  Pages are pulled into a
// shared-memory ring with cp.async.bulk + mbarrier (one bulk copy per page: a page is one contiguous
// byte range by construction of the format).  Per iteration of IT_PAGES pages (64 tokens each):
//   phase A  QK on mma.sync m16n8k16:  S^T[tokens x (head,hi/lo)] = L_k[tokens x ch] . q~^T, the latent
//            query split into an fp16 hi+lo pair that occupies two MMA columns per head, so that
//            hi+lo lands in one thread and the score keeps fp32 accuracy; int4/int8 fields go to fp16
//            with the magic-number lop3/prmt trick (exact), per-token scales are applied to the fp32 sums.
//   phase B  online softmax (base 2, running max per head), P -> fp16 with a 2^14 offset, written to
//            shared memory in the k-order the PV fragments want.
//   phase C  PV on mma.sync:  O^T[ch x heads] += L_v^T[ch x tokens] . P^T[tokens x heads]; L_v is
//            stored channel-major so a 32-bit word holds consecutive tokens of one channel = the A
//            fragment's k pairs; value scales are applied element-wise in fp16 (c*s, one rounding).
// The partial (m, l, acc[H_q x r_v]) goes to the workspace; combine_kernel merges and up-projects.
#include <string.h>

#include "decode_common.cuh"
#include "decode_fast.h"

namespace {

constexpr int NWARPS = 8;
constexpr int NTHREADS = NWARPS * 32;
constexpr int PTOK = 64;          // tokens per page on this path
constexpr float P_OFFSET = 14.f;  // P is stored as 2^(s - m + 14) in fp16 (keeps small weights normal)
constexpr float kLog2e = 1.4426950408889634f;

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
// and laid out as the B fragments of the QK MMAs (see FastPlan).  grid (ceil(words/256), batch).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) qproj_kernel(const __grid_constant__ StarkvLayout L,
                                                    const __grid_constant__ FastPlan PL,
                                                    const __half* __restrict__ q, const __half* __restrict__ B_k,
                                                    uint32_t* __restrict__ qimg_all, size_t qimg_stride_words) {
  const int wi = blockIdx.x * blockDim.x + threadIdx.x;
  const int n_words = PL.n_qsteps * PL.ntq * 64;
  if (wi >= n_words) return;
  const int b = blockIdx.y;
  const int reg = wi & 1, lane = (wi >> 1) & 31;
  const int ntile = (wi >> 6) % PL.ntq, step = (wi >> 6) / PL.ntq;
  int g = 0;
  while (step >= PL.qstep_begin[g + 1]) ++g;
  int local = step - PL.qstep_begin[g];
  const int n_hi = L.k_hi_n[g], n_lo = L.k_lo_n[g];
  const int mh = L.bits_hi == 4 ? 2 * ((n_hi + 31) >> 5) : (n_hi + 15) >> 4;
  int blk = 0;
  if (local >= mh) { blk = 1; local -= mh; }
  const int bits = blk ? L.bits_lo : L.bits_hi;
  const int n = blk ? n_lo : n_hi;
  const int chunk = bits == 4 ? local >> 1 : local, m = bits == 4 ? local & 1 : 0;
  const int col = ntile * 8 + (lane >> 2);
  const int i = col >> 1, hilo = col & 1;
  const int j = lane & 3;
  uint32_t word = 0;
  if (i < L.group) {
    const __half* qrow = q + ((size_t)b * L.n_q_heads + g * L.group + i) * L.head_dim;
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int k = 2 * j + e + 8 * reg;
      const int ch = chunk * (bits == 4 ? 32 : 16) + fast_k_to_channel(bits, m, k);
      if (ch >= n) continue;
      const __half* brow = B_k + (size_t)(L.koff[g] + (blk ? n_hi : 0) + ch) * L.head_dim;
      float a = 0.f;
      for (int d = 0; d < L.head_dim; d += 2) {
        const float2 qq = __half22float2(*reinterpret_cast<const __half2*>(qrow + d));
        const float2 bb = __half22float2(*reinterpret_cast<const __half2*>(brow + d));
        a = fmaf(qq.x, bb.x, a);
        a = fmaf(qq.y, bb.y, a);
      }
      a *= L.sm_scale * kLog2e;
      const __half hi = __float2half_rn(a);
      const __half v = hilo ? __float2half_rn(a - __half2float(hi)) : hi;
      word |= (uint32_t)__half_as_ushort(v) << (16 * e);
    }
  }
  qimg_all[(size_t)b * qimg_stride_words + wi] = word;
}

// ---------------------------------------------------------------------------------------------
// QK helpers (phase A).  TPW = 16-token tiles per warp.
// ---------------------------------------------------------------------------------------------
struct RowPtr {            // per-thread addressing of its two token rows in each of its tiles
  const uint8_t* page[4];  // page base of tile t
  int slot[4];             // slot of row R in tile t (second row = slot + 8)
};

template <int TPW>
__device__ __forceinline__ void qk_block(float (&acc)[TPW][4], const RowPtr& rp, int block_off, int n, int bits,
                                         const uint2* __restrict__ qimg, int& step, int ntq, int ntile, int lane) {
  const int j = lane & 3;
  if (bits == 4) {
    const int rowbytes = n >> 1;
    const int nchunks = (n + 31) >> 5;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf0 = qimg[(step * ntq + ntile) * 32 + lane];
      const uint2 bf1 = qimg[((step + 1) * ntq + ntile) * 32 + lane];
      step += 2;
      const bool valid = c * 32 + 8 * j < n;
#pragma unroll
      for (int t = 0; t < TPW; ++t) {
        const uint8_t* r0 = rp.page[t] + block_off + rp.slot[t] * rowbytes + c * 16 + 4 * j;
        const uint32_t w0 = valid ? *reinterpret_cast<const uint32_t*>(r0) : 0x88888888u;
        const uint32_t w1 = valid ? *reinterpret_cast<const uint32_t*>(r0 + 8 * rowbytes) : 0x88888888u;
        uint32_t h0[4], h1[4];
        deq4_pairs(w0, h0);
        deq4_pairs(w1, h1);
        mma16816(acc[t], h0[0], h1[0], h0[1], h1[1], bf0.x, bf0.y);
        mma16816(acc[t], h0[2], h1[2], h0[3], h1[3], bf1.x, bf1.y);
      }
    }
  } else if (bits == 8) {
    const int rowbytes = n;
    const int nchunks = (n + 15) >> 4;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf = qimg[(step * ntq + ntile) * 32 + lane];
      step += 1;
      const bool valid = c * 16 + 4 * j < n;
#pragma unroll
      for (int t = 0; t < TPW; ++t) {
        const uint8_t* r0 = rp.page[t] + block_off + rp.slot[t] * rowbytes + c * 16 + 4 * j;
        const uint32_t w0 = valid ? *reinterpret_cast<const uint32_t*>(r0) : 0x80808080u;
        const uint32_t w1 = valid ? *reinterpret_cast<const uint32_t*>(r0 + 8 * rowbytes) : 0x80808080u;
        uint32_t a0, a1, a2, a3;
        deq8_pairs(w0, a0, a2);
        deq8_pairs(w1, a1, a3);
        mma16816(acc[t], a0, a1, a2, a3, bf.x, bf.y);
      }
    }
  } else {
    const int rowbytes = 2 * n;
    const int nchunks = (n + 15) >> 4;
    for (int c = 0; c < nchunks; ++c) {
      const uint2 bf = qimg[(step * ntq + ntile) * 32 + lane];
      step += 1;
      const bool valid = c * 16 + 4 * j < n;
#pragma unroll
      for (int t = 0; t < TPW; ++t) {
        const uint8_t* r0 = rp.page[t] + block_off + rp.slot[t] * rowbytes + c * 32 + 8 * j;
        uint2 x0 = make_uint2(0, 0), x1 = make_uint2(0, 0);
        if (valid) {
          x0 = *reinterpret_cast<const uint2*>(r0);
          x1 = *reinterpret_cast<const uint2*>(r0 + 8 * rowbytes);
        }
        mma16816(acc[t], x0.x, x1.x, x0.y, x1.y, bf.x, bf.y);
      }
    }
  }
}

// ---------------------------------------------------------------------------------------------
// Main kernel.  grid (n_splits, batch), 256 threads, 1 CTA / SM.
//   QUANT   integer latents (else fp16)     NT  head tiles of 8 (ceil(H_q/8))
//   MT      value M tiles (16 channels) per warp        ITP  pages per iteration
// ---------------------------------------------------------------------------------------------
template <bool QUANT, int NT, int MT, int ITP>
__global__ void __launch_bounds__(NTHREADS, 1) decode_fast_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ FastPlan PL, const uint8_t* __restrict__ pool,
    const int32_t* __restrict__ table, int max_pages, const int32_t* __restrict__ seq_lens,
    const uint8_t* __restrict__ qimg_all, size_t qimg_stride, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr int TILES = 4 * ITP;       // 16-token tiles per iteration
  constexpr int TPW = TILES / 2;       // QK: tiles per warp (2 tile-sets x 4 head-sets)
  constexpr int SP = 64 * ITP;         // S row pitch (floats)
  constexpr int PPITCH = 128 * ITP;    // P row pitch (bytes)
  constexpr int NCH = 4 * ITP;         // 16-token chunks per iteration

  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int j = lane & 3, R = lane >> 2;
  const int split = blockIdx.x, b = blockIdx.y;
  const int len = seq_lens[b];
  const int n_pages = (len + PTOK - 1) / PTOK;
  int p0, p1;
  sk_split_range(n_pages, n_splits, ITP, split, &p0, &p1);
  const int n_it = (p1 - p0 + ITP - 1) / ITP;
  const size_t pstride = sk_part_stride(L.rank_v);
  float* my_parts = parts + ((size_t)b * n_splits + split) * L.n_q_heads * pstride;

  if (n_it == 0) {   // empty range: neutral partial
    for (int i = tid; i < L.n_q_heads * (int)pstride; i += NTHREADS) {
      const int c = i % (int)pstride;
      my_parts[i] = c == 0 ? -INFINITY : 0.f;
    }
    return;
  }

  uint8_t* stage_base = smem + PL.off_stage;
  const uint2* qimg = reinterpret_cast<const uint2*>(smem + PL.off_qimg);
  float* S = reinterpret_cast<float*>(smem + PL.off_s);
  uint8_t* Pm = smem + PL.off_p;
  float* maxbuf = reinterpret_cast<float*>(smem + PL.off_max);      // [2][NT*8]
  float* alpha_s = reinterpret_cast<float*>(smem + PL.off_alpha);   // [NT*8]
  const uint32_t bar0 = smem_u32(smem + PL.off_bar);                // full[nstage], then qbar
  const uint32_t qbar = bar0 + 8 * PL.nstage;
  const int32_t* my_table = table + (size_t)b * max_pages;

  auto issue = [&](int it) {   // thread 0 only
    const int st = it % PL.nstage;
    const int pg0 = p0 + it * ITP;
    const int npg = min(ITP, p1 - pg0);
    const uint32_t bar = bar0 + 8 * st;
    mbar_expect_tx(bar, (uint32_t)(npg * L.page_bytes));
    for (int k = 0; k < npg; ++k)
      bulk_g2s(smem_u32(stage_base + (size_t)st * PL.stage_bytes + (size_t)k * L.page_bytes),
               pool + (size_t)my_table[pg0 + k] * L.page_bytes, (uint32_t)L.page_bytes, bar);
  };

  if (tid == 0) {
    for (int s = 0; s < PL.nstage; ++s) mbar_init(bar0 + 8 * s, 1);
    mbar_init(qbar, 1);
    fence_barrier_init();
    mbar_expect_tx(qbar, (uint32_t)PL.qimg_bytes);
    bulk_g2s(smem_u32(smem + PL.off_qimg), qimg_all + (size_t)b * qimg_stride, (uint32_t)PL.qimg_bytes, qbar);
    for (int it = 0; it < min(PL.nstage, n_it); ++it) issue(it);
  }
  for (int i = tid; i < NT * 8 * PPITCH / 16; i += NTHREADS) reinterpret_cast<uint4*>(Pm)[i] = make_uint4(0, 0, 0, 0);
  if (tid < NT * 8) alpha_s[tid] = 1.f;
  __syncthreads();

  // phase-B identity of this thread: (head, 16-token chunk); persistent running max / sum
  const int hb = warp % NT, cb = warp / NT;
  const int b_head = hb * 8 + (lane & 7), b_chunk = cb * 4 + (lane >> 3);
  const bool b_active = warp < NT * ITP && b_head < L.n_q_heads;
  float m_run = -INFINITY, l_run = 0.f;

  float acc[MT][NT][4];
#pragma unroll
  for (int a = 0; a < MT; ++a)
#pragma unroll
    for (int c = 0; c < NT; ++c)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[a][c][e] = 0.f;

  const int hs = warp & 3, ts = warp >> 2;
  mbar_wait(qbar, 0);

  for (int it = 0; it < n_it; ++it) {
    const int st = it % PL.nstage;
    uint8_t* stg = stage_base + (size_t)st * PL.stage_bytes;
    const int pg0 = p0 + it * ITP;
    mbar_wait(bar0 + 8 * st, (uint32_t)((it / PL.nstage) & 1));
    const bool tail = (pg0 + ITP > p1) || ((pg0 + ITP) * PTOK > len);

    if (tail) {   // neutralise value data of slots past the sequence end (they may hold any bits)
      for (int k = 0; k < ITP; ++k) {
        if (pg0 + k >= p1) break;
        const int nvalid = min(PTOK, len - (pg0 + k) * PTOK);
        if (nvalid >= PTOK) continue;
        uint8_t* pg = stg + (size_t)k * L.page_bytes;
        if (QUANT) {
          if (tid < 2 * PTOK && (tid & (PTOK - 1)) >= nvalid) reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[tid] = 0;
        } else {
          const int nbad = PTOK - nvalid;
          for (int i = tid; i < L.rank_v * nbad; i += NTHREADS)
            reinterpret_cast<uint16_t*>(pg + L.v_hi_off)[(i / nbad) * PTOK + nvalid + i % nbad] = 0;
        }
      }
      fence_proxy_async();
      __syncthreads();
    }

    // ================= phase A: S^T = L_k . q~^T =================
    {
      RowPtr rp;
#pragma unroll
      for (int t = 0; t < TPW; ++t) {
        const int tile = ts * TPW + t;
        rp.page[t] = stg + (size_t)(tile >> 2) * L.page_bytes;
        rp.slot[t] = (tile & 3) * 16 + R;
      }
      for (int g = 0; g < L.n_kv_heads; ++g) {
        if (PL.qk_owner[g] != hs) continue;
        for (int ntile = 0; ntile < PL.ntq; ++ntile) {
          float chi[TPW][4], clo[TPW][4];
#pragma unroll
          for (int t = 0; t < TPW; ++t)
#pragma unroll
            for (int e = 0; e < 4; ++e) chi[t][e] = clo[t][e] = 0.f;
          int step = PL.qstep_begin[g];
          qk_block<TPW>(chi, rp, L.k_hi_off[g], L.k_hi_n[g], L.bits_hi, qimg, step, PL.ntq, ntile, lane);
          if (QUANT && L.k_lo_n[g] > 0)
            qk_block<TPW>(clo, rp, L.k_lo_off[g], L.k_lo_n[g], L.bits_lo, qimg, step, PL.ntq, ntile, lane);
          const int hi_in_group = ntile * 4 + j;
          const int head = g * L.group + hi_in_group;
          const bool hvalid = hi_in_group < L.group;
          float mx = -INFINITY;
#pragma unroll
          for (int t = 0; t < TPW; ++t) {
            float s0 = chi[t][0] + chi[t][1], s1 = chi[t][2] + chi[t][3];
            if (QUANT) {
              const __half* ksc = reinterpret_cast<const __half*>(rp.page[t] + L.k_scale_off) + (g * 2) * PTOK + rp.slot[t];
              s0 *= __half2float(ksc[0]);
              s1 *= __half2float(ksc[8]);
              if (L.k_lo_n[g] > 0) {
                s0 = fmaf(clo[t][0] + clo[t][1], __half2float(ksc[PTOK]), s0);
                s1 = fmaf(clo[t][2] + clo[t][3], __half2float(ksc[PTOK + 8]), s1);
              }
            }
            const int tile = ts * TPW + t;
            if (tail) {
              const int tok = (pg0 + (tile >> 2)) * PTOK + rp.slot[t];
              const bool pok = pg0 + (tile >> 2) < p1;
              if (!(pok && tok < len)) s0 = -INFINITY;
              if (!(pok && tok + 8 < len)) s1 = -INFINITY;
            }
            mx = fmaxf(mx, fmaxf(s0, s1));
            if (hvalid) {
              const int swz = ((head & 3) << 3) ^ (((head >> 2) & 1) << 2);
              const int tk = tile * 16 + R;
              S[head * SP + (tk ^ swz)] = s0;
              S[head * SP + ((tk + 8) ^ swz)] = s1;
            }
          }
          mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 4));
          mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 8));
          mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, 16));
          if (R == 0 && hvalid) maxbuf[ts * (NT * 8) + head] = mx;
        }
      }
    }
    __syncthreads();   // #1: S and maxbuf complete; every warp is done with iteration it-1
    if (tid == 0 && it >= 1 && it - 1 + PL.nstage < n_it) issue(it - 1 + PL.nstage);

    // ================= phase B: online softmax, P -> fp16 =================
    int changed = 0;
    if (b_active) {
      const float m_blk = fmaxf(maxbuf[b_head], maxbuf[NT * 8 + b_head]);
      const float m_new = fmaxf(m_run, m_blk);
      const float alpha = exp2f(m_run - m_new);
      changed = alpha != 1.f;
      const int swz = ((b_head & 3) << 3) ^ (((b_head >> 2) & 1) << 2);
      float p[16];
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        const float4 v = *reinterpret_cast<const float4*>(S + b_head * SP + ((16 * b_chunk + 4 * i) ^ swz));
        p[4 * i + 0] = v.x; p[4 * i + 1] = v.y; p[4 * i + 2] = v.z; p[4 * i + 3] = v.w;
      }
      const float sh = P_OFFSET - m_new;
      float sum = 0.f;
#pragma unroll
      for (int x = 0; x < 16; ++x) {
        p[x] = exp2f(p[x] + sh);   // -inf -> 0
        sum += p[x];
      }
      l_run = l_run * alpha + sum;
      m_run = m_new;
      // position 4s + 2half + e  <->  token x = 8half + (QUANT ? s + 4e : 2s + e)
      uint32_t w[8];
#pragma unroll
      for (int s = 0; s < 4; ++s)
#pragma unroll
        for (int half = 0; half < 2; ++half) {
          const int x0 = 8 * half + (QUANT ? s : 2 * s), x1 = 8 * half + (QUANT ? s + 4 : 2 * s + 1);
          w[2 * s + half] = pack_h2(p[x0], p[x1]);
        }
      uint8_t* prow = Pm + b_head * PPITCH;
      const int g0 = 2 * b_chunk, key = b_head & 7;
      *reinterpret_cast<uint4*>(prow + ((g0 ^ key) << 4)) = make_uint4(w[0], w[1], w[2], w[3]);
      *reinterpret_cast<uint4*>(prow + (((g0 + 1) ^ key) << 4)) = make_uint4(w[4], w[5], w[6], w[7]);
      if (b_chunk == 0) alpha_s[b_head] = alpha;
    }
    const int need = __syncthreads_or(changed);   // #2: P and alpha complete

    // ================= phase C: O^T += L_v^T . P^T =================
    if (need) {
#pragma unroll
      for (int c = 0; c < NT; ++c) {
        const float2 al = *reinterpret_cast<const float2*>(alpha_s + 8 * c + 2 * j);
#pragma unroll
        for (int a = 0; a < MT; ++a) {
          acc[a][c][0] *= al.x; acc[a][c][1] *= al.y; acc[a][c][2] *= al.x; acc[a][c][3] *= al.y;
        }
      }
    }
#pragma unroll 1
    for (int k = 0; k < ITP; ++k) {
      if (pg0 + k >= p1) break;
      const uint8_t* pg = stg + (size_t)k * L.page_bytes;
      uint4 pf[2][NT];   // [k-step pair][head tile]: b0,b1 of step 2sp, b0,b1 of step 2sp+1
#pragma unroll
      for (int sp = 0; sp < 2; ++sp)
#pragma unroll
        for (int c = 0; c < NT; ++c)
          pf[sp][c] = *reinterpret_cast<const uint4*>(Pm + (8 * c + R) * PPITCH + (((8 * k + 2 * j + sp) ^ R) << 4));
      int cur_blk = -1;
      uint32_t sc0[4], sc2[4];
#pragma unroll
      for (int a = 0; a < MT; ++a) {
        const int tile = warp + NWARPS * a;
        if (tile >= PL.v_tiles) break;
        const int blk = tile >= PL.v_tiles_hi ? 1 : 0;
        const int ch0 = 16 * (tile - (blk ? PL.v_tiles_hi : 0));
        const int n = blk ? L.v_lo_n : L.v_hi_n;
        const int bits = blk ? L.bits_lo : L.bits_hi;
        const int c0 = min(ch0 + R, n - 1), c1 = min(ch0 + R + 8, n - 1);   // clamped; dead rows zeroed below
        const uint8_t* vb = pg + (blk ? L.v_lo_off : L.v_hi_off);
        uint32_t A0[4], A1[4], A2[4], A3[4];
        if (QUANT) {
          if (blk != cur_blk) {
            cur_blk = blk;
            const uint4* sp4 = reinterpret_cast<const uint4*>(pg + L.v_scale_off + (blk * PTOK + 16 * j) * 2);
            const uint4 u = sp4[0], v = sp4[1];
            sc0[0] = prmt(u.x, u.z, 0x5410u); sc0[1] = prmt(u.x, u.z, 0x7632u);
            sc0[2] = prmt(u.y, u.w, 0x5410u); sc0[3] = prmt(u.y, u.w, 0x7632u);
            sc2[0] = prmt(v.x, v.z, 0x5410u); sc2[1] = prmt(v.x, v.z, 0x7632u);
            sc2[2] = prmt(v.y, v.w, 0x5410u); sc2[3] = prmt(v.y, v.w, 0x7632u);
          }
          if (bits == 4) {
            const uint2 x0 = *reinterpret_cast<const uint2*>(vb + c0 * (PTOK / 2) + 8 * j);
            const uint2 x1 = *reinterpret_cast<const uint2*>(vb + c1 * (PTOK / 2) + 8 * j);
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
            const uint4 x0 = *reinterpret_cast<const uint4*>(vb + c0 * PTOK + 16 * j);
            const uint4 x1 = *reinterpret_cast<const uint4*>(vb + c1 * PTOK + 16 * j);
            auto deq8v = [&](uint32_t wa, uint32_t wb, const uint32_t (&sc)[4], uint32_t (&out)[4]) {
              const uint32_t ta = prmt(wa, wb, 0x5140u), tb = prmt(wa, wb, 0x7362u);
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
          const uint4* r0 = reinterpret_cast<const uint4*>(vb + c0 * (PTOK * 2) + 32 * j);
          const uint4* r1 = reinterpret_cast<const uint4*>(vb + c1 * (PTOK * 2) + 32 * j);
          const uint4 x0 = r0[0], y0 = r0[1], x1 = r1[0], y1 = r1[1];
          A0[0] = x0.x; A0[1] = x0.y; A0[2] = x0.z; A0[3] = x0.w;
          A2[0] = y0.x; A2[1] = y0.y; A2[2] = y0.z; A2[3] = y0.w;
          A1[0] = x1.x; A1[1] = x1.y; A1[2] = x1.z; A1[3] = x1.w;
          A3[0] = y1.x; A3[1] = y1.y; A3[2] = y1.z; A3[3] = y1.w;
        }
        if (ch0 + 16 > n) {   // ragged last tile of a block: rows past the block contribute nothing
          const bool d0 = ch0 + R >= n, d1 = ch0 + R + 8 >= n;
#pragma unroll
          for (int s = 0; s < 4; ++s) {
            if (d0) { A0[s] = 0; A2[s] = 0; }
            if (d1) { A1[s] = 0; A3[s] = 0; }
          }
        }
#pragma unroll
        for (int s = 0; s < 4; ++s)
#pragma unroll
          for (int c = 0; c < NT; ++c) {
            const uint4 f = pf[s >> 1][c];
            mma16816(acc[a][c], A0[s], A1[s], A2[s], A3[s], (s & 1) ? f.z : f.x, (s & 1) ? f.w : f.y);
          }
      }
    }
  }

  // ================= D7: write the split-K partial =================
  __syncthreads();
  float* stgf = reinterpret_cast<float*>(stage_base);   // [NT*8][rank_v] fp32 staging (ring is drained)
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
      if (ch0 + R < n) {
        stgf[h0 * L.rank_v + cg + ch0 + R] = acc[a][c][0];
        stgf[(h0 + 1) * L.rank_v + cg + ch0 + R] = acc[a][c][1];
      }
      if (ch0 + R + 8 < n) {
        stgf[h0 * L.rank_v + cg + ch0 + R + 8] = acc[a][c][2];
        stgf[(h0 + 1) * L.rank_v + cg + ch0 + R + 8] = acc[a][c][3];
      }
    }
  }
  // running sum: lanes of one head differ in bits 3,4; chunk blocks cb live in different warps
  float lsum = l_run;
  lsum += __shfl_xor_sync(0xffffffffu, lsum, 8);
  lsum += __shfl_xor_sync(0xffffffffu, lsum, 16);
  float* lsm = reinterpret_cast<float*>(smem + PL.off_s);   // S is free now: [ITP][NT*8] sums, then [NT*8] maxima
  if (b_active && (lane >> 3) == 0) {
    lsm[cb * (NT * 8) + b_head] = lsum;
    if (cb == 0) lsm[ITP * (NT * 8) + b_head] = m_run;
  }
  __syncthreads();
  for (int i = tid; i < L.n_q_heads * L.rank_v; i += NTHREADS) {
    const int head = i / L.rank_v, c = i % L.rank_v;
    my_parts[head * pstride + 2 + c] = stgf[i];
  }
  if (tid < L.n_q_heads) {
    float l = 0.f;
    for (int c = 0; c < ITP; ++c) l += lsm[c * (NT * 8) + tid];
    my_parts[tid * pstride + 0] = lsm[ITP * (NT * 8) + tid];
    my_parts[tid * pstride + 1] = l;
  }
}

template <bool QUANT, int NT, int MT, int ITP>
cudaError_t launch_fast(const starkv_ctx* ctx, dim3 grid, const uint8_t* pool, const int32_t* table, int max_pages,
                        const int32_t* seq_lens, const uint8_t* qimg, size_t qimg_stride, float* parts, int n_splits) {
  auto kern = decode_fast_kernel<QUANT, NT, MT, ITP>;
  cudaError_t e = cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, ctx->plan.smem_bytes);
  if (e != cudaSuccess) return e;
  kern<<<grid, NTHREADS, ctx->plan.smem_bytes, ctx->stream>>>(ctx->L, ctx->plan, pool, table, max_pages, seq_lens, qimg,
                                                              qimg_stride, parts, n_splits);
  return cudaGetLastError();
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: plan, workspace, launch
// ---------------------------------------------------------------------------------------------
static int round_up(int x, int m) { return (x + m - 1) / m * m; }

int sk_fast_plan(starkv_ctx* ctx) {
  const StarkvLayout& L = ctx->L;
  FastPlan& P = ctx->plan;
  memset(&P, 0, sizeof(P));
  ctx->fast_ok = 0;
  if (L.page_tokens != PTOK || L.n_q_heads > 32 || L.rank_v > 512 || L.n_kv_heads > STARKV_MAX_KV_HEADS) return 0;
  const bool quant = L.bits_hi != 16;
  // q steps and the head-set that scores each KV head (longest-processing-time-first over 4 sets)
  int cost[STARKV_MAX_KV_HEADS];
  int steps = 0;
  for (int g = 0; g < L.n_kv_heads; ++g) {
    P.qstep_begin[g] = steps;
    const int mh = L.bits_hi == 4 ? 2 * ((L.k_hi_n[g] + 31) / 32) : (L.k_hi_n[g] + 15) / 16;
    const int ml = !quant ? 0 : (L.bits_lo == 4 ? 2 * ((L.k_lo_n[g] + 31) / 32) : (L.k_lo_n[g] + 15) / 16);
    cost[g] = mh + ml;
    steps += mh + ml;
  }
  for (int g = L.n_kv_heads; g <= STARKV_MAX_KV_HEADS; ++g) P.qstep_begin[g] = steps;
  P.n_qsteps = steps;
  int load[4] = {0, 0, 0, 0};
  bool done[STARKV_MAX_KV_HEADS] = {false};
  for (int k = 0; k < L.n_kv_heads; ++k) {
    int best = -1;
    for (int g = 0; g < L.n_kv_heads; ++g)
      if (!done[g] && (best < 0 || cost[g] > cost[best])) best = g;
    int s = 0;
    for (int i = 1; i < 4; ++i)
      if (load[i] < load[s]) s = i;
    done[best] = true;
    P.qk_owner[best] = s;
    load[s] += cost[best];
  }
  P.ntq = (2 * L.group + 7) / 8;
  P.qimg_bytes = P.n_qsteps * P.ntq * 256;
  P.nt = L.n_q_heads <= 8 ? 1 : 4;
  P.v_tiles_hi = (L.v_hi_n + 15) / 16;
  P.v_tiles = P.v_tiles_hi + (L.v_lo_n + 15) / 16;
  if (P.v_tiles > 4 * NWARPS) return 0;
  const int max_smem = ctx->smem_optin;
  for (int itp = 2; itp >= 1; --itp) {
    const int s_bytes = P.nt * 8 * 64 * itp * 4, p_bytes = P.nt * 8 * 128 * itp;
    const int fixed = round_up(P.qimg_bytes, 128) + s_bytes + p_bytes + 2 * P.nt * 8 * 4 + P.nt * 8 * 4 + 128;
    const int stage_bytes = itp * L.page_bytes;
    int nstage = (max_smem - fixed - 128) / stage_bytes;
    if (nstage > 4) nstage = 4;
    if (nstage < (itp == 2 ? 3 : 2)) continue;
    int stage_area = nstage * stage_bytes;
    const int staging = P.nt * 8 * L.rank_v * 4;
    if (stage_area < staging) stage_area = round_up(staging, 128);
    if (stage_area + fixed > max_smem) continue;
    P.it_pages = itp; P.nstage = nstage; P.stage_bytes = stage_bytes;
    int off = 0;
    P.off_stage = off; off += stage_area;
    P.off_qimg = off; off += round_up(P.qimg_bytes, 128);
    P.off_s = off; off += s_bytes;
    P.off_p = off; off += p_bytes;
    P.off_max = off; off += 2 * P.nt * 8 * 4;
    P.off_alpha = off; off += P.nt * 8 * 4;
    P.off_bar = round_up(off, 8); off = P.off_bar + 8 * (nstage + 1);
    P.smem_bytes = round_up(off, 128);
    ctx->fast_ok = 1;
    return 1;
  }
  return 0;
}

int sk_fast_supported(const starkv_ctx* ctx) { return ctx->fast_ok; }

void sk_plan_workspace(const starkv_ctx* ctx, int batch, int max_pages, SkWorkspace* w) {
  const StarkvLayout& L = ctx->L;
  const int gran = ctx->fast_ok ? ctx->plan.it_pages : 1;
  int ns = ctx->n_splits_override > 0 ? ctx->n_splits_override : ctx->n_sm / (batch > 0 ? batch : 1);
  const int units = (max_pages + gran - 1) / gran;
  if (ns > units) ns = units;
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
  const FastPlan& P = ctx->plan;
  ctx->last_launches = 0;
  if (!ctx->fast_ok) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  uint8_t* qimg = (uint8_t*)ws + w.qimg_off;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  const int n_words = P.n_qsteps * P.ntq * 64;
  qproj_kernel<<<dim3((n_words + 255) / 256, batch), 256, 0, ctx->stream>>>(L, P, (const __half*)q, (const __half*)B_k,
                                                                            (uint32_t*)qimg, w.qimg_stride / 4);
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  const dim3 grid(w.n_splits, batch);
  const bool quant = L.bits_hi != 16;
  const int mt = P.v_tiles <= 2 * NWARPS ? 2 : 4;
  const uint8_t* pl = (const uint8_t*)pool;
  cudaError_t e = cudaErrorInvalidValue;
#define SK_LAUNCH(Q, NTv, MTv, ITPv) \
  e = launch_fast<Q, NTv, MTv, ITPv>(ctx, grid, pl, table, max_pages, seq_lens, qimg, w.qimg_stride, parts, w.n_splits)
#define SK_PICK_ITP(Q, NTv, MTv) \
  do { if (P.it_pages == 2) SK_LAUNCH(Q, NTv, MTv, 2); else SK_LAUNCH(Q, NTv, MTv, 1); } while (0)
#define SK_PICK_MT(Q, NTv) \
  do { if (mt == 2) SK_PICK_ITP(Q, NTv, 2); else SK_PICK_ITP(Q, NTv, 4); } while (0)
#define SK_PICK_NT(Q) \
  do { if (P.nt == 1) SK_PICK_MT(Q, 1); else SK_PICK_MT(Q, 4); } while (0)
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  if (quant) SK_PICK_NT(true); else SK_PICK_NT(false);
#undef SK_PICK_NT
#undef SK_PICK_MT
#undef SK_PICK_ITP
#undef SK_LAUNCH
  SK_CUDA_CHECK(ctx, e);
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out);
  ctx->last_launches = 3;
  return rc;
}
