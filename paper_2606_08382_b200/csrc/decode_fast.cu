// Tensor-core decode attention over the latent cache (rows D1-D7 of the hot path), sm_100a.
//
//   PAPER.md §3.3: scores in latent space  s_t = q~ . L_k[t],  q~ = sm_scale q B_k^T  (no RoPE on
//   this path, A1), and the value side reordered as (p L_v) B_v  ("(p V') U_V").
//   PAPER.md A.6 L627: stack p over heads so that p L_v is ONE GEMM  P[H_q x T] . L_v[T x r_v]  -> tensor cores.
//   PAPER.md Eq.12 L208 / A.6 L625: latents are dequantised in registers, never materialised.
//
// One CTA per SM walks a contiguous page range of one sequence (split-K).  16 warps = two independent groups of
// 8 warps; group A takes the even pages of the range, group B the odd ones, each with its own running (m, l, acc)
// and ONE named barrier per page, so that one group's QK/softmax phase overlaps the other's PV phase.  The groups
// are merged in shared memory at the end.  Pages arrive in a shared-memory ring by cp.async.bulk + one "full"
// mbarrier per stage (a page is one contiguous byte range by construction of the format); a stage is refilled by
// whichever warp of the consuming group finishes its PV phase last (a shared-memory ticket), so no warp ever
// blocks on behalf of the ring.
// The latent-space query image (row D1, qproj_kernel) arrives by one more bulk copy.  Per page and group:
//   QK       warp w scores "quad" w (4 query heads) against all 64 tokens on mma.sync m16n8k16:
//            S^T[tokens x (head, hi/lo)] = L_k[tokens x ch] . q~^T.  The latent query is an fp16 hi+lo pair in
//            two MMA columns per head, so hi+lo meets in one thread and the score keeps fp32 accuracy;
//            int4/int8 fields go to fp16 by the magic-number lop3/prmt trick (exact); per-token scales
//            multiply the fp32 sums.  With G < 4 several KV heads feed one quad (zero columns elsewhere).
//   softmax  in registers: page maximum by 3 shuffles, running (m, l) per thread; the running maximum is only
//            moved when a page exceeds it by more than 2^TAU (lazy rescale), P -> fp16 with a 2^8 offset; an 8x8
//            movmatrix transpose turns the accumulator layout into the B fragments of the PV product, which
//            go to a double-buffered 4 KB exchange area (the only cross-warp traffic).
//   PV       after the barrier, warp w owns value channels [16(w+8a), +16): O^T[ch x heads] += L_v^T[ch x tok] . P^T,
//            L_v channel-major so that a 32-bit word holds consecutive tokens of one channel = the A
//            fragment's k pairs; value scales are applied element-wise in fp16 (c*s, one rounding).
//   The row of the QK tile that holds token t is chosen so that the transposed P lands in the token order
//   the dequantised value words produce (no shuffles on the value side).
// The partial (m, l, acc[H_q x r_v]) goes to the workspace; combine_kernel merges and up-projects.
#include <stdlib.h>
#include <string.h>

#include "append_small.cuh"
#include "decode_common.cuh"
#include "decode_plan.h"


namespace {

constexpr int GW = 8;                     // warps per group
constexpr int NG_MAX = 2;                 // groups per CTA
constexpr int BAR_ALL = 8;                // named barrier of all warps (1..NG are the groups' own)
constexpr int TBL_SMEM = 256;             // block-table entries of the CTA's range kept in shared memory
constexpr int PTOK = 64;         // tokens per page on this path
constexpr float P_OFFSET = 8.f;  // P is stored as 2^(s - m + 8) in fp16 (keeps small weights normal)
constexpr float TAU = 6.f;       // the running maximum may lag the true one by 2^TAU: P <= 2^14
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
// same with an L2 evict-first hint: the cache pages are read exactly once per step; without the hint the stream
// (134 MB on C2 against 126 MB of L2) evicts everything else the step keeps in L2 -- factors, query image, split-K
// partials and the kernel's own instruction lines
__device__ __forceinline__ uint64_t l2_evict_first_policy() {
  uint64_t pol;
  asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
  return pol;
}
__device__ __forceinline__ void bulk_g2s_stream(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
      "l"(src), "r"(bytes), "r"(bar), "l"(pol)
      : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bar_sync(int id, int count) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(count) : "memory");
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
// same, D = A.B + (c0, c1, c0, c1): starts an accumulator from a per-column constant without register moves
__device__ __forceinline__ void mma16816_init(float (&d)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3, uint32_t b0,
                                              uint32_t b1, float c0, float c1) {
  asm volatile(
      "mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%10,%11,%10,%11};"
      : "=f"(d[0]), "=f"(d[1]), "=f"(d[2]), "=f"(d[3])
      : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1), "f"(c0), "f"(c1));
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
// D1: latent-space query image.  grid (H_kv, batch), 256 threads; one warp per latent channel at a time, the
// B_k row read coalesced (8 halves per lane), 4 query heads per pass, warp-shuffle reduction.
// q~ = sm_scale * log2e * q B_k^T in fp32, split into an fp16 hi+lo pair and laid out as the B fragments of
// the QK MMAs (see DecodePlan).  KV head g's G query heads sit in columns 2*((g*G + i) mod 4) + {hi, lo};
// the other columns are zero.  Per sequence the output is  [image: n_qsteps * 256 B][kcst: H_kv * 8 fp32],
// kcst = accumulator start values of the quantised QK blocks (see qk_block below).
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void qproj_body(const StarkvLayout& L, const DecodePlan& PL, const __half* __restrict__ q,
                                           const __half* __restrict__ B_k, uint8_t* __restrict__ qimg_all, size_t qimg_stride,
                                           int g, int b, float (*qt)[4] /* [256][4] shared: q~[ch][i] */) {
  const int G = L.group, dh = L.head_dim, r = L.rank_k[g];
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const bool act = lane * 8 < dh;
  float qv[4][8];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    uint4 x = make_uint4(0, 0, 0, 0);
    if (i < G && act) x = *reinterpret_cast<const uint4*>(q + ((size_t)b * L.n_q_heads + g * G + i) * dh + lane * 8);
    const float2 a = h2_to_f2(x.x), c = h2_to_f2(x.y), d = h2_to_f2(x.z), e = h2_to_f2(x.w);
    qv[i][0] = a.x; qv[i][1] = a.y; qv[i][2] = c.x; qv[i][3] = c.y;
    qv[i][4] = d.x; qv[i][5] = d.y; qv[i][6] = e.x; qv[i][7] = e.y;
  }
  const float qscale = L.sm_scale * kLog2e;
  constexpr int QU = 4;                        // channels per warp in flight
  for (int ch0 = 0; ch0 < r; ch0 += 8 * QU) {
    float a[QU][4];
#pragma unroll
    for (int u = 0; u < QU; ++u) {
      const int ch = ch0 + warp + 8 * u;
      uint4 x = make_uint4(0, 0, 0, 0);
      if (ch < r && act) x = *reinterpret_cast<const uint4*>(B_k + (size_t)(L.koff[g] + ch) * dh + lane * 8);
      const float2 b0 = h2_to_f2(x.x), b1 = h2_to_f2(x.y), b2 = h2_to_f2(x.z), b3 = h2_to_f2(x.w);
#pragma unroll
      for (int i = 0; i < 4; ++i) {
        float s = qv[i][0] * b0.x;
        s = fmaf(qv[i][1], b0.y, s); s = fmaf(qv[i][2], b1.x, s); s = fmaf(qv[i][3], b1.y, s);
        s = fmaf(qv[i][4], b2.x, s); s = fmaf(qv[i][5], b2.y, s); s = fmaf(qv[i][6], b3.x, s);
        a[u][i] = fmaf(qv[i][7], b3.y, s);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1)
#pragma unroll
      for (int u = 0; u < QU; ++u)
#pragma unroll
        for (int i = 0; i < 4; ++i) a[u][i] += __shfl_xor_sync(0xffffffffu, a[u][i], o);
    if (lane == 0) {
#pragma unroll
      for (int u = 0; u < QU; ++u) {
        const int ch = ch0 + warp + 8 * u;
        if (ch < r) *reinterpret_cast<float4*>(qt[ch]) = make_float4(a[u][0] * qscale, a[u][1] * qscale, a[u][2] * qscale, a[u][3] * qscale);
      }
    }
  }
  __syncthreads();
  const int n_hi = L.k_hi_n[g], n_lo = L.k_lo_n[g];
  const int mh = L.bits_hi == 4 ? 2 * ((n_hi + 31) >> 5) : (n_hi + 15) >> 4;
  const int s0 = PL.qstep_begin[g], steps = PL.qstep_begin[g + 1] - s0;
  uint8_t* out_b = qimg_all + (size_t)b * qimg_stride;
  uint32_t* dst = reinterpret_cast<uint32_t*>(out_b) + (size_t)s0 * 64;
  for (int wi = tid; wi < steps * 64; wi += 256) {
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
        const int ch = chunk * (bits == 4 ? 32 : 16) + sk_k_to_channel(bits, m, k);
        if (ch >= n) continue;
        // the odd nibble of a 4-bit byte reaches the MMA as 16u: take the 16 out of its query column
        const float a = qt[(blk ? n_hi : 0) + ch][i] * ((bits == 4 && (ch & 1)) ? 0.0625f : 1.f);
        const __half hi = __float2half_rn(a);
        const __half v = hilo ? __float2half_rn(a - __half2float(hi)) : hi;
        word |= (uint32_t)__half_as_ushort(v) << (16 * e);
      }
    }
    dst[wi] = word;
  }
  // accumulator start values of the quantised QK blocks: -2^(b-1) * 2^-24 * sum_c q~_c over the block, with q~_c
  // exactly as the image holds it (fp16 hi + lo, power-of-two channel factor undone).  One warp per (block, column).
  if (warp < 8) {
    const int blk = warp >> 2, jq = warp & 3;
    const int i = jq - ((g * G) & 3);
    float Q = 0.f;
    const int n = blk ? n_lo : n_hi, bits = blk ? L.bits_lo : L.bits_hi;
    if (i >= 0 && i < G && bits != 16) {
      for (int ch = lane; ch < n; ch += 32) {
        const bool odd4 = bits == 4 && (ch & 1);
        const float a = qt[(blk ? n_hi : 0) + ch][i] * (odd4 ? 0.0625f : 1.f);
        const __half hi = __float2half_rn(a);
        const __half lo = __float2half_rn(a - __half2float(hi));
        Q += (__half2float(hi) + __half2float(lo)) * (odd4 ? 16.f : 1.f);
      }
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) Q += __shfl_xor_sync(0xffffffffu, Q, o);
    if (lane == 0)
      reinterpret_cast<float*>(out_b + PL.qimg_bytes)[g * 8 + warp] =
          bits == 16 ? 0.f : -(float)(1 << (bits - 1)) * 5.9604644775390625e-8f * Q;
  }
}

__global__ void __launch_bounds__(256) qproj_kernel(const __grid_constant__ StarkvLayout L,
                                                    const __grid_constant__ DecodePlan PL, const __half* __restrict__ q,
                                                    const __half* __restrict__ B_k, uint8_t* __restrict__ qimg_all,
                                                    size_t qimg_stride) {
  __shared__ float qt[256][4];
  sk_pdl_enter();
  qproj_body(L, PL, q, B_k, qimg_all, qimg_stride, blockIdx.x, blockIdx.y, qt);
}

// First launch of a fused decode step on this file's kernels (starkv_decode_step): the query image and the
// compress-on-append of the step's new tokens are independent, so they share one grid -- blocks [0, n_qp) build the
// image, the rest run the one-launch append (append_small.cuh).  Both finish before the decode kernel's
// griddepcontrol.wait returns.
static_assert(APS_THREADS == 256 && APS_SM_FLOATS >= 256 * 4, "the two bodies share a block size and the shared memory");
template <bool FUSED>
__global__ void __launch_bounds__(256) step_pre_fast_kernel(const __grid_constant__ StarkvLayout L,
                                                            const __grid_constant__ DecodePlan PL, const __half* __restrict__ q,
                                                            const __half* __restrict__ B_k, uint8_t* __restrict__ qimg_all,
                                                            size_t qimg_stride, int n_qp,
                                                            const __grid_constant__ AppendSmallArgs a) {
  __shared__ __align__(16) float sm[APS_SM_FLOATS];
  sk_pdl_enter();
  const int i = blockIdx.x;
  if (i < n_qp) {
    qproj_body(L, PL, q, B_k, qimg_all, qimg_stride, i % L.n_kv_heads, i / L.n_kv_heads, reinterpret_cast<float (*)[4]>(sm));
  } else {
    const int j = i - n_qp;
    append_small_body<FUSED>(L, a, j % a.n_tiles, j / a.n_tiles, sm);
  }
}

// ---------------------------------------------------------------------------------------------
// QK of one precision block of one KV head for the warp's 64 tokens (4 m-tiles of 16 rows).
// Row r of m-tile s holds token  tb(r & 7) + s*TS + 8*(r >> 3)  with tb / TS chosen per mode so that the
// movmatrix transpose of P yields the k order of the PV A fragments (see the header comment):
//   quantised: tb(R) = 16(R>>1) + 4(R&1), TS = 1     fp16: tb(R) = 16(R>>1) + (R&1), TS = 2
// p0 = this lane's first byte of row tb of the block; qi = this lane's B fragments of the block's q steps.
// There is no ragged-chunk predicate: lanes past the block end read the next row / block (always inside the
// page and finite: a tail page is sanitised first) against zero query columns.
//
// Integer fields are NOT converted to fp16 numbers with a bias: the offset-binary field u sits in the low
// mantissa bits of an fp16 SUBNORMAL (u * 2^-24; the odd nibbles of a 4-bit byte as 16u * 2^-24), which the
// tensor core multiplies exactly.  The factor 16 of the odd 4-bit channels is taken out of their query
// columns, the offset 2^(b-1) becomes the constant  -2^(b-1) sum_c q~_c  the accumulator starts from, and the
// common 2^-24 is undone when the score is exponentiated.  One PRMT / LOP3 per two fields, nothing else.
// ---------------------------------------------------------------------------------------------
template <bool QUANT>
__device__ __forceinline__ int tok_base(int R) { return QUANT ? 16 * (R >> 1) + 4 * (R & 1) : 16 * (R >> 1) + (R & 1); }

// Each function OVERWRITES acc: the first chunk's MMAs start from the per-column constant (cinit, 0).
__device__ __forceinline__ void qk_f16(float (&acc)[4][4], const uint8_t* __restrict__ p0, int rowbytes, int nch,
                                       const uint2* __restrict__ qi, float cinit) {
  const int rb2 = 2 * rowbytes, rb8 = 8 * rowbytes;
  {
    const uint2 bf = *qi;
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rb2;
      const uint2 x0 = *reinterpret_cast<const uint2*>(p);
      const uint2 x1 = *reinterpret_cast<const uint2*>(p + rb8);
      mma16816_init(acc[s], x0.x, x1.x, x0.y, x1.y, bf.x, bf.y, cinit, 0.f);
    }
  }
  for (int c = 1; c < nch; ++c) {
    p0 += 32; qi += 32;
    const uint2 bf = *qi;
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rb2;
      const uint2 x0 = *reinterpret_cast<const uint2*>(p);
      const uint2 x1 = *reinterpret_cast<const uint2*>(p + rb8);
      mma16816(acc[s], x0.x, x1.x, x0.y, x1.y, bf.x, bf.y);
    }
  }
}

__device__ __forceinline__ void qk_i8(float (&acc)[4][4], const uint8_t* __restrict__ p0, int rowbytes, int nch,
                                      const uint2* __restrict__ qi, float cinit) {
  const int rb8 = 8 * rowbytes;
  {
    const uint2 bf = *qi;
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rowbytes;
      const uint32_t w0 = *reinterpret_cast<const uint32_t*>(p);
      const uint32_t w1 = *reinterpret_cast<const uint32_t*>(p + rb8);
      mma16816_init(acc[s], prmt(w0, 0u, 0x4140u), prmt(w1, 0u, 0x4140u), prmt(w0, 0u, 0x4342u), prmt(w1, 0u, 0x4342u),
                    bf.x, bf.y, cinit, 0.f);
    }
  }
  for (int c = 1; c < nch; ++c) {
    p0 += 16; qi += 32;
    const uint2 bf = *qi;
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rowbytes;
      const uint32_t w0 = *reinterpret_cast<const uint32_t*>(p);
      const uint32_t w1 = *reinterpret_cast<const uint32_t*>(p + rb8);
      mma16816(acc[s], prmt(w0, 0u, 0x4140u), prmt(w1, 0u, 0x4140u), prmt(w0, 0u, 0x4342u), prmt(w1, 0u, 0x4342u), bf.x,
               bf.y);
    }
  }
}

__device__ __forceinline__ void qk_i4(float (&acc)[4][4], const uint8_t* __restrict__ p0, int rowbytes, int nch,
                                      const uint2* __restrict__ qi, float cinit) {
  const int rb8 = 8 * rowbytes;
  {
    const uint2 bf0 = qi[0], bf1 = qi[32];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rowbytes;
      const uint32_t w0 = *reinterpret_cast<const uint32_t*>(p);
      const uint32_t w1 = *reinterpret_cast<const uint32_t*>(p + rb8);
      const uint32_t v0 = w0 >> 8, v1 = w1 >> 8;
      mma16816_init(acc[s], w0 & 0x000f000fu, w1 & 0x000f000fu, w0 & 0x00f000f0u, w1 & 0x00f000f0u, bf0.x, bf0.y, cinit, 0.f);
      mma16816(acc[s], v0 & 0x000f000fu, v1 & 0x000f000fu, v0 & 0x00f000f0u, v1 & 0x00f000f0u, bf1.x, bf1.y);
    }
  }
  for (int c = 1; c < nch; ++c) {
    p0 += 16; qi += 64;
    const uint2 bf0 = qi[0], bf1 = qi[32];
#pragma unroll
    for (int s = 0; s < 4; ++s) {
      const uint8_t* p = p0 + s * rowbytes;
      const uint32_t w0 = *reinterpret_cast<const uint32_t*>(p);
      const uint32_t w1 = *reinterpret_cast<const uint32_t*>(p + rb8);
      const uint32_t v0 = w0 >> 8, v1 = w1 >> 8;
      mma16816(acc[s], w0 & 0x000f000fu, w1 & 0x000f000fu, w0 & 0x00f000f0u, w1 & 0x00f000f0u, bf0.x, bf0.y);
      mma16816(acc[s], v0 & 0x000f000fu, v1 & 0x000f000fu, v0 & 0x00f000f0u, v1 & 0x00f000f0u, bf1.x, bf1.y);
    }
  }
}

template <int BITS>
__device__ __forceinline__ void qk_block(float (&acc)[4][4], const uint8_t* __restrict__ blk, int n, int tb, int j,
                                         const uint2* __restrict__ qi, float cinit) {
  if (BITS == 16) {
    qk_f16(acc, blk + tb * (2 * n) + 8 * j, 2 * n, (n + 15) >> 4, qi, cinit);
  } else if (BITS == 8) {
    qk_i8(acc, blk + tb * n + 4 * j, n, (n + 15) >> 4, qi, cinit);
  } else {
    qk_i4(acc, blk + tb * (n >> 1) + 4 * j, n >> 1, (n + 31) >> 5, qi, cinit);
  }
}

// ---------------------------------------------------------------------------------------------
// PV of one 16-channel m-tile over the page's 64 tokens (4 k-steps) against all NT head tiles.
//   vrow0/vrow1: this thread's two channel rows (R, R+8) of the value block, already clamped
//   sc0/sc2    : value scales as (t, t+4) fp16 pairs of this thread's 16 tokens (quantised modes)
//   pf_lane    : this lane's P^T B fragments in the exchange buffer, [k-step pair][head tile][lane] uint4 =
//                (b0, b1 of step 2sp, b0, b1 of step 2sp+1)
// ---------------------------------------------------------------------------------------------
template <int BITS, int NT>
__device__ __forceinline__ void pv_tile(float (&acc)[NT][4], const uint8_t* __restrict__ vrow0,
                                        const uint8_t* __restrict__ vrow1, bool dead0, bool dead1,
                                        const uint32_t (&sc0)[4], const uint32_t (&sc2)[4],
                                        const uint4* __restrict__ pf_lane, int j) {
  uint32_t A0[4], A1[4], A2[4], A3[4];
  if (BITS == 4) {
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
  } else if (BITS == 8) {
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
  // P^T fragments are read from the exchange buffer right before use (4 KB, L1-resident in effect): keeping all
  // of them in registers across the dequantisation would cost 32 registers per thread
#pragma unroll
  for (int sp = 0; sp < 2; ++sp)
#pragma unroll
    for (int c = 0; c < NT; ++c) {
      const uint4 f = pf_lane[(sp * 4 + c) * 32];
      mma16816(acc[c], A0[2 * sp], A1[2 * sp], A2[2 * sp], A3[2 * sp], f.x, f.y);
      mma16816(acc[c], A0[2 * sp + 1], A1[2 * sp + 1], A2[2 * sp + 1], A3[2 * sp + 1], f.z, f.w);
    }
}

__device__ __forceinline__ float ex2(float x) {
  float r;
  asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
  return r;
}

// acc += (chi.x + chi.y pairs) * per-token scale   (scales: 4 fp16 of rows tb.., 4 of rows tb+8..)
__device__ __forceinline__ void apply_k_scales(float (&sc)[4][2], const float (&chi)[4][4], const __half* __restrict__ ksc) {
  const uint2 h0 = *reinterpret_cast<const uint2*>(ksc), h1 = *reinterpret_cast<const uint2*>(ksc + 8);
  const float2 a01 = h2_to_f2(h0.x), a23 = h2_to_f2(h0.y), b01 = h2_to_f2(h1.x), b23 = h2_to_f2(h1.y);
  sc[0][0] = fmaf(chi[0][0] + chi[0][1], a01.x, sc[0][0]); sc[0][1] = fmaf(chi[0][2] + chi[0][3], b01.x, sc[0][1]);
  sc[1][0] = fmaf(chi[1][0] + chi[1][1], a01.y, sc[1][0]); sc[1][1] = fmaf(chi[1][2] + chi[1][3], b01.y, sc[1][1]);
  sc[2][0] = fmaf(chi[2][0] + chi[2][1], a23.x, sc[2][0]); sc[2][1] = fmaf(chi[2][2] + chi[2][3], b23.x, sc[2][1]);
  sc[3][0] = fmaf(chi[3][0] + chi[3][1], a23.y, sc[3][0]); sc[3][1] = fmaf(chi[3][2] + chi[3][3], b23.y, sc[3][1]);
}

// ---------------------------------------------------------------------------------------------
// QK + softmax of one page for one warp's quad.  Leaves P (fp16, transposed into PV B-fragment words) in the
// group's exchange buffer, alpha per head in `al`, a "some head rescaled" flag, and updates the running (m, l).
//   BH / BL: bit widths of the leading / trailing blocks (16/16 = fp16 latents).
//   kcst: per (KV head, block, quad column) accumulator start value (the offset term, see above).
// ---------------------------------------------------------------------------------------------
//   UM: P goes out as the K-major canonical (no-swizzle, 8 x 16-byte core matrices) B operand of the tcgen05 PV
//       product instead: element (head, token) at (head >> 3) * 1024 + (token >> 3) * 128 + (head & 7) * 16 +
//       (token & 7) * 2; no transpose, this thread's 4 + 4 consecutive tokens of head 4 gw + j are two 8-byte stores.
template <int BH, int BL, bool UM = false>
__device__ __forceinline__ void score_page(const StarkvLayout& L, const DecodePlan& PL, const uint8_t* __restrict__ pg,
                                           const uint2* __restrict__ qimg_lane, const float* __restrict__ kcst, int kv0,
                                           int kv1, int nvalid, int R, int j, int gw, float& m_run, float& l_run,
                                           uint8_t* __restrict__ Pb, int p_thr_off, float* __restrict__ al,
                                           uint8_t* __restrict__ flag) {
  constexpr bool QUANT = BH != 16;
  constexpr int TS = QUANT ? 1 : 2;
  constexpr float kUnscale = QUANT ? 16777216.f : 1.f;   // 2^24: undoes the subnormal field scaling
  const int tb = tok_base<QUANT>(R);
  float sc[4][2];
#pragma unroll
  for (int s = 0; s < 4; ++s) sc[s][0] = sc[s][1] = 0.f;
  for (int g = kv0; g < kv1; ++g) {
    const uint2* qi = qimg_lane + PL.qstep_begin[g] * 32;
    const int n_hi = L.k_hi_n[g];
    float chi[4][4];
    if (!QUANT) {
      qk_block<16>(chi, pg + L.k_hi_off[g], n_hi, tb, j, qi, 0.f);
#pragma unroll
      for (int s = 0; s < 4; ++s) {
        sc[s][0] += chi[s][0] + chi[s][1];
        sc[s][1] += chi[s][2] + chi[s][3];
      }
    } else {
      const __half* ksc = reinterpret_cast<const __half*>(pg + L.k_scale_off) + (g * 2) * PTOK + tb;
      qk_block<BH>(chi, pg + L.k_hi_off[g], n_hi, tb, j, qi, kcst[g * 8 + j]);
      apply_k_scales(sc, chi, ksc);
      const int n_lo = L.k_lo_n[g];
      if (n_lo > 0) {
        qi += 32 * (BH == 4 ? 2 * ((n_hi + 31) >> 5) : (n_hi + 15) >> 4);
        qk_block<BL>(chi, pg + L.k_lo_off[g], n_lo, tb, j, qi, kcst[g * 8 + 4 + j]);
        apply_k_scales(sc, chi, ksc + PTOK);
      }
    }
  }
  if (nvalid < PTOK) {
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
  mx *= kUnscale;
  // lazy rescale: move the running maximum only when the page exceeds it by more than TAU
  // (first page: m_run = -inf, mx finite because slot 0 of every page in range is valid)
  const bool up = mx > m_run + TAU;
  const float m_new = up ? mx : m_run;
  const float alpha = up ? ex2(m_run - m_new) : 1.f;   // 0 on the first page
  const float sh = P_OFFSET - m_new;
  float sum = 0.f;
#pragma unroll
  for (int s = 0; s < 4; ++s) {
    sc[s][0] = ex2(fmaf(sc[s][0], kUnscale, sh));   // -inf -> 0
    sc[s][1] = ex2(fmaf(sc[s][1], kUnscale, sh));
    sum += sc[s][0] + sc[s][1];
  }
  l_run = fmaf(l_run, alpha, sum);
  m_run = m_new;
  if (UM) {
    static_assert(!UM || QUANT, "tcgen05 PV is built for the quantised modes (token order tb + s)");
#pragma unroll
    for (int be = 0; be < 2; ++be)
      *reinterpret_cast<uint2*>(Pb + p_thr_off + be * 128) =
          make_uint2(pack_h2(sc[0][be], sc[1][be]), pack_h2(sc[2][be], sc[3][be]));
  } else {
#pragma unroll
    for (int u = 0; u < 2; ++u)
#pragma unroll
      for (int be = 0; be < 2; ++be) {
        const uint32_t y = movmatrix_trans(pack_h2(sc[2 * u][be], sc[2 * u + 1][be]));
        *reinterpret_cast<uint32_t*>(Pb + p_thr_off + u * (4 * 32 * 16) + be * 4) = y;
      }
  }
  const bool any_up = __any_sync(0xffffffffu, up);
  if (R == 0) al[4 * gw + j] = alpha;
  if ((R | j) == 0) flag[gw] = any_up ? 1 : 0;
}

// ---------------------------------------------------------------------------------------------
// Main kernel.  grid (n_splits, batch), NG groups of 8 warps (NG = 2: 512 threads, 128 registers; NG = 3: 768
// threads, 80 registers -- more warps to hide the dequantisation latency of the integer modes).
//   BH/BL  bit widths of the leading / trailing blocks (16/16 = fp16 latents)
//   NT  head tiles of 8   MT  value m-tiles (16 channels) per warp
// ---------------------------------------------------------------------------------------------
template <int BH, int BL, int NT, int MT, int NG>
__global__ void __launch_bounds__(NG * GW * 32, 1) decode_fast_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ DecodePlan PL, const uint8_t* __restrict__ qimg_all,
    size_t qimg_stride, const uint8_t* __restrict__ pool, const int32_t* __restrict__ table, int max_pages,
    const int32_t* __restrict__ seq_lens, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(128) uint8_t smem[];
  constexpr bool QUANT = BH != 16;
  constexpr int NTHREADS = NG * GW * 32;

  const int tid = threadIdx.x, lane = tid & 31;
  // warp index as a value the compiler knows to be warp-uniform (shuffle from lane 0): group and ring addressing
  // derived from it can live in uniform registers
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int j = lane & 3, R = lane >> 2;
  const int split = blockIdx.x, b = blockIdx.y;
  sk_pdl_trigger();
  // Nothing global is read before the dependency wait: seq_lens and the block table may have been written by a kernel the
  // caller enqueued right before this call (CUDA makes a predecessor's writes visible only after griddepcontrol.wait).
  sk_pdl_wait();
  const int len = seq_lens[b];
  int n_pages = len > 0 ? (len + PTOK - 1) / PTOK : 0;
  if (n_pages > max_pages) n_pages = max_pages;   // (a length past the table is a caller error: memory-safe, result undefined)
  int p0, p1;
  sk_split_range(n_pages, n_splits, 1, split, &p0, &p1);
  const int n_it = p1 - p0;
  const size_t pstride = sk_part_stride(L.rank_v);
  float* my_parts = parts + ((size_t)b * n_splits + split) * L.n_q_heads * pstride;

  if (n_it <= 0) {   // empty range (CTA-uniform): neutral partial
    sk_pdl_wait();
    for (int i = tid; i < L.n_q_heads * (int)pstride; i += NTHREADS) {
      const int c = i % (int)pstride;
      my_parts[i] = c == 0 ? -INFINITY : 0.f;
    }
    return;
  }

  uint8_t* stage_base = smem + PL.off_stage;
  const int nstage = PL.nstage;
  const uint32_t full0 = smem_u32(smem + PL.off_bar);   // full[nstage], then qbar
  const uint32_t qbar = full0 + 8 * nstage;
  int* done = reinterpret_cast<int*>(smem + PL.off_bar + 8 * nstage + 8);   // [nstage] warps finished with the stage
  volatile int* issued = done + nstage;                                 // [nstage] ring iteration loaded into the stage
  int32_t* tbl_s = reinterpret_cast<int32_t*>(smem + PL.off_tbl);       // first TBL_SMEM table entries of the range
  const uint32_t page_bytes = (uint32_t)L.page_bytes;
  const int32_t* my_table = table + (size_t)b * max_pages + p0;

  auto issue = [&](int it, int page) {   // D2: one page -> ring stage (single thread)
    const int st = it % nstage;
    const uint32_t bar = full0 + 8 * st;
    mbar_expect_tx(bar, page_bytes);
    __threadfence_block();   // the barrier is armed before any consumer can see the stage as issued
    issued[st] = it;
    bulk_g2s_stream(smem_u32(stage_base + (size_t)st * page_bytes), pool + (size_t)max(page, 0) * page_bytes, page_bytes, bar,
                    l2_evict_first_policy());
  };
  if (tid == 0) {
    for (int s = 0; s < nstage; ++s) {
      mbar_init(full0 + 8 * s, 1);
      done[s] = 0;
      issued[s] = -1;
    }
    mbar_init(qbar, 1);
    fence_barrier_init();
    int pgs[8];
#pragma unroll
    for (int s = 0; s < 8; ++s) pgs[s] = s < min(nstage, n_it) ? my_table[s] : 0;
    sk_pdl_wait();
    const uint32_t qbytes = (uint32_t)(PL.qimg_bytes + L.n_kv_heads * 32);   // image + accumulator start values
    mbar_expect_tx(qbar, qbytes);
    bulk_g2s(smem_u32(smem + PL.off_qimg), qimg_all + (size_t)b * qimg_stride, qbytes, qbar);
#pragma unroll
    for (int s = 0; s < 8; ++s)
      if (s < min(nstage, n_it)) issue(s, pgs[s]);
  }
  for (int i = tid; i < min(n_it, TBL_SMEM); i += NTHREADS) tbl_s[i] = my_table[i];
  sk_pdl_wait();   // (thread 0 has waited already; a second wait returns at once)
  __syncthreads();

  // ================= consumers =================
  const int grp = warp >> 3, gw = warp & (GW - 1);
  {
    uint4* pz = reinterpret_cast<uint4*>(smem + PL.off_p);
    for (int i = tid; i < NG * 2 * P_BUF_BYTES / 16; i += NTHREADS) pz[i] = make_uint4(0, 0, 0, 0);
    if (tid < NG * 64) reinterpret_cast<float*>(smem + PL.off_alpha)[tid] = 1.f;
    if (tid < NG * 4) reinterpret_cast<uint32_t*>(smem + PL.off_flag)[tid] = 0;
  }
  bar_sync(BAR_ALL, NTHREADS);
  mbar_wait(qbar, 0);

  const uint2* qimg_lane = reinterpret_cast<const uint2*>(smem + PL.off_qimg) + lane;
  const float* kcst = reinterpret_cast<const float*>(smem + PL.off_kcst);
  uint8_t* Pm = smem + PL.off_p + grp * 2 * P_BUF_BYTES;                        // [2][P_BUF_BYTES]
  float* alpha_s = reinterpret_cast<float*>(smem + PL.off_alpha) + grp * 64;    // [2][32]
  uint8_t* flag_s = smem + PL.off_flag + grp * 16;                              // [2][8]

  // this warp's quad (QK + softmax) and where its transposed P words go
  const bool has_quad = gw < PL.nq;
  const int kv0 = gw * PL.kv_per_quad;
  const int kv1 = min(kv0 + PL.kv_per_quad, L.n_kv_heads);
  // after the transpose lane (R' = 2j'' + e', j) holds the b-register of head j'' for k-step 2u + e';
  // its consumer is lane (4*(quad&1) + j'', j) of head tile quad>>1
  const int p_thr_off = (((gw >> 1) * 32 + (4 * (gw & 1) + (R >> 1)) * 4 + j) << 4) + ((R & 1) << 3);
  float m_run = -INFINITY, l_run = 0.f;

  float acc[MT][NT][4];
#pragma unroll
  for (int a = 0; a < MT; ++a)
#pragma unroll
    for (int c = 0; c < NT; ++c)
#pragma unroll
      for (int e = 0; e < 4; ++e) acc[a][c][e] = 0.f;
  int st = grp % nstage, use = grp / nstage;   // ring stage and use count of iteration `it`, kept incrementally
  int gi = 0;                                  // this group's iteration count
  for (int it = grp; it < n_it; it += NG, ++gi) {
    uint8_t* pg = stage_base + (size_t)st * page_bytes;
    const int nvalid = len - (p0 + it) * PTOK;   // >= 1
    const int buf = gi & 1;
    uint8_t* Pb = Pm + buf * P_BUF_BYTES;
    float* al = alpha_s + buf * 32;
    uint8_t* fl = flag_s + buf * 8;
    // With an odd ring depth the two groups share stages and may be a whole barrier phase apart, which a parity
    // wait cannot tell from "done": first wait until the stage has been armed for THIS iteration.
    if (lane == 0)
      while (issued[st] != it) {}
    __syncwarp();
    mbar_wait(full0 + 8 * st, (uint32_t)(use & 1));

    if (nvalid < PTOK) {   // tail page: slots past the sequence end may hold any bits.  Zero their key rows (the
                           // unpredicated QK loads may touch them) and neutralise their value data, then sync.
      const int gt = tid & 255;
      for (int g = 0; g < L.n_kv_heads; ++g) {
        for (int blk = 0; blk < (QUANT ? 2 : 1); ++blk) {
          const int n = blk ? L.k_lo_n[g] : L.k_hi_n[g];
          const int rowb = n * (blk ? BL : BH) / 8;   // multiple of 4
          uint32_t* dst = reinterpret_cast<uint32_t*>(pg + (blk ? L.k_lo_off[g] : L.k_hi_off[g]) + nvalid * rowb);
          for (int i = gt; i < (PTOK - nvalid) * rowb / 4; i += 256) dst[i] = 0;
        }
      }
      if (QUANT) {
        if (gt < 2 * PTOK && (gt & (PTOK - 1)) >= nvalid) reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[gt] = 0;
      } else {
        const int nbad = PTOK - nvalid;
        for (int i = gt; i < L.rank_v * nbad; i += 256)
          reinterpret_cast<uint16_t*>(pg + L.v_hi_off)[(i / nbad) * PTOK + nvalid + i % nbad] = 0;
      }
      bar_sync(1 + grp, GW * 32);
    }

    // ================= QK + softmax for this warp's quad =================
    if (has_quad)
      score_page<BH, BL>(L, PL, pg, qimg_lane, kcst, kv0, kv1, nvalid, R, j, gw, m_run, l_run, Pb, p_thr_off, al, fl);
    bar_sync(1 + grp, GW * 32);   // P and alpha of this page complete

    // ================= PV: O^T += L_v^T . P^T =================
    {
      const uint2 f8 = *reinterpret_cast<const uint2*>(fl);
      if ((f8.x | f8.y) != 0) {   // some head moved its maximum on this page (rare after the first pages)
#pragma unroll
        for (int c = 0; c < NT; ++c) {
          const float2 alv = *reinterpret_cast<const float2*>(al + 8 * c + 2 * j);
#pragma unroll
          for (int a = 0; a < MT; ++a) {
            acc[a][c][0] *= alv.x; acc[a][c][1] *= alv.y; acc[a][c][2] *= alv.x; acc[a][c][3] *= alv.y;
          }
        }
      }
    }
    const uint4* pf = reinterpret_cast<const uint4*>(Pb) + lane;   // [k-step pair][head tile][lane]
    int cur_blk = -1;
    uint32_t sc0[4] = {0, 0, 0, 0}, sc2[4] = {0, 0, 0, 0};
#pragma unroll
    for (int a = 0; a < MT; ++a) {
      const int tile = gw + GW * a;
      if (tile >= PL.v_tiles) break;
      const int blk = tile >= PL.v_tiles_hi ? 1 : 0;
      const int ch0 = 16 * (tile - (blk ? PL.v_tiles_hi : 0));
      const int n = blk ? L.v_lo_n : L.v_hi_n;
      const int c0 = min(ch0 + R, n - 1), c1 = min(ch0 + R + 8, n - 1);   // clamped; dead rows zeroed in pv_tile
      const uint8_t* vb = pg + (blk ? L.v_lo_off : L.v_hi_off);
      const int rowb = PTOK * (blk ? BL : BH) / 8;
      if (QUANT && blk != cur_blk) {
        cur_blk = blk;
        const uint4* sp4 = reinterpret_cast<const uint4*>(pg + L.v_scale_off + (blk * PTOK + 16 * j) * 2);
        const uint4 u = sp4[0], v = sp4[1];
        sc0[0] = prmt(u.x, u.z, 0x5410u); sc0[1] = prmt(u.x, u.z, 0x7632u);
        sc0[2] = prmt(u.y, u.w, 0x5410u); sc0[3] = prmt(u.y, u.w, 0x7632u);
        sc2[0] = prmt(v.x, v.z, 0x5410u); sc2[1] = prmt(v.x, v.z, 0x7632u);
        sc2[2] = prmt(v.y, v.w, 0x5410u); sc2[3] = prmt(v.y, v.w, 0x7632u);
      }
      if (blk)
        pv_tile<BL, NT>(acc[a], vb + c0 * rowb, vb + c1 * rowb, ch0 + R >= n, ch0 + R + 8 >= n, sc0, sc2, pf, j);
      else
        pv_tile<BH, NT>(acc[a], vb + c0 * rowb, vb + c1 * rowb, ch0 + R >= n, ch0 + R + 8 >= n, sc0, sc2, pf, j);
    }
    __syncwarp();
    if (lane == 0) {   // the last warp of the group to finish with the stage refills it
      if (atomicAdd(&done[st], 1) == GW - 1) {
        atomicExch(&done[st], 0);
        const int nxt = it + nstage;
        if (nxt < n_it) issue(nxt, nxt < TBL_SMEM ? tbl_s[nxt] : my_table[nxt]);
      }
    }
    st += NG;
    while (st >= nstage) { st -= nstage; ++use; }
  }

  // ================= merge the groups and write the split-K partial (D7) =================
  // Stage memory is free (every issued page was consumed): it holds m[NG][32], l[NG][32] and the partial in its
  // global layout [head][4 + r_v], which is then streamed out with coalesced 16-byte stores.
  bar_sync(BAR_ALL, NTHREADS);
  float* mg = reinterpret_cast<float*>(smem + PL.off_stage);   // m at [g * 32 + head], l at [128 + g * 32 + head]
  float* ost = mg + 256;
  const int ST = (int)pstride;
  if (has_quad) {
    float lsum = l_run;
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 4);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 8);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 16);
    if (R == 0) {
      mg[grp * 32 + 4 * gw + j] = m_run;
      mg[128 + grp * 32 + 4 * gw + j] = lsum;
    }
  }
  bar_sync(BAR_ALL, NTHREADS);
  float fme[NT][2];   // this group's weight per head column: 2^(m_own - max_g m_g); group 0 always has a page
#pragma unroll
  for (int c = 0; c < NT; ++c)
#pragma unroll
    for (int e = 0; e < 2; ++e) {
      const int head = 8 * c + 2 * j + e;
      float ms = mg[head];
#pragma unroll
      for (int g = 1; g < NG; ++g) ms = fmaxf(ms, mg[g * 32 + head]);
      const float mo = mg[grp * 32 + head];
      fme[c][e] = mo == -INFINITY ? 0.f : ex2(mo - ms);
    }
  if (tid < L.n_q_heads) {
    float ms = mg[tid];
#pragma unroll
    for (int g = 1; g < NG; ++g) ms = fmaxf(ms, mg[g * 32 + tid]);
    float lm = 0.f;
#pragma unroll
    for (int g = 0; g < NG; ++g) {
      const float mo = mg[g * 32 + tid];
      lm += mo == -INFINITY ? 0.f : mg[128 + g * 32 + tid] * ex2(mo - ms);
    }
    *reinterpret_cast<float4*>(ost + tid * ST) = make_float4(ms, lm, 0.f, 0.f);
  }
#pragma unroll
  for (int pass = NG - 1; pass >= 0; --pass) {   // the last group stores, the others add one after the other
    if (grp == pass) {
#pragma unroll
      for (int a = 0; a < MT; ++a) {
        const int tile = gw + GW * a;
        if (tile < PL.v_tiles) {
          const int blk = tile >= PL.v_tiles_hi ? 1 : 0;
          const int ch0 = 16 * (tile - (blk ? PL.v_tiles_hi : 0));
          const int n = blk ? L.v_lo_n : L.v_hi_n;
          float* o0 = ost + 4 + (blk ? L.v_hi_n : 0) + ch0 + R;
#pragma unroll
          for (int c = 0; c < NT; ++c)
#pragma unroll
            for (int e = 0; e < 4; ++e) {
              const int head = 8 * c + 2 * j + (e & 1), dch = 8 * (e >> 1);
              if (head < L.n_q_heads && ch0 + R + dch < n) {
                float* o = o0 + head * ST + dch;
                const float v = acc[a][c][e] * fme[c][e & 1];
                *o = pass == NG - 1 ? v : *o + v;
              }
            }
        }
      }
    }
    bar_sync(BAR_ALL, NTHREADS);
  }
  {
    const float4* src = reinterpret_cast<const float4*>(ost);
    float4* dst = reinterpret_cast<float4*>(my_parts);
    for (int i = tid; i < L.n_q_heads * ST / 4; i += NTHREADS) dst[i] = src[i];
  }
}

// ---------------------------------------------------------------------------------------------
// tcgen05 variant of the kernel for the integer modes (rows D2-D7): QK and the softmax exactly as above, but the
// PV product  O^T[ch x heads] += L_v^T[ch x tok] . P^T[tok x heads]  runs on the 5th-generation tensor cores:
//   A = dequantised value page (c * s in fp16, one rounding, as in the mma.sync kernel), written by the group's
//       256 threads into the K-major no-swizzle canonical layout (8 channels x 8 tokens core matrices):
//       element (ch, t) at (ch >> 3) * 1024 + (t >> 3) * 128 + (ch & 7) * 16 + (t & 7) * 2  -- one 16-byte
//       LDS of packed codes -> 2 (int8) or 4 (int4) 16-byte STS, about 2 instructions per value pair;
//   B = P^T in the same layout (score_page<UM>), N = 32 heads;
//   D = fp32 accumulators in TMEM, 32 columns per 128-channel M tile and group; M = 128, N = 32, K = 16 per
//       tcgen05.mma (kind::f16, cta_group::1), 4 K steps per page, issued by one thread of the group, which then
//       commits to the group's mbarrier and refills the page's ring stage (every warp of the group is past its
//       shared-memory reads of the page at that point: no ticket).
// The lazy softmax rescale (rare after the first pages) reads, scales and writes back the TMEM tile
// (tcgen05.ld / st); the first page of a group starts its accumulators with the MMA's accumulate flag off.
// One named barrier per page and group, as before; the MMAs of page i run under the QK phase of page i + 1.
// ---------------------------------------------------------------------------------------------
constexpr int UM_ROWS = 128;                         // channels per M tile
constexpr int UM_TILE_BYTES = UM_ROWS * PTOK * 2;     // 16 KB of A per M tile and page

__device__ __forceinline__ uint64_t umma_desc_k(uint32_t saddr) {
  // SWIZZLE_NONE K-major matrix descriptor: start >> 4 | LBO (next core matrix along K) = 128 B |
  // SBO (next 8 rows) = 1024 B | version 1 (sm_100)
  return (uint64_t)((saddr & 0x3FFFF) >> 4) | ((uint64_t)(128 >> 4) << 16) | ((uint64_t)(1024 >> 4) << 32) |
         ((uint64_t)1 << 46);
}
__device__ __forceinline__ void umma_f16(uint32_t tmem_d, uint64_t da, uint64_t db, uint32_t idesc, uint32_t accum) {
  asm volatile(
      "{\n\t.reg .pred p;\n\tsetp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(tmem_d),
      "l"(da), "l"(db), "r"(idesc), "r"(accum)
      : "memory");
}
__device__ __forceinline__ void umma_commit(uint32_t bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
// one lane of a converged warp; the code around it stays warp-uniform, so that descriptor and TMEM operands computed
// from warp-uniform values live in uniform registers (no per-MMA R2UR waterfall loop)
__device__ __forceinline__ bool elect_one() {
  uint32_t p;
  asm volatile("{\n\t.reg .pred P;\n\telect.sync _|P, 0xffffffff;\n\tselp.u32 %0, 1, 0, P;\n\t}" : "=r"(p));
  return p != 0;
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tmem_ld32(uint32_t taddr, uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x32.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,"
      "%22,%23,%24,%25,%26,%27,%28,%29,%30,%31}, [%32];"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]), "=r"(v[9]),
        "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15]), "=r"(v[16]), "=r"(v[17]), "=r"(v[18]),
        "=r"(v[19]), "=r"(v[20]), "=r"(v[21]), "=r"(v[22]), "=r"(v[23]), "=r"(v[24]), "=r"(v[25]), "=r"(v[26]), "=r"(v[27]),
        "=r"(v[28]), "=r"(v[29]), "=r"(v[30]), "=r"(v[31])
      : "r"(taddr));
  asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_st32(uint32_t taddr, const uint32_t (&v)[32]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15,%16,%17,%18,%19,%20,%21,"
      "%22,%23,%24,%25,%26,%27,%28,%29,%30,%31,%32};" ::"r"(taddr),
      "r"(v[0]), "r"(v[1]), "r"(v[2]), "r"(v[3]), "r"(v[4]), "r"(v[5]), "r"(v[6]), "r"(v[7]), "r"(v[8]), "r"(v[9]), "r"(v[10]),
      "r"(v[11]), "r"(v[12]), "r"(v[13]), "r"(v[14]), "r"(v[15]), "r"(v[16]), "r"(v[17]), "r"(v[18]), "r"(v[19]), "r"(v[20]),
      "r"(v[21]), "r"(v[22]), "r"(v[23]), "r"(v[24]), "r"(v[25]), "r"(v[26]), "r"(v[27]), "r"(v[28]), "r"(v[29]), "r"(v[30]),
      "r"(v[31])
      : "memory");
  asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory");
}

// One precision block of the value page -> A operand.  Work item = one 16-byte segment of a channel row
// (32 int4 / 16 int8 slots = NTB 8-token blocks); item i -> channel 8 ((i >> 3) / SEGS) + (i & 7), segment
// (i >> 3) % SEGS, so 8 consecutive lanes write 8 consecutive channels of one token block (128 contiguous bytes,
// conflict-free) and a thread keeps its segment -- hence its scale registers -- across its items (i += 256).
template <int BITS, int NTHR = 256>
__device__ __forceinline__ void deq_block_to_a(const uint8_t* __restrict__ vb, const uint8_t* __restrict__ vsc, int n_ch,
                                               int row0, uint8_t* __restrict__ abuf, int t) {
  constexpr int SEGS = BITS / 2;   // 16-byte segments per channel row of PTOK slots
  constexpr int NTB = 8 / SEGS;    // 8-token blocks per segment
  const int n_items = n_ch * SEGS;
  if (t >= n_items) return;
  const int seg = (t >> 3) % SEGS;
  uint32_t sc[4 * NTB];            // the segment's per-token scales as natural (t, t+1) fp16 pairs
#pragma unroll
  for (int k = 0; k < NTB; ++k) {
    const uint4 u = *reinterpret_cast<const uint4*>(vsc + (seg * NTB + k) * 16);
    sc[4 * k] = u.x; sc[4 * k + 1] = u.y; sc[4 * k + 2] = u.z; sc[4 * k + 3] = u.w;
  }
  for (int i = t; i < n_items; i += NTHR) {
    const int ch = ((i >> 3) / SEGS) * 8 + (i & 7);
    const uint4 x = *reinterpret_cast<const uint4*>(vb + ch * (PTOK * BITS / 8) + seg * 16);
    const int row = row0 + ch;
    uint8_t* dst = abuf + (row >> 3) * 1024 + (seg * NTB) * 128 + (row & 7) * 16;
    if (BITS == 4) {
      const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        uint32_t h[4];
        deq4_pairs(w[k], h);   // (c0,c4), (c1,c5), (c2,c6), (c3,c7)
        uint4 o;
        o.x = h2mul(prmt(h[0], h[1], 0x5410u), sc[4 * k]);
        o.y = h2mul(prmt(h[2], h[3], 0x5410u), sc[4 * k + 1]);
        o.z = h2mul(prmt(h[0], h[1], 0x7632u), sc[4 * k + 2]);
        o.w = h2mul(prmt(h[2], h[3], 0x7632u), sc[4 * k + 3]);
        *reinterpret_cast<uint4*>(dst + k * 128) = o;
      }
    } else {
      const uint32_t w[4] = {x.x, x.y, x.z, x.w};
#pragma unroll
      for (int k = 0; k < 2; ++k) {
        uint32_t a, b, c, d;
        deq8_pairs(w[2 * k], a, b);
        deq8_pairs(w[2 * k + 1], c, d);
        uint4 o;
        o.x = h2mul(a, sc[4 * k]);
        o.y = h2mul(b, sc[4 * k + 1]);
        o.z = h2mul(c, sc[4 * k + 2]);
        o.w = h2mul(d, sc[4 * k + 3]);
        *reinterpret_cast<uint4*>(dst + k * 128) = o;
      }
    }
  }
}

template <int BH, int BL, int NG>
__global__ void __launch_bounds__(NG * GW * 32, 1) decode_tc5_kernel(
    const __grid_constant__ StarkvLayout L, const __grid_constant__ DecodePlan PL, const uint8_t* __restrict__ qimg_all,
    size_t qimg_stride, const uint8_t* __restrict__ pool, const int32_t* __restrict__ table, int max_pages,
    const int32_t* __restrict__ seq_lens, float* __restrict__ parts, int n_splits) {
  extern __shared__ __align__(128) uint8_t smem[];
  static_assert(BH != 16, "integer modes only");
  constexpr int NTHREADS = NG * GW * 32;

  const int tid = threadIdx.x, lane = tid & 31;
  // warp index as a value the compiler knows to be warp-uniform (shuffle from lane 0): group, ring and MMA operands
  // derived from it stay in uniform registers
  const int warp = __shfl_sync(0xffffffffu, tid >> 5, 0);
  const int j = lane & 3, R = lane >> 2;
  const int split = blockIdx.x, b = blockIdx.y;
  sk_pdl_trigger();
  // Nothing global is read before the dependency wait: seq_lens and the block table may have been written by a kernel the
  // caller enqueued right before this call (CUDA makes a predecessor's writes visible only after griddepcontrol.wait).
  sk_pdl_wait();
  const int len = seq_lens[b];
  int n_pages = len > 0 ? (len + PTOK - 1) / PTOK : 0;
  if (n_pages > max_pages) n_pages = max_pages;   // (a length past the table is a caller error: memory-safe, result undefined)
  int p0, p1;
  sk_split_range(n_pages, n_splits, 1, split, &p0, &p1);
  const int n_it = p1 - p0;
  const size_t pstride = sk_part_stride(L.rank_v);
  float* my_parts = parts + ((size_t)b * n_splits + split) * L.n_q_heads * pstride;

  if (n_it <= 0) {   // empty range (CTA-uniform): neutral partial
    sk_pdl_wait();
    for (int i = tid; i < L.n_q_heads * (int)pstride; i += NTHREADS) {
      const int c = i % (int)pstride;
      my_parts[i] = c == 0 ? -INFINITY : 0.f;
    }
    return;
  }

  uint8_t* stage_base = smem + PL.off_stage;
  const int nstage = PL.nstage;
  const int n_mt = PL.um_mt;                              // 128-channel M tiles
  // barrier area: full[nstage], image, mma_done[NG] mbarriers, TMEM base address, issued[nstage]
  const uint32_t full0 = smem_u32(smem + PL.off_bar);
  const uint32_t qbar = full0 + 8 * nstage;
  const uint32_t mbar0 = qbar + 8;
  const uint32_t afree0 = mbar0 + 8 * NG;   // afree[2]: the MMAs of the page that last used A buffer (it & 1) are complete
  volatile uint32_t& tmem_base_s = *reinterpret_cast<volatile uint32_t*>(smem + PL.off_bar + 8 * nstage + 8 + 8 * NG + 16);
  volatile int* issued = reinterpret_cast<int*>(smem + PL.off_bar + 8 * nstage + 8 + 8 * NG + 24);   // [nstage]
  int32_t* tbl_s = reinterpret_cast<int32_t*>(smem + PL.off_tbl);
  const uint32_t page_bytes = (uint32_t)L.page_bytes;
  const int32_t* my_table = table + (size_t)b * max_pages + p0;

  auto issue = [&](int it, int page) {   // D2: one page -> ring stage (single thread)
    const int st = it % nstage;
    const uint32_t bar = full0 + 8 * st;
    mbar_expect_tx(bar, page_bytes);
    __threadfence_block();   // the barrier is armed before any consumer can see the stage as issued (the refill runs on
                             // a warp of its own, off the group's critical path)
    issued[st] = it;
    bulk_g2s_stream(smem_u32(stage_base + (size_t)st * page_bytes), pool + (size_t)max(page, 0) * page_bytes, page_bytes, bar,
                    l2_evict_first_policy());
  };

  if (tid == 0) {
    for (int s = 0; s < nstage; ++s) {
      mbar_init(full0 + 8 * s, 1);
      issued[s] = -1;
    }
    mbar_init(qbar, 1);
    for (int g = 0; g < NG + 2; ++g) mbar_init(mbar0 + 8 * g, n_mt > 1 ? 2 : 1);   // one commit per issuing warp
    fence_barrier_init();
    int pgs[8];
#pragma unroll
    for (int s = 0; s < 8; ++s) pgs[s] = s < min(nstage, n_it) ? my_table[s] : 0;
    sk_pdl_wait();
    const uint32_t qbytes = (uint32_t)(PL.qimg_bytes + L.n_kv_heads * 32);
    mbar_expect_tx(qbar, qbytes);
    bulk_g2s(smem_u32(smem + PL.off_qimg), qimg_all + (size_t)b * qimg_stride, qbytes, qbar);
#pragma unroll
    for (int s = 0; s < 8; ++s)
      if (s < min(nstage, n_it)) issue(s, pgs[s]);
  }
  if (warp == 1) {   // TMEM: 32 fp32 columns per (group, M tile)
    const uint32_t dst = smem_u32(smem + PL.off_bar + 8 * nstage + 8 + 8 * NG + 16);
    const uint32_t ncol = (uint32_t)PL.um_cols;
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst), "r"(ncol) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
  }
  for (int i = tid; i < min(n_it, TBL_SMEM); i += NTHREADS) tbl_s[i] = my_table[i];

  const int grp = warp >> 3, gw = warp & (GW - 1), gt = tid & 255;
  {
    uint4* pz = reinterpret_cast<uint4*>(smem + PL.off_p);
    for (int i = tid; i < NG * 2 * P_BUF_BYTES / 16; i += NTHREADS) pz[i] = make_uint4(0, 0, 0, 0);
    if (tid < NG * 64) reinterpret_cast<float*>(smem + PL.off_alpha)[tid] = 1.f;
    if (tid < NG * 4) reinterpret_cast<uint32_t*>(smem + PL.off_flag)[tid] = 0;
  }
  sk_pdl_wait();   // (thread 0 has waited already; a second wait returns at once)
  tc_fence_before();
  __syncthreads();
  tc_fence_after();
  // this group's accumulator columns
  const uint32_t tmem_grp = __shfl_sync(0xffffffffu, (uint32_t)tmem_base_s, 0) + (uint32_t)(grp * n_mt * 32);
  mbar_wait(qbar, 0);

  const uint2* qimg_lane = reinterpret_cast<const uint2*>(smem + PL.off_qimg) + lane;
  const float* kcst = reinterpret_cast<const float*>(smem + PL.off_kcst);
  uint8_t* Pm = smem + PL.off_p + grp * 2 * P_BUF_BYTES;
  float* alpha_s = reinterpret_cast<float*>(smem + PL.off_alpha) + grp * 64;
  uint8_t* flag_s = smem + PL.off_flag + grp * 16;
  // two A buffers shared by all groups: page `it` uses buffer it & 1 (with two groups that is the group's own)
  const uint32_t mbar = mbar0 + 8 * grp;

  const bool has_quad = gw < PL.nq;
  const int kv0 = gw * PL.kv_per_quad;
  const int kv1 = min(kv0 + PL.kv_per_quad, L.n_kv_heads);
  // P^T element (head 4 gw + j, token 16 (R >> 1) + 4 (R & 1)) of the canonical B operand
  const int p_thr_off = (gw >> 1) * 1024 + (2 * (R >> 1)) * 128 + (4 * (gw & 1) + j) * 16 + 8 * (R & 1);
  float m_run = -INFINITY, l_run = 0.f;

  // dequantisation work split: the trailing block first, the leading block on the threads its last pass leaves idle
  // (the item slices get lighter with the thread index; the plan hands the light ones to the warps with long QK phases)
  const int n_lo_items = L.v_lo_n * (BL / 2);
  const int gtd = PL.deq_slice[gw] * 32 + lane;
  const int t_hi = (gtd + 256 - (n_lo_items & 255)) & 255;
  // instruction descriptor: D fp32 (bit 4), A and B fp16 K-major, N = 32 (bits 17..), M = 128 (bits 24..)
  constexpr uint32_t IDESC = (1u << 4) | ((uint32_t)(32 >> 3) << 17) | ((uint32_t)(UM_ROWS >> 4) << 24);

  int st = grp % nstage, use = grp / nstage;
  int gi = 0;
  const bool shared_stages = (nstage % NG) != 0;
  for (int it = grp; it < n_it; it += NG, ++gi) {
    uint8_t* pg = stage_base + (size_t)st * page_bytes;
    const int nvalid = len - (p0 + it) * PTOK;   // >= 1
    const int buf = gi & 1;
    uint8_t* Pb = Pm + buf * P_BUF_BYTES;
    float* al = alpha_s + buf * 32;
    uint8_t* fl = flag_s + buf * 8;
    uint8_t* abuf = smem + PL.off_a + (it & 1) * n_mt * UM_TILE_BYTES;
    // A stage shared by several groups can be a whole mbarrier phase behind this group's view, which a parity wait
    // cannot tell from "done": wait until it has been armed for THIS iteration first.  When the ring depth is a multiple
    // of the group count every stage belongs to one group and the parity wait alone is unambiguous.
    if (shared_stages) {
      if (lane == 0)
        while (issued[st] != it) {}
      __syncwarp();
    }
    mbar_wait(full0 + 8 * st, (uint32_t)(use & 1));

    if (nvalid < PTOK) {   // tail page: zero the key rows and the value scales of the slots past the sequence end
      for (int g = 0; g < L.n_kv_heads; ++g) {
        for (int blk = 0; blk < 2; ++blk) {
          const int n = blk ? L.k_lo_n[g] : L.k_hi_n[g];
          const int rowb = n * (blk ? BL : BH) / 8;
          uint32_t* dst = reinterpret_cast<uint32_t*>(pg + (blk ? L.k_lo_off[g] : L.k_hi_off[g]) + nvalid * rowb);
          for (int i = gt; i < (PTOK - nvalid) * rowb / 4; i += 256) dst[i] = 0;
        }
      }
      if (gt < 2 * PTOK && (gt & (PTOK - 1)) >= nvalid) reinterpret_cast<uint16_t*>(pg + L.v_scale_off)[gt] = 0;
      bar_sync(1 + grp, GW * 32);
    }

    // ================= QK + softmax for this warp's quad =================
    if (has_quad)
      score_page<BH, BL, true>(L, PL, pg, qimg_lane, kcst, kv0, kv1, nvalid, R, j, gw, m_run, l_run, Pb, p_thr_off, al, fl);
    // ================= value page -> A operand =================
    if (gi > 0) mbar_wait(mbar, (uint32_t)((gi - 1) & 1));   // the group's previous MMAs are done with P and its TMEM tiles
    if (NG != 2 && it >= 2) mbar_wait(afree0 + 8 * (it & 1), (uint32_t)(((it >> 1) - 1) & 1));   // page it - 2 is done with A
    deq_block_to_a<BL>(pg + L.v_lo_off, pg + L.v_scale_off + PTOK * 2, L.v_lo_n, L.v_hi_n, abuf, gtd);
    deq_block_to_a<BH>(pg + L.v_hi_off, pg + L.v_scale_off, L.v_hi_n, 0, abuf, t_hi);
    fence_proxy_async();   // P and A (generic-proxy stores) -> visible to the tensor-core (async) proxy
    bar_sync(1 + grp, GW * 32);

    // ================= lazy rescale of the TMEM accumulators (rare) =================
    {
      const uint2 f8 = *reinterpret_cast<const uint2*>(fl);
      if ((f8.x | f8.y) != 0 && gi > 0) {
        tc_fence_after();
        for (int mt = gw >> 2; mt < n_mt; mt += 2) {
          const uint32_t taddr = tmem_grp + ((uint32_t)((gw & 3) * 32) << 16) + (uint32_t)(mt * 32);
          uint32_t v[32];
          tmem_ld32(taddr, v);
#pragma unroll
          for (int c = 0; c < 32; ++c) v[c] = __float_as_uint(__uint_as_float(v[c]) * al[c]);
          tmem_st32(taddr, v);
        }
        tc_fence_before();
        bar_sync(1 + grp, GW * 32);
      }
    }

    // ================= PV: one thread issues the MMAs, commits, refills the stage =================
    // warp-uniform roles, one elected lane each, operands are uniform values: warps 0 and 4 issue the MMAs of the even
    // and odd M tiles (different TMEM tiles: no ordering between them) and commit; warp 2 refills the ring stage
    if (gw == 0 || (gw == 4 && n_mt > 1)) {
      tc_fence_after();
      const uint64_t da0 = umma_desc_k(smem_u32(abuf)), db0 = umma_desc_k(smem_u32(Pb));
      if (elect_one()) {
        for (int mt = gw >> 2; mt < n_mt; mt += (n_mt > 1 ? 2 : 1))
#pragma unroll
          for (int ks = 0; ks < PTOK / 16; ++ks)
            umma_f16(tmem_grp + (uint32_t)(mt * 32), da0 + (uint64_t)((mt * UM_TILE_BYTES + ks * 256) >> 4),
                     db0 + (uint64_t)((ks * 256) >> 4), IDESC, (gi > 0 || ks > 0) ? 1u : 0u);
        umma_commit(mbar);
        if (NG != 2) umma_commit(afree0 + 8 * (it & 1));
      }
      __syncwarp();
    } else if (gw == 2) {
      const int nxt = it + nstage;
      if (nxt < n_it && elect_one()) issue(nxt, nxt < TBL_SMEM ? tbl_s[nxt] : my_table[nxt]);
      __syncwarp();
    }
    st += NG;
    while (st >= nstage) { st -= nstage; ++use; }
  }

  // ================= merge the groups and write the split-K partial (D7) =================
  if (gi > 0) mbar_wait(mbar, (uint32_t)((gi - 1) & 1));   // this group's last MMAs are complete
  tc_fence_after();
  bar_sync(BAR_ALL, NTHREADS);
  float* mg = reinterpret_cast<float*>(smem + PL.off_stage);   // m at [g * 32 + head], l at [96 + ..], weight at [192 + ..]
  float* ost = mg + 384;
  const int ST = (int)pstride;
  if (has_quad) {
    float lsum = l_run;
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 4);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 8);
    lsum += __shfl_xor_sync(0xffffffffu, lsum, 16);
    if (R == 0) {
      mg[grp * 32 + 4 * gw + j] = m_run;
      mg[96 + grp * 32 + 4 * gw + j] = lsum;
    }
  }
  bar_sync(BAR_ALL, NTHREADS);
  if (tid < 32) {
    const bool live = tid < L.n_q_heads;
    float ms = -INFINITY, lm = 0.f;
    if (live) {
#pragma unroll
      for (int g = 0; g < NG; ++g) ms = fmaxf(ms, mg[g * 32 + tid]);   // group 0 always has a page: ms is finite
#pragma unroll
      for (int g = 0; g < NG; ++g) {
        const float mo = mg[g * 32 + tid];
        const float w = mo == -INFINITY ? 0.f : ex2(mo - ms);
        mg[192 + g * 32 + tid] = w;
        lm += mg[96 + g * 32 + tid] * w;
      }
      *reinterpret_cast<float4*>(ost + tid * ST) = make_float4(ms, lm, 0.f, 0.f);
    }
  }
  bar_sync(BAR_ALL, NTHREADS);
#pragma unroll
  for (int pass = 0; pass < NG; ++pass) {   // group 0 stores, the others add one after the other (if they had a page)
    if (grp == pass && gi > 0) {
      const float* wt = mg + 192 + 32 * grp;
      for (int mt = gw >> 2; mt < n_mt; mt += 2) {
        const uint32_t taddr = tmem_grp + ((uint32_t)((gw & 3) * 32) << 16) + (uint32_t)(mt * 32);
        uint32_t v[32];
        tmem_ld32(taddr, v);
        const int ch = mt * UM_ROWS + (gw & 3) * 32 + lane;
        if (ch < L.rank_v) {
          float* o = ost + 4 + ch;
#pragma unroll
          for (int h = 0; h < 32; ++h)
            if (h < L.n_q_heads) {
              const float x = __uint_as_float(v[h]) * wt[h];
              o[h * ST] = pass == 0 ? x : o[h * ST] + x;
            }
        }
      }
    }
    bar_sync(BAR_ALL, NTHREADS);
  }
  {
    const float4* src = reinterpret_cast<const float4*>(ost);
    float4* dst = reinterpret_cast<float4*>(my_parts);
    for (int i = tid; i < L.n_q_heads * ST / 4; i += NTHREADS) dst[i] = src[i];
  }
  tc_fence_before();
  __syncthreads();
  if (warp == 1) {
    const uint32_t ncol = (uint32_t)PL.um_cols;
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"((uint32_t)tmem_base_s), "r"(ncol) : "memory");
  }
}

template <int BH, int BL, int NG>
cudaError_t launch_tc5(const starkv_ctx* ctx, dim3 grid, const uint8_t* qimg, size_t qimg_stride, const uint8_t* pool,
                       const int32_t* table, int max_pages, const int32_t* seq_lens, float* parts, int n_splits) {
  auto kern = decode_tc5_kernel<BH, BL, NG>;
  const cudaError_t ea = sk_need_smem(ctx, kern, ctx->plan.smem_bytes);
  if (ea != cudaSuccess) return ea;
  return sk_launch(ctx, kern, grid, dim3(NG * GW * 32), (size_t)ctx->plan.smem_bytes, ctx->L, ctx->plan, qimg, qimg_stride, pool,
                   table, max_pages, seq_lens, parts, n_splits);
}

template <int BH, int BL, int NT, int MT, int NG>
cudaError_t launch_fast(const starkv_ctx* ctx, dim3 grid, const uint8_t* qimg, size_t qimg_stride, const uint8_t* pool,
                        const int32_t* table, int max_pages, const int32_t* seq_lens, float* parts, int n_splits) {
  auto kern = decode_fast_kernel<BH, BL, NT, MT, NG>;
  const cudaError_t ea = sk_need_smem(ctx, kern, ctx->plan.smem_bytes);
  if (ea != cudaSuccess) return ea;
  return sk_launch(ctx, kern, grid, dim3(NG * GW * 32), (size_t)ctx->plan.smem_bytes, ctx->L, ctx->plan, qimg, qimg_stride,
                   pool, table, max_pages, seq_lens, parts, n_splits);
}

template <int BH, int BL, int NG>
cudaError_t dispatch_fast(const starkv_ctx* ctx, dim3 grid, const uint8_t* qimg, size_t qimg_stride, const uint8_t* pool,
                          const int32_t* table, int max_pages, const int32_t* seq_lens, float* parts, int n_splits) {
  const int nt = ctx->plan.nt, mt = ctx->plan.mt;
#define SK_FAST(NTv, MTv) \
  if (nt == NTv && mt == MTv) \
    return launch_fast<BH, BL, NTv, MTv, NG>(ctx, grid, qimg, qimg_stride, pool, table, max_pages, seq_lens, parts, n_splits)
  SK_FAST(1, 1); SK_FAST(1, 2); SK_FAST(1, 3); SK_FAST(1, 4);
  SK_FAST(2, 1); SK_FAST(2, 2); SK_FAST(2, 3); SK_FAST(2, 4);
  SK_FAST(4, 1); SK_FAST(4, 2); SK_FAST(4, 3); SK_FAST(4, 4);
#undef SK_FAST
  return cudaErrorInvalidValue;
}

}  // namespace

// ---------------------------------------------------------------------------------------------
// host: plan, workspace, launch
// ---------------------------------------------------------------------------------------------
static int round_up(int x, int m) { return (x + m - 1) / m * m; }

int sk_fast_plan(starkv_ctx* ctx) {
  const StarkvLayout& L = ctx->L;
  DecodePlan& P = ctx->plan;
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
  P.mt = (P.v_tiles + GW - 1) / GW;
  if (P.mt > 4) return 0;
  const int p_area = NG_MAX * 2 * P_BUF_BYTES;
  const int qarea = round_up(P.qimg_bytes + L.n_kv_heads * 32, 128);   // image + accumulator start values
  const int merge_bytes = 1536 + L.n_q_heads * (L.rank_v + 4) * 4;
  const int fixed = qarea + p_area + NG_MAX * 2 * 32 * 4 /* alpha */ + 128 /* flags */ +
                    256 /* barriers */ + 4 * TBL_SMEM + 128 /* base align */;
  const int avail = ctx->smem_optin - fixed;
  int ns = avail / L.page_bytes;
  if (ns > 8) ns = 8;
  if (ns < 2) return 0;   // one stage per group at least (a third keeps a copy in flight while both compute)
  if ((long long)ns * L.page_bytes < merge_bytes) {
    if (merge_bytes > avail) return 0;
  }
  // tcgen05 PV for the integer modes (decode_tc5_kernel): 2 x um_mt x 16 KB of A operand come out of the ring's memory.
  // Taken when at least 4 ring stages remain (3 when the variant is requested explicitly); SK_VARIANT_MMA keeps mma.sync.
  if (quant && L.rank_v <= 4 * 128 && ctx->variant != SK_VARIANT_MMA) {
    const int um_mt = (L.rank_v + 127) / 128;
    const int need = ctx->variant == SK_VARIANT_TC5 ? 3 : 4;
    const int a_bytes = 2 * um_mt * 128 * PTOK * 2;   // two A buffers, shared by the groups
    int ns5 = (avail - a_bytes) / L.page_bytes;
    if (ns5 > 8) ns5 = 8;
    if (ns5 >= need && avail - a_bytes >= merge_bytes) {
      P.um = 1;
      P.um_mt = um_mt;
      int cols = 32;
      while (cols < 2 * um_mt * 32) cols *= 2;
      P.um_cols = cols;
      ns = ns5;
    }
  }
  {   // dequantisation slices by QK load: lightest QK warp -> slice 0 (the heaviest), ties in warp order
    int cost[GW], order[GW];
    for (int w = 0; w < GW; ++w) {
      const int k0 = w * P.kv_per_quad, k1 = k0 + P.kv_per_quad < L.n_kv_heads ? k0 + P.kv_per_quad : L.n_kv_heads;
      cost[w] = (w < P.nq && k0 < L.n_kv_heads) ? P.qstep_begin[k1] - P.qstep_begin[k0] : 0;
      // the page's bookkeeping counts too (measured: MMA issue about 0.25 us = 3 QK steps, ring refill about half of that)
      if (w == 0 || (w == 4 && L.rank_v > 128)) cost[w] += 3;
      if (w == 2) cost[w] += 1;
      order[w] = w;
    }
    for (int i = 1; i < GW; ++i)
      for (int j2 = i; j2 > 0 && cost[order[j2]] < cost[order[j2 - 1]]; --j2) { const int t = order[j2]; order[j2] = order[j2 - 1]; order[j2 - 1] = t; }
    for (int pos = 0; pos < GW; ++pos) P.deq_slice[order[pos]] = pos;
  }
  P.nstage = ns;
  // pages so large that only two fit: one group, so that the second stage is a copy in flight instead of a
  // second page being computed on (built for the fp16 and int8/int4 modes)
  P.ng = (ns == 2 && (L.bits_hi == 16 || (L.bits_hi == 8 && L.bits_lo == 4))) ? 1 : 2;
  int off = 0;
  P.off_stage = off;
  off += round_up(ns * L.page_bytes > merge_bytes ? ns * L.page_bytes : merge_bytes, 128);
  P.off_qimg = off; P.off_kcst = off + P.qimg_bytes; off += qarea;
  P.off_p = off; off += p_area;
  P.off_alpha = off; off += NG_MAX * 2 * 32 * 4;
  P.off_flag = off; off += 128;
  P.off_bar = off; off += 8 * ns + 8 + 4 * ns + 4 * ns + 128;
  off = round_up(off, 128);
  if (P.um) { P.off_a = off; off += 2 * P.um_mt * 128 * PTOK * 2; }
  P.off_tbl = off; off += 4 * TBL_SMEM;
  P.smem_bytes = round_up(off, 128);
  if (P.smem_bytes > ctx->smem_optin) return 0;
  ctx->fast_ok = 1;
  return 1;
}

int sk_fast_supported(const starkv_ctx* ctx) { return ctx->fast_ok; }

void sk_plan_workspace(const starkv_ctx* ctx, int batch, int max_pages, SkWorkspace* w) {
  const StarkvLayout& L = ctx->L;
  const int slots = ctx->n_sm;   // one CTA per SM
  int ns = ctx->n_splits_override > 0 ? ctx->n_splits_override : slots / (batch > 0 ? batch : 1);
  if (ns > max_pages) ns = max_pages;
  if (ns < 1) ns = 1;
  w->n_splits = ns;
  size_t off = 0;
  int qb_img = ctx->fast_ok ? ctx->plan.qimg_bytes + L.n_kv_heads * 32 : 0;
  if (ctx->tm.ok && ctx->tm.img_bytes > qb_img) qb_img = ctx->tm.img_bytes;
  w->qimg_stride = (size_t)round_up(qb_img, 256);
  w->qimg_off = off; off += w->qimg_stride * batch;
  w->part_off = off; off += ((size_t)batch * ns * L.n_q_heads * sk_part_stride(L.rank_v) * 4 + 255) / 256 * 256;
  w->slice_off = off;   // per-slice up-projection partials of the sliced combine: [batch][H_q][slices of 32 channels][d_h]
  off += ((size_t)batch * L.n_q_heads * ((L.rank_v + 31) / 32) * L.head_dim * 4 + 255) / 256 * 256;
  w->host_off = off;
  const size_t qb = ((size_t)batch * L.n_q_heads * L.head_dim * 2 + 255) / 256 * 256;
  off += 2 * qb + ((size_t)batch * 4 + 255) / 256 * 256;
  w->total = off;
}

int sk_decode_fast(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                   const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws, size_t ws_bytes,
                   void* out, const AppendSmallArgs* app) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (!ctx->fast_ok) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  uint8_t* qimg = (uint8_t*)ws + w.qimg_off;
  if (app) {
    const int n_qp = L.n_kv_heads * batch;
    if (app->fused) {
      SK_PREFER_SMEM(ctx, step_pre_fast_kernel<true>);
      SK_CUDA_CHECK(ctx, sk_launch(ctx, step_pre_fast_kernel<true>, dim3(n_qp + app->n_tiles * app->n_part), dim3(256), 0, L,
                                   ctx->plan, (const __half*)q, (const __half*)B_k, qimg, w.qimg_stride, n_qp, *app));
    } else {   // projection partials with the query image, then the quantiser / paged write as a launch of its own
      SK_PREFER_SMEM(ctx, step_pre_fast_kernel<false>);
      SK_CUDA_CHECK(ctx, sk_launch(ctx, step_pre_fast_kernel<false>, dim3(n_qp + app->n_tiles * app->n_part), dim3(256), 0, L,
                                   ctx->plan, (const __half*)q, (const __half*)B_k, qimg, w.qimg_stride, n_qp, *app));
      const int rw = sk_append_small_write(ctx, app);
      if (rw) return rw;
    }
  } else {
    SK_PREFER_SMEM(ctx, qproj_kernel);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, qproj_kernel, dim3(L.n_kv_heads, batch), dim3(256), 0, L, ctx->plan, (const __half*)q,
                                 (const __half*)B_k, qimg, w.qimg_stride));
  }
  const dim3 grid(w.n_splits, batch);
  const uint8_t* pl = (const uint8_t*)pool;
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  cudaError_t e = cudaErrorInvalidValue;
#define SK_KIND(BHv, BLv, NGv) \
  e = dispatch_fast<BHv, BLv, NGv>(ctx, grid, qimg, w.qimg_stride, pl, table, max_pages, seq_lens, parts, w.n_splits)
  // NG = 3 (768 threads, 80 registers) was measured on C3: 43.1 us against 32.7 us with NG = 2 -- the 412-byte
  // spill frame costs more than the third group hides -- so only NG = 2 is instantiated.
  const bool one = ctx->plan.ng == 1;
#define SK_TC5(BHv, BLv, NGv) \
  e = launch_tc5<BHv, BLv, NGv>(ctx, grid, qimg, w.qimg_stride, pl, table, max_pages, seq_lens, parts, w.n_splits)
  if (ctx->plan.um) {
    if (L.bits_hi == 8 && L.bits_lo == 4) SK_TC5(8, 4, 2);
    else if (L.bits_hi == 8 && L.bits_lo == 8) SK_TC5(8, 8, 2);
    else if (L.bits_hi == 4 && L.bits_lo == 4) SK_TC5(4, 4, 2);
  } else
#undef SK_TC5
  if (L.bits_hi == 16) { if (one) SK_KIND(16, 16, 1); else SK_KIND(16, 16, 2); }
  else if (L.bits_hi == 8 && L.bits_lo == 4) { if (one) SK_KIND(8, 4, 1); else SK_KIND(8, 4, 2); }
  else if (L.bits_hi == 8 && L.bits_lo == 8) SK_KIND(8, 8, 2);
  else if (L.bits_hi == 4 && L.bits_lo == 4) SK_KIND(4, 4, 2);
#undef SK_KIND
  SK_CUDA_CHECK(ctx, e);
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out, reinterpret_cast<float*>((uint8_t*)ws + w.slice_off));
  ctx->last_launches = 3 + ((app && !app->fused) ? 1 : 0);
  return rc;
}
