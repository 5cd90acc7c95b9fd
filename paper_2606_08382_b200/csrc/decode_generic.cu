// Plain scalar decode-attention kernel (any page_tokens / head count; fp32 math, exact dequantisation),
// the split-K combine + B_v up-projection kernel (rows D8, D9), and the workspace carve-up.
//   PAPER.md §3.1 L54 (softmax attention), §3.2 L58 (K = K' U_K^T, V = V' U_V^T),
//   §3.3 L62-68 (reordering: score in latent space, (p V') U_V), Eq.12 L208 (dequantisation).
#include "decode_common.cuh"

namespace {

// largest joint value rank of the scalar path (the paper's 75%-compressed MHA layer has r_v = 1024: PAPER.md Fig.11)
constexpr int SK_GEN_MAX_RV = 1024, GEN_VT = SK_GEN_MAX_RV / 128;


constexpr float kLog2e = 1.4426950408889634f;

__device__ __forceinline__ float block_reduce(float v, bool is_max, float* red) {
  const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
#pragma unroll
  for (int o = 16; o; o >>= 1) {
    const float x = __shfl_xor_sync(0xffffffffu, v, o);
    v = is_max ? fmaxf(v, x) : v + x;
  }
  __syncthreads();
  if (lane == 0) red[w] = v;
  __syncthreads();
  float r = red[0];
  for (int i = 1; i < (int)(blockDim.x >> 5); ++i) r = is_max ? fmaxf(r, red[i]) : r + red[i];
  return r;
}

// field `idx` of a row of `bits`-wide fields starting at `row`
__device__ __forceinline__ float field_value(const uint8_t* row, int idx, int bits) {
  if (bits == 16) return __half2float(reinterpret_cast<const __half*>(row)[idx]);
  if (bits == 8) return (float)((int)row[idx] - 128);
  return (float)((int)((row[idx >> 1] >> (4 * (idx & 1))) & 0xF) - 8);
}

// grid (n_splits, H_q, batch), 128 threads.
// ROPE = the paper's own key path (NEXT-1; §3.3, A.6 L619-627): the latent keys are cached pre-RoPE, so the
// score cannot be taken in latent space -- per token: dequantise the latent, reconstruct K = L_k B_k, rotate it at the
// token's position (half-split pairing, reading R1), then q . K with the caller's already-rotated q.  Scalar and
// correctness-first (r_h d_h multiply-adds per token and head; angles in double so that positions of 10^5 keep the
// 2e-3 parity bar): the tensor-core form ([T x r_h] . [r_h x d_h] per KV head) is the next step.
template <bool ROPE>
__global__ void __launch_bounds__(128) decode_generic_kernel(
    const __grid_constant__ StarkvLayout L, const __half* __restrict__ q, const uint8_t* __restrict__ pool,
    const int32_t* __restrict__ table, int max_pages, const int32_t* __restrict__ seq_lens,
    const __half* __restrict__ B_k, float* __restrict__ parts, int n_splits, float rope_theta,
    const int32_t* __restrict__ pos_offset) {
  __shared__ float qt[256];   // latent-space query of this head (r_g <= head_dim <= 256); ROPE: the query itself
  __shared__ float pbuf[128];
  __shared__ float red[4];
  extern __shared__ __align__(16) uint8_t dyn_smem[];   // ROPE: B_k block of the KV head [r][d_h] fp16, inverse frequencies [d_h/2] double
  const int split = blockIdx.x, head = blockIdx.y, b = blockIdx.z;
  const int g = head / L.group;
  const int P = L.page_tokens;
  const bool quant = L.bits_hi != 16;
  const int r = L.rank_k[g];
  const int len = seq_lens[b];
  int n_pages = len > 0 ? (len + P - 1) / P : 0;
  if (n_pages > max_pages) n_pages = max_pages;
  int p0, p1;
  sk_split_range(n_pages, n_splits, 1, split, &p0, &p1);
  const int dh = L.head_dim, half_d = dh >> 1;
  __half* bks = reinterpret_cast<__half*>(dyn_smem);
  double* invf = reinterpret_cast<double*>(dyn_smem + (((size_t)r * dh * 2 + 15) / 16) * 16);

  const __half* qrow = q + ((size_t)b * L.n_q_heads + head) * dh;
  if (ROPE) {
    for (int i = threadIdx.x; i < dh; i += blockDim.x) qt[i] = __half2float(qrow[i]) * L.sm_scale * kLog2e;
    for (int i = threadIdx.x; i < r * dh; i += blockDim.x) bks[i] = B_k[(size_t)L.koff[g] * dh + i];
    for (int i = threadIdx.x; i < half_d; i += blockDim.x) invf[i] = pow((double)rope_theta, -2.0 * (double)i / (double)dh);
  } else {
    // D1: q~ = sm_scale * log2e * q B_k^T
    for (int c = threadIdx.x; c < r; c += blockDim.x) {
      const __half* brow = B_k + (size_t)(L.koff[g] + c) * dh;
      float a = 0.f;
      for (int d = 0; d < dh; ++d) a = fmaf(__half2float(qrow[d]), __half2float(brow[d]), a);
      qt[c] = a * L.sm_scale * kLog2e;
    }
  }
  __syncthreads();

  float m_run = -INFINITY, l_run = 0.f;
  float acc[GEN_VT];   // channels threadIdx.x + 128*k  (rank_v <= 128 GEN_VT = 1024)
#pragma unroll
  for (int k = 0; k < GEN_VT; ++k) acc[k] = 0.f;
  const int n_hi = L.k_hi_n[g], n_lo = L.k_lo_n[g];
  for (int pg = p0; pg < p1; ++pg) {
    const uint8_t* page = pool + (size_t)table[(size_t)b * max_pages + pg] * L.page_bytes;
    for (int s0 = 0; s0 < P; s0 += 128) {
      const int slot = s0 + threadIdx.x;
      const int tok = pg * P + slot;
      const bool valid = slot < P && tok < len;
      float s = -INFINITY;
      if (ROPE && valid) {
        // dequantised latent of the token, its reconstructed and rotated key against the query, one pair at a time
        float lat[128];
        const __half* ksc = reinterpret_cast<const __half*>(page + L.k_scale_off);
        const uint8_t* row = page + L.k_hi_off[g] + (size_t)slot * (n_hi * L.bits_hi / 8);
        const float s_hi = quant ? __half2float(ksc[(g * 2 + 0) * P + slot]) : 1.f;
        for (int c = 0; c < n_hi; ++c) lat[c] = field_value(row, c, L.bits_hi) * s_hi;
        if (quant && n_lo) {
          const uint8_t* row2 = page + L.k_lo_off[g] + (size_t)slot * (n_lo * L.bits_lo / 8);
          const float s_lo = __half2float(ksc[(g * 2 + 1) * P + slot]);
          for (int c = 0; c < n_lo; ++c) lat[n_hi + c] = field_value(row2, c, L.bits_lo) * s_lo;
        }
        const double pos = (double)(tok + (pos_offset ? pos_offset[b] : 0));
        float d = 0.f;
        for (int i = 0; i < half_d; ++i) {
          float k1 = 0.f, k2 = 0.f;
          for (int c = 0; c < r; ++c) {
            k1 = fmaf(lat[c], __half2float(bks[c * dh + i]), k1);
            k2 = fmaf(lat[c], __half2float(bks[c * dh + i + half_d]), k2);
          }
          double sn, cs;
          sincos(pos * invf[i], &sn, &cs);
          const float cf = (float)cs, sf = (float)sn;
          d = fmaf(qt[i], k1 * cf - k2 * sf, d);
          d = fmaf(qt[i + half_d], k2 * cf + k1 * sf, d);
        }
        s = d;
      } else if (valid) {
        const uint8_t* row = page + L.k_hi_off[g] + (size_t)slot * (n_hi * L.bits_hi / 8);
        float d = 0.f;
        for (int c = 0; c < n_hi; ++c) d = fmaf(qt[c], field_value(row, c, L.bits_hi), d);
        if (quant) {
          const __half* ksc = reinterpret_cast<const __half*>(page + L.k_scale_off);
          d *= __half2float(ksc[(g * 2 + 0) * P + slot]);
          if (n_lo) {
            const uint8_t* row2 = page + L.k_lo_off[g] + (size_t)slot * (n_lo * L.bits_lo / 8);
            float d2 = 0.f;
            for (int c = 0; c < n_lo; ++c) d2 = fmaf(qt[n_hi + c], field_value(row2, c, L.bits_lo), d2);
            d = fmaf(d2, __half2float(ksc[(g * 2 + 1) * P + slot]), d);
          }
        }
        s = d;
      }
      const float m_blk = block_reduce(s, true, red);
      if (m_blk == -INFINITY) continue;   // uniform
      const float m_new = fmaxf(m_run, m_blk);
      const float alpha = exp2f(m_run - m_new);   // 0 on the first block
      const float p = valid ? exp2f(s - m_new) : 0.f;
      const float psum = block_reduce(p, false, red);
      l_run = l_run * alpha + psum;
      m_run = m_new;
      __syncthreads();
      pbuf[threadIdx.x] = p;
      __syncthreads();
      const int nt = min(128, P - s0);
#pragma unroll
      for (int k = 0; k < GEN_VT; ++k) {
        const int c = threadIdx.x + 128 * k;
        if (c >= L.rank_v) break;
        const int blk = (quant && c >= L.v_hi_n) ? 1 : 0;
        const int idx = blk ? c - L.v_hi_n : c;
        const int bits = blk ? L.bits_lo : L.bits_hi;
        const uint8_t* row = page + (blk ? L.v_lo_off : L.v_hi_off) + (size_t)idx * (P * bits / 8);
        const __half* vsc = quant ? reinterpret_cast<const __half*>(page + L.v_scale_off) + blk * P : nullptr;
        float a = 0.f;
        for (int t = 0; t < nt; ++t) {
          const float pv = pbuf[t];
          if (pv == 0.f) continue;   // masked slots may hold arbitrary bits
          float v = field_value(row, s0 + t, bits);
          if (quant) v *= __half2float(vsc[s0 + t]);
          a = fmaf(pv, v, a);
        }
        acc[k] = acc[k] * alpha + a;
      }
    }
  }
  float* out = parts + (((size_t)b * n_splits + split) * L.n_q_heads + head) * sk_part_stride(L.rank_v);
  if (threadIdx.x == 0) { out[0] = m_run; out[1] = l_run; }
#pragma unroll
  for (int k = 0; k < GEN_VT; ++k) {
    const int c = threadIdx.x + 128 * k;
    if (c < L.rank_v) out[SK_PART_ACC + c] = acc[k];
  }
}

// grid (H_q, batch), 256 threads.  D8: LSE merge; D9: out_i = o_i . B_v[:, g d_h : (g+1) d_h]
//   1. split weights w_s = 2^(m_s - m*) and l* by block reductions
//   2. o[c] = sum_s w_s acc_s[c], one channel per thread (coalesced over c), loads independent over s
//   3. up-projection with the channel range cut into slices: each thread takes 8 output columns (one 16-byte
//      load of a B_v row) of one slice, slices reduced through shared memory
__global__ void __launch_bounds__(256) combine_kernel(const __grid_constant__ StarkvLayout L,
                                                      const float* __restrict__ parts, int n_splits,
                                                      const __half* __restrict__ B_v, __half* __restrict__ out) {
  __shared__ float o_lat[SK_GEN_MAX_RV];
  __shared__ float wsm[512];
  __shared__ __align__(16) float red[32 * 64];   // [slice][d] partial outputs (slices * d_h <= 2048)
  __shared__ float rsm[8];
  const int head = blockIdx.x, b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int g = head / L.group;
  const size_t ps = sk_part_stride(L.rank_v);
  const float* base = parts + ((size_t)b * n_splits * L.n_q_heads + head) * ps;
  const size_t sstride = (size_t)L.n_q_heads * ps;
  // m* = max_s m_s
  float mx = -INFINITY;
  for (int s = tid; s < n_splits; s += 256) mx = fmaxf(mx, base[s * sstride]);
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) rsm[warp] = mx;
  __syncthreads();
  float mstar = rsm[0];
#pragma unroll
  for (int i = 1; i < 8; ++i) mstar = fmaxf(mstar, rsm[i]);
  float lstar = 0.f;
  for (int s0 = 0; s0 < n_splits; s0 += 512) {   // weights staged in chunks of 512 splits
    const int ns = min(512, n_splits - s0);
    __syncthreads();
    float lp = 0.f;
    for (int s = tid; s < ns; s += 256) {
      const float m = base[(s0 + s) * sstride];
      const float w = (m == -INFINITY) ? 0.f : exp2f(m - mstar);
      wsm[s] = w;
      lp = fmaf(w, base[(s0 + s) * sstride + 1], lp);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, o);
    if (lane == 0) rsm[warp] = lp;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < 8; ++i) lstar += rsm[i];
    for (int c = tid; c < L.rank_v; c += 256) {
      const float* col = base + (size_t)s0 * sstride + SK_PART_ACC + c;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f, a3 = 0.f;
      int s = 0;
      for (; s + 4 <= ns; s += 4) {
        const float v0 = col[(s + 0) * sstride], v1 = col[(s + 1) * sstride], v2 = col[(s + 2) * sstride],
                    v3 = col[(s + 3) * sstride];
        a0 = fmaf(wsm[s + 0], v0, a0); a1 = fmaf(wsm[s + 1], v1, a1);
        a2 = fmaf(wsm[s + 2], v2, a2); a3 = fmaf(wsm[s + 3], v3, a3);
      }
      for (; s < ns; ++s) a0 = fmaf(wsm[s], col[s * sstride], a0);
      o_lat[c] = (s0 ? o_lat[c] : 0.f) + ((a0 + a1) + (a2 + a3));
    }
  }
  __syncthreads();
  const float inv = (mstar == -INFINITY || lstar == 0.f) ? 0.f : 1.f / lstar;
  const int dh = L.head_dim, dv = L.n_kv_heads * dh;
  const int nd8 = dh >> 3;            // 16-byte column groups (<= 32)
  const int nsl = 256 / nd8;          // channel slices (>= 8)
  const int d8 = tid % nd8, sl = tid / nd8;
  float a[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (sl < nsl && inv != 0.f) {
    const __half* bcol = B_v + (size_t)g * dh + 8 * d8;
#pragma unroll 4
    for (int c = sl; c < L.rank_v; c += nsl) {
      const uint4 x = *reinterpret_cast<const uint4*>(bcol + (size_t)c * dv);
      const float w = o_lat[c];
      const float2 x0 = __half22float2(*reinterpret_cast<const __half2*>(&x.x)), x1 = __half22float2(*reinterpret_cast<const __half2*>(&x.y)),
                   x2 = __half22float2(*reinterpret_cast<const __half2*>(&x.z)), x3 = __half22float2(*reinterpret_cast<const __half2*>(&x.w));
      a[0] = fmaf(w, x0.x, a[0]); a[1] = fmaf(w, x0.y, a[1]); a[2] = fmaf(w, x1.x, a[2]); a[3] = fmaf(w, x1.y, a[3]);
      a[4] = fmaf(w, x2.x, a[4]); a[5] = fmaf(w, x2.y, a[5]); a[6] = fmaf(w, x3.x, a[6]); a[7] = fmaf(w, x3.y, a[7]);
    }
  }
  if (sl < nsl) {
    float* r = red + sl * dh + 8 * d8;   // nsl * dh = 256 * 8 = 2048 floats
    *reinterpret_cast<float4*>(r) = make_float4(a[0], a[1], a[2], a[3]);
    *reinterpret_cast<float4*>(r + 4) = make_float4(a[4], a[5], a[6], a[7]);
  }
  __syncthreads();
  for (int d = tid; d < dh; d += 256) {
    float s = 0.f;
    for (int k = 0; k < nsl; ++k) s += red[k * dh + d];
    out[((size_t)b * L.n_q_heads + head) * dh + d] = __float2half_rn(s * inv);
  }
}

// Fast D8 + D9 for n_splits <= 512 and r_v <= 512: one block of 1024 threads per (head, sequence) with every
// global load that does not depend on another issued up front (the B_v slice, the split maxima, the first 16
// accumulator rows per thread), so the kernel costs about two memory round trips instead of one per split.
//   thread = (channel c, split group sg); sg strides the splits; partial sums over sg meet in shared memory.
__global__ void __launch_bounds__(1024) combine_fast_kernel(const __grid_constant__ StarkvLayout L,
                                                            const float* __restrict__ parts, int n_splits,
                                                            const __half* __restrict__ B_v, __half* __restrict__ out) {
  __shared__ float wsm[512];
  __shared__ float psum[1024];
  __shared__ __align__(16) float red[8192];   // [slice][d]: slices * d_h = 1024 * 8
  __shared__ float rsm[64];
  const int head = blockIdx.x, b = blockIdx.y, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  sk_pdl_enter();
  const int g = head / L.group;
  const int rv = L.rank_v, dh = L.head_dim, dv = L.n_kv_heads * dh;
  const size_t ps = sk_part_stride(rv);
  const float* base = parts + ((size_t)b * n_splits * L.n_q_heads + head) * ps;
  const size_t sstride = (size_t)L.n_q_heads * ps;
  // ---- loads that depend on nothing
  const int nd8 = dh >> 3, nsl = 1024 / nd8;   // 16-byte column groups, channel slices
  const int d8 = tid % nd8, sl = tid / nd8;
  const __half* bcol = B_v + (size_t)g * dh + 8 * d8;
  uint4 bq[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int c = sl + k * nsl;
    bq[k] = (sl < nsl && c < rv) ? *reinterpret_cast<const uint4*>(bcol + (size_t)c * dv) : make_uint4(0, 0, 0, 0);
  }
  float2 ml = make_float2(-INFINITY, 0.f);
  if (tid < n_splits) ml = *reinterpret_cast<const float2*>(base + (size_t)tid * sstride);
  const int CW = rv <= 256 ? 256 : 512, nsg = 1024 / CW;
  const int c = tid % CW, sg = tid / CW;
  const float* col = base + SK_PART_ACC + c;
  float v[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) {
    const int s = sg + nsg * k;
    v[k] = (c < rv && s < n_splits) ? col[(size_t)s * sstride] : 0.f;
  }
  // ---- m* and the split weights
  float mx = ml.x;
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) rsm[warp] = mx;
  __syncthreads();
  float mstar = rsm[0];
#pragma unroll
  for (int i = 1; i < 32; ++i) mstar = fmaxf(mstar, rsm[i]);
  const float w = ml.x == -INFINITY ? 0.f : exp2f(ml.x - mstar);
  if (tid < 512) wsm[tid] = w;
  float lp = w * ml.y;
#pragma unroll
  for (int o = 16; o; o >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, o);
  if (lane == 0) rsm[32 + warp] = lp;
  __syncthreads();
  float lstar = 0.f;
#pragma unroll
  for (int i = 0; i < 32; ++i) lstar += rsm[32 + i];
  // ---- o[c] = sum_s w_s acc_s[c]
  float a0 = 0.f, a1 = 0.f;
#pragma unroll
  for (int k = 0; k < 16; k += 2) {
    const int s = sg + nsg * k;
    a0 = fmaf(s < n_splits ? wsm[s] : 0.f, v[k], a0);
    a1 = fmaf(s + nsg < n_splits ? wsm[s + nsg] : 0.f, v[k + 1], a1);
  }
  for (int k0 = 16; sg + nsg * k0 < n_splits; k0 += 16) {   // more than 16 splits per thread
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int s = sg + nsg * (k0 + k);
      v[k] = (c < rv && s < n_splits) ? col[(size_t)s * sstride] : 0.f;
    }
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const int s = sg + nsg * (k0 + k);
      a0 = fmaf(s < n_splits ? wsm[s] : 0.f, v[k], a0);
    }
  }
  psum[tid] = a0 + a1;
  __syncthreads();
  // ---- up-projection: thread (d8, sl) takes channels sl, sl + nsl, ...
  const float inv = (mstar == -INFINITY || lstar == 0.f) ? 0.f : 1.f / lstar;
  float acc[8] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
  if (sl < nsl) {
    auto fma8 = [&](const uint4& x, int cc) {
      float o = psum[cc];
      for (int q = 1; q < nsg; ++q) o += psum[cc + q * CW];
      const float2 x0 = __half22float2(*reinterpret_cast<const __half2*>(&x.x)), x1 = __half22float2(*reinterpret_cast<const __half2*>(&x.y)),
                   x2 = __half22float2(*reinterpret_cast<const __half2*>(&x.z)), x3 = __half22float2(*reinterpret_cast<const __half2*>(&x.w));
      acc[0] = fmaf(o, x0.x, acc[0]); acc[1] = fmaf(o, x0.y, acc[1]); acc[2] = fmaf(o, x1.x, acc[2]); acc[3] = fmaf(o, x1.y, acc[3]);
      acc[4] = fmaf(o, x2.x, acc[4]); acc[5] = fmaf(o, x2.y, acc[5]); acc[6] = fmaf(o, x3.x, acc[6]); acc[7] = fmaf(o, x3.y, acc[7]);
    };
#pragma unroll
    for (int k = 0; k < 4; ++k)
      if (sl + k * nsl < rv) fma8(bq[k], sl + k * nsl);
    for (int cc = sl + 4 * nsl; cc < rv; cc += nsl) fma8(*reinterpret_cast<const uint4*>(bcol + (size_t)cc * dv), cc);
    float* r = red + sl * dh + 8 * d8;
    *reinterpret_cast<float4*>(r) = make_float4(acc[0], acc[1], acc[2], acc[3]);
    *reinterpret_cast<float4*>(r + 4) = make_float4(acc[4], acc[5], acc[6], acc[7]);
  }
  __syncthreads();
  // ---- reduce the slices: (d, part) sums every np-th slice, then np partial sums per column
  const int np = 1024 / dh;   // >= 4
  {
    const int d = tid % dh, p = tid / dh;
    float s = 0.f;
    if (p < np)
      for (int k = p; k < nsl; k += np) s += red[k * dh + d];
    __syncthreads();
    if (p < np) psum[p * dh + d] = s;
  }
  __syncthreads();
  if (tid < dh) {
    float s = 0.f;
    for (int p = 0; p < np; ++p) s += psum[p * dh + tid];
    out[((size_t)b * L.n_q_heads + head) * dh + tid] = __float2half_rn(s * inv);
  }
}

// D8 + D9 spread over (head, channel slice, sequence) blocks, for few sequences and many splits (C3: one sequence, 148
// splits -- one block per head reads 150 KB of partials on its own).  Block (head, slice of 32 channels): every global load
// that depends on nothing -- the (m, l) pairs, this thread's accumulator rows, its B_v elements -- is issued up front, so
// the block costs about one memory round trip: split weights, o[c] = sum_s w_s acc_s[c] (thread = (channel, split group)),
// its part of the up-projection  po[d] = sum_c o[c] B_v[c, g d_h + d] / l*  to the workspace; the LAST slice block of a
// head to arrive (atomic ticket in context-owned memory, reset by that block) adds the slices and writes the fp16 row.
constexpr int CS_THREADS = 256, CS_CH = 32, CS_SG = CS_THREADS / CS_CH, CS_PF = 20;
__global__ void __launch_bounds__(CS_THREADS) combine_sliced_kernel(const __grid_constant__ StarkvLayout L,
                                                                    const float* __restrict__ parts, int n_splits,
                                                                    const __half* __restrict__ B_v, __half* __restrict__ out,
                                                                    float* __restrict__ pslice, int* __restrict__ tickets, int nsl) {
  __shared__ float wsm[512];
  __shared__ float osum[CS_SG][CS_CH];
  __shared__ float po[2][256];
  __shared__ float rsm[16];
  __shared__ int last_s;
  const int head = blockIdx.x, sl = blockIdx.y, b = blockIdx.z, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  sk_pdl_enter();
  const int g = head / L.group;
  const int rv = L.rank_v, dh = L.head_dim, dv = L.n_kv_heads * dh;
  const size_t ps = sk_part_stride(rv);
  const float* base = parts + ((size_t)b * n_splits * L.n_q_heads + head) * ps;
  const size_t sstride = (size_t)L.n_q_heads * ps;
  // ---- loads that depend on nothing
  float2 ml0 = make_float2(-INFINITY, 0.f), ml1 = make_float2(-INFINITY, 0.f);
  if (tid < n_splits) ml0 = *reinterpret_cast<const float2*>(base + (size_t)tid * sstride);
  if (tid + CS_THREADS < n_splits) ml1 = *reinterpret_cast<const float2*>(base + (size_t)(tid + CS_THREADS) * sstride);
  const int c = tid & (CS_CH - 1), sg = tid >> 5;   // channel of the slice, split group
  const int ch = sl * CS_CH + c;
  const float* col = base + SK_PART_ACC + ch;
  float v[CS_PF];
#pragma unroll
  for (int k = 0; k < CS_PF; ++k) {
    const int s = sg + CS_SG * k;
    v[k] = (ch < rv && s < n_splits) ? col[(size_t)s * sstride] : 0.f;
  }
  // up-projection operand: thread (d, half) takes channels half * 16 .. + 16 of the slice (head dims above 128: two passes)
  const int nc = min(CS_CH, rv - sl * CS_CH);
  const int d = tid & 127, hf = tid >> 7;
  const __half* bcol = B_v + (size_t)(sl * CS_CH + hf * 16) * dv + (size_t)g * dh + d;
  __half bq[16];
#pragma unroll
  for (int k = 0; k < 16; ++k) bq[k] = (d < dh && hf * 16 + k < nc) ? bcol[(size_t)k * dv] : __float2half(0.f);
  // ---- m*, the split weights, l*
  float mx = fmaxf(ml0.x, ml1.x);
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) rsm[warp] = mx;
  __syncthreads();
  float mstar = rsm[0];
#pragma unroll
  for (int i = 1; i < CS_THREADS / 32; ++i) mstar = fmaxf(mstar, rsm[i]);
  const float w0 = ml0.x == -INFINITY ? 0.f : exp2f(ml0.x - mstar);
  const float w1 = ml1.x == -INFINITY ? 0.f : exp2f(ml1.x - mstar);
  wsm[tid] = w0;
  wsm[tid + CS_THREADS] = w1;
  float lp = w0 * ml0.y + w1 * ml1.y;
#pragma unroll
  for (int o = 16; o; o >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, o);
  if (lane == 0) rsm[8 + warp] = lp;
  __syncthreads();
  float lstar = 0.f;
#pragma unroll
  for (int i = 0; i < CS_THREADS / 32; ++i) lstar += rsm[8 + i];
  const float inv = (mstar == -INFINITY || lstar == 0.f) ? 0.f : 1.f / lstar;
  // ---- o[c] over this thread's splits (wsm is 0 past n_splits: neutral)
  float a0 = 0.f, a1 = 0.f;
#pragma unroll
  for (int k = 0; k < CS_PF; k += 2) {
    a0 = fmaf(wsm[sg + CS_SG * k], v[k], a0);
    a1 = fmaf(wsm[sg + CS_SG * (k + 1)], v[k + 1], a1);
  }
  if (ch < rv)
    for (int s = sg + CS_SG * CS_PF; s < n_splits; s += CS_SG) a0 = fmaf(wsm[s], col[(size_t)s * sstride], a0);
  osum[sg][c] = a0 + a1;
  __syncthreads();
  if (tid < CS_CH) {
    float o = 0.f;
#pragma unroll
    for (int k = 0; k < CS_SG; ++k) o += osum[k][tid];
    osum[0][tid] = o * inv;
  }
  __syncthreads();
  // ---- this slice's part of the up-projection
  {
    float acc = 0.f;
#pragma unroll
    for (int k = 0; k < 16; ++k) acc = fmaf(osum[0][hf * 16 + k], __half2float(bq[k]), acc);
    po[hf][d] = acc;
  }
  for (int d2 = 128 + d; d2 < dh; d2 += 128) {   // head dims above 128
    float acc = 0.f;
    for (int k = 0; k < 16 && hf * 16 + k < nc; ++k) acc = fmaf(osum[0][hf * 16 + k], __half2float(bcol[(size_t)k * dv + (d2 - d)]), acc);
    po[hf][d2] = acc;
  }
  __syncthreads();
  float* mine = pslice + (((size_t)b * L.n_q_heads + head) * nsl + sl) * dh;
  if (tid < dh) mine[tid] = po[0][tid] + po[1][tid];
  __threadfence();
  __syncthreads();
  if (tid == 0) {
    int* tk = tickets + (size_t)b * L.n_q_heads + head;
    const int t = atomicAdd(tk, 1);
    const int last = t == nsl - 1;
    if (last) *tk = 0;   // ready for the next call (calls of a context are ordered on its stream)
    last_s = last;
  }
  __syncthreads();
  if (last_s) {
    __threadfence();
    if (tid < dh) {
      const float* ph = pslice + ((size_t)b * L.n_q_heads + head) * nsl * dh + tid;
      float sacc = 0.f;
      for (int k = 0; k < nsl; ++k) sacc += __ldcg(ph + (size_t)k * dh);
      out[((size_t)b * L.n_q_heads + head) * dh + tid] = __float2half_rn(sacc);
    }
  }
}

// ---------------------------------------------------------------------------------------------
// D8 alone, latent-output mode (NEXT-3; section 3.3: the attention emits p . V' and an output projection with
// U_V absorbed consumes it): LSE merge of the split partials, normalise, write o~ fp16 [batch][H_q][r_v].  No B_v.
// grid (H_q, slices of 64 channels, batch), 256 threads = 64 channels x 4 groups of splits.
// ---------------------------------------------------------------------------------------------
constexpr int CL_CH = 64, CL_SG = 4, CL_THREADS = CL_CH * CL_SG;
__global__ void __launch_bounds__(CL_THREADS) combine_latent_kernel(const __grid_constant__ StarkvLayout L,
                                                                    const float* __restrict__ parts, int n_splits,
                                                                    __half* __restrict__ out) {
  __shared__ float wsm[512];
  __shared__ float rsm[CL_THREADS / 32];
  __shared__ float red[CL_SG][CL_CH];
  sk_pdl_enter();
  const int head = blockIdx.x, c0 = blockIdx.y * CL_CH, b = blockIdx.z;
  const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5, ch = tid % CL_CH, sg = tid / CL_CH;
  const size_t ps = sk_part_stride(L.rank_v);
  const float* base = parts + ((size_t)b * n_splits * L.n_q_heads + head) * ps;
  const size_t sstride = (size_t)L.n_q_heads * ps;
  float mx = -INFINITY;
  for (int s = tid; s < n_splits; s += CL_THREADS) mx = fmaxf(mx, base[s * sstride]);
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) rsm[warp] = mx;
  __syncthreads();
  float mstar = rsm[0];
#pragma unroll
  for (int i = 1; i < CL_THREADS / 32; ++i) mstar = fmaxf(mstar, rsm[i]);
  float lstar = 0.f, acc = 0.f;
  const bool ok = c0 + ch < L.rank_v;
  for (int s0 = 0; s0 < n_splits; s0 += 512) {   // weights staged in chunks of 512 splits
    const int ns = min(512, n_splits - s0);
    __syncthreads();
    float lp = 0.f;
    for (int s = tid; s < ns; s += CL_THREADS) {
      const float m = base[(s0 + s) * sstride];
      const float w = (m == -INFINITY) ? 0.f : exp2f(m - mstar);
      wsm[s] = w;
      lp = fmaf(w, base[(s0 + s) * sstride + 1], lp);
    }
#pragma unroll
    for (int o = 16; o; o >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, o);
    if (lane == 0) rsm[warp] = lp;
    __syncthreads();
#pragma unroll
    for (int i = 0; i < CL_THREADS / 32; ++i) lstar += rsm[i];
    if (ok) {
      const float* col = base + (size_t)s0 * sstride + SK_PART_ACC + c0 + ch;
#pragma unroll 4
      for (int s = sg; s < ns; s += CL_SG) acc = fmaf(wsm[s], col[s * sstride], acc);
    }
  }
  red[sg][ch] = acc;
  __syncthreads();
  if (sg == 0 && ok) {
    const float inv = (mstar == -INFINITY || lstar == 0.f) ? 0.f : 1.f / lstar;   // empty sequence: a zero row
    const float o = (red[0][ch] + red[1][ch]) + (red[2][ch] + red[3][ch]);
    out[((size_t)b * L.n_q_heads + head) * L.rank_v + c0 + ch] = __float2half_rn(o * inv);
  }
}

// The same for n_splits <= 512, in the style of combine_sliced_kernel: one (head, slice of 32 channels, sequence) per
// block, 32 channels x 8 split groups, every load that depends on nothing issued before the first reduction.
__global__ void __launch_bounds__(CS_THREADS) combine_latent_sliced_kernel(const __grid_constant__ StarkvLayout L,
                                                                          const float* __restrict__ parts, int n_splits,
                                                                          __half* __restrict__ out) {
  __shared__ float wsm[512];
  __shared__ float osum[CS_SG][CS_CH];
  __shared__ float rsm[16];
  const int head = blockIdx.x, sl = blockIdx.y, b = blockIdx.z, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  sk_pdl_enter();
  const int rv = L.rank_v;
  const size_t ps = sk_part_stride(rv);
  const float* base = parts + ((size_t)b * n_splits * L.n_q_heads + head) * ps;
  const size_t sstride = (size_t)L.n_q_heads * ps;
  float2 ml0 = make_float2(-INFINITY, 0.f), ml1 = make_float2(-INFINITY, 0.f);
  if (tid < n_splits) ml0 = *reinterpret_cast<const float2*>(base + (size_t)tid * sstride);
  if (tid + CS_THREADS < n_splits) ml1 = *reinterpret_cast<const float2*>(base + (size_t)(tid + CS_THREADS) * sstride);
  const int c = tid & (CS_CH - 1), sg = tid >> 5;   // channel of the slice, split group
  const int ch = sl * CS_CH + c;
  const float* col = base + SK_PART_ACC + ch;
  float v[CS_PF];
#pragma unroll
  for (int k = 0; k < CS_PF; ++k) {
    const int s = sg + CS_SG * k;
    v[k] = (ch < rv && s < n_splits) ? col[(size_t)s * sstride] : 0.f;
  }
  float mx = fmaxf(ml0.x, ml1.x);
#pragma unroll
  for (int o = 16; o; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
  if (lane == 0) rsm[warp] = mx;
  __syncthreads();
  float mstar = rsm[0];
#pragma unroll
  for (int i = 1; i < CS_THREADS / 32; ++i) mstar = fmaxf(mstar, rsm[i]);
  const float w0 = ml0.x == -INFINITY ? 0.f : exp2f(ml0.x - mstar);
  const float w1 = ml1.x == -INFINITY ? 0.f : exp2f(ml1.x - mstar);
  wsm[tid] = w0;
  wsm[tid + CS_THREADS] = w1;
  float lp = w0 * ml0.y + w1 * ml1.y;
#pragma unroll
  for (int o = 16; o; o >>= 1) lp += __shfl_xor_sync(0xffffffffu, lp, o);
  if (lane == 0) rsm[8 + warp] = lp;
  __syncthreads();
  float lstar = 0.f;
#pragma unroll
  for (int i = 0; i < CS_THREADS / 32; ++i) lstar += rsm[8 + i];
  const float inv = (mstar == -INFINITY || lstar == 0.f) ? 0.f : 1.f / lstar;   // empty sequence: a zero row
  float a0 = 0.f, a1 = 0.f;   // (wsm is 0 past n_splits: neutral)
#pragma unroll
  for (int k = 0; k < CS_PF; k += 2) {
    a0 = fmaf(wsm[sg + CS_SG * k], v[k], a0);
    a1 = fmaf(wsm[sg + CS_SG * (k + 1)], v[k + 1], a1);
  }
  if (ch < rv)
    for (int s = sg + CS_SG * CS_PF; s < n_splits; s += CS_SG) a0 = fmaf(wsm[s], col[(size_t)s * sstride], a0);
  osum[sg][c] = a0 + a1;
  __syncthreads();
  if (tid < CS_CH && sl * CS_CH + tid < rv) {
    float o = 0.f;
#pragma unroll
    for (int k = 0; k < CS_SG; ++k) o += osum[k][tid];
    out[((size_t)b * L.n_q_heads + head) * rv + sl * CS_CH + tid] = __float2half_rn(o * inv);
  }
}

}  // namespace

int sk_launch_combine(starkv_ctx* ctx, const float* parts, int n_splits, int batch, const void* B_v, void* out,
                      float* pslice) {
  const StarkvLayout& L = ctx->L;
  if (!B_v && n_splits <= 512) {   // latent-output mode (starkv_decode_attn_latent): merge and normalise only
    SK_PREFER_SMEM(ctx, combine_latent_sliced_kernel);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, combine_latent_sliced_kernel, dim3(L.n_q_heads, (L.rank_v + CS_CH - 1) / CS_CH, batch),
                                 dim3(CS_THREADS), 0, L, parts, n_splits, (__half*)out));
    return STARKV_OK;
  }
  if (!B_v) {
    SK_PREFER_SMEM(ctx, combine_latent_kernel);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, combine_latent_kernel, dim3(L.n_q_heads, (L.rank_v + CL_CH - 1) / CL_CH, batch), dim3(CL_THREADS),
                                 0, L, parts, n_splits, (__half*)out));
    return STARKV_OK;
  }
  const int nsl = (L.rank_v + CS_CH - 1) / CS_CH;
  // sliced combine where one block per head would be the long pole: few sequences, many splits
  // (measured: C3, 148 splits x 1 sequence: step 57.6 -> 53.2 us; C2, 37 splits x 4 sequences: 50.0 -> 54.1 us)
  if (ctx->tickets && pslice && n_splits >= 64 && n_splits <= 512 && L.head_dim <= CS_THREADS && nsl > 1 &&
      (size_t)batch * L.n_q_heads <= (size_t)SK_TICKETS && batch * L.n_q_heads < 2 * ctx->n_sm) {
    SK_PREFER_SMEM(ctx, combine_sliced_kernel);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, combine_sliced_kernel, dim3(L.n_q_heads, nsl, batch), dim3(CS_THREADS), 0, L, parts, n_splits,
                                 (const __half*)B_v, (__half*)out, pslice, ctx->tickets, nsl));
  } else if (n_splits <= 512 && L.rank_v <= 512) {
    SK_PREFER_SMEM(ctx, combine_fast_kernel);
    SK_CUDA_CHECK(ctx, sk_launch(ctx, combine_fast_kernel, dim3(L.n_q_heads, batch), dim3(1024), 0, L, parts, n_splits,
                                 (const __half*)B_v, (__half*)out));
  } else {
    SK_PREFER_SMEM(ctx, combine_kernel);
    combine_kernel<<<dim3(L.n_q_heads, batch), 256, 0, ctx->stream>>>(L, parts, n_splits, (const __half*)B_v, (__half*)out);
  }
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  return STARKV_OK;
}

int sk_decode_generic(starkv_ctx* ctx, const void* q, const void* pool, const int32_t* table, int max_pages,
                      const int32_t* seq_lens, int batch, const void* B_k, const void* B_v, void* ws,
                      size_t ws_bytes, void* out, int rope, float rope_theta, const int32_t* pos_offset) {
  const StarkvLayout& L = ctx->L;
  ctx->last_launches = 0;
  if (L.rank_v > SK_GEN_MAX_RV) return STARKV_ERR_UNSUPPORTED;
  SkWorkspace w;
  sk_plan_workspace(ctx, batch, max_pages, &w);
  if (ws_bytes < w.total) return STARKV_ERR_WORKSPACE;
  float* parts = reinterpret_cast<float*>((uint8_t*)ws + w.part_off);
  if (ctx->timing_on) SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev0, ctx->stream));
  if (rope) {
    int r_max = 0;
    for (int h = 0; h < L.n_kv_heads; ++h) r_max = L.rank_k[h] > r_max ? L.rank_k[h] : r_max;
    if (r_max > 128) return STARKV_ERR_UNSUPPORTED;
    const int smem = ((r_max * L.head_dim * 2 + 15) / 16) * 16 + (L.head_dim / 2) * 8;
    if (smem > ctx->smem_optin) return STARKV_ERR_UNSUPPORTED;
    SK_CUDA_CHECK(ctx, sk_need_smem(ctx, decode_generic_kernel<true>, smem));
    decode_generic_kernel<true><<<dim3(w.n_splits, L.n_q_heads, batch), 128, smem, ctx->stream>>>(
        L, (const __half*)q, (const uint8_t*)pool, table, max_pages, seq_lens, (const __half*)B_k, parts, w.n_splits, rope_theta,
        pos_offset);
  } else {
    decode_generic_kernel<false><<<dim3(w.n_splits, L.n_q_heads, batch), 128, 0, ctx->stream>>>(
        L, (const __half*)q, (const uint8_t*)pool, table, max_pages, seq_lens, (const __half*)B_k, parts, w.n_splits, 0.f, nullptr);
  }
  SK_CUDA_CHECK(ctx, cudaGetLastError());
  if (ctx->timing_on) {
    SK_CUDA_CHECK(ctx, cudaEventRecord(ctx->ev1, ctx->stream));
    ctx->timing_valid = 1;
  }
  const int rc = sk_launch_combine(ctx, parts, w.n_splits, batch, B_v, out, reinterpret_cast<float*>((uint8_t*)ws + w.slice_off));
  ctx->last_launches = 2;
  return rc;
}
