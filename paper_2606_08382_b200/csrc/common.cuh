// Shared device helpers for libstarkv (CUDA side only).
#pragma once
#include <cuda_fp16.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "starkv_layout.h"

// ---- quantiser (reading A11; Eq.12) ---------------------------------
// s = RN_fp16(max|z| / qmax); c = clamp(RNE(z / s), +-qmax); s == 0 -> c = 0.
// IEEE fp32 division + rintf reproduces the exactly rounded result for every fp16 (z, s) pair
// (reciprocal-multiply does not), so __fdiv_rn is load-bearing and fast-math must stay off.
__device__ __forceinline__ int sk_qmax(int bits) { return (1 << (bits - 1)) - 1; }

__device__ __forceinline__ __half sk_scale_of(float amax, int qmax) {
  return __float2half_rn(__fdiv_rn(amax, (float)qmax));
}

__device__ __forceinline__ int sk_code_of(float z, float s, int qmax) {
  if (s == 0.f) return 0;
  float c = rintf(__fdiv_rn(z, s));
  c = fminf(fmaxf(c, -(float)qmax), (float)qmax);
  return (int)c;
}

__device__ __forceinline__ uint16_t sk_half_bits(__half h) { return __half_as_ushort(h); }

// head of a key latent column (linear scan; n_kv_heads <= 64)
__device__ __forceinline__ int sk_head_of_col(const StarkvLayout& L, int col) {
  int h = 0;
  while (h + 1 < L.n_kv_heads && col >= L.koff[h + 1]) ++h;
  return h;
}

