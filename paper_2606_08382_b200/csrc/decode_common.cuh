// Pieces shared by the two decode kernels: split-K partial format and the combine kernel launcher.
#pragma once
#include "common.cuh"
#include "ctx.h"

// Split-K partial of one (sequence, split, query head):  [m, l, 0, 0, acc[r_v]] fp32 (16-byte aligned rows), where
//   m   = running maximum of the base-2 scores (s * log2 e), -inf for an empty range
//   l   = sum_t 2^(s_t - m)          acc[c] = sum_t 2^(s_t - m) L_v[t, c]
// (both may carry a common power-of-two factor: only acc / l is used).
constexpr int SK_PART_ACC = 4;   // offset of acc[] inside a partial row
__host__ __device__ inline size_t sk_part_stride(int rank_v) { return (size_t)rank_v + SK_PART_ACC; }

// page range [p0, p1) of split `s` of a sequence with n_pages pages, in units of `gran` pages
__host__ __device__ inline void sk_split_range(int n_pages, int n_splits, int gran, int s, int* p0, int* p1) {
  const int units = (n_pages + gran - 1) / gran;
  const int per = (units + n_splits - 1) / n_splits;
  int a = s * per * gran, b = (s + 1) * per * gran;
  if (a > n_pages) a = n_pages;
  if (b > n_pages) b = n_pages;
  *p0 = a;
  *p1 = b;
}

// D8 + D9: log-sum-exp merge of the split partials, normalise, up-project with B_v.
int sk_launch_combine(starkv_ctx* ctx, const float* parts, int n_splits, int batch, const void* B_v, void* out,
                      float* pslice);
