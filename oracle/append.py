"""Compress-on-append by the plain definition.  TEST INFRASTRUCTURE.

PAPER.md §3.2: the cache stores K' = x (Sigma V)_K and V' = x (Sigma V)_V instead of K, V.
Head-wise for keys (one down-projection A_k^h per KV head, §4.3.1 "A_h"), joint for values
(one A_v over the concatenated heads).  Then Eq.12: quantise the latent per token with the
leading/trailing precision split, and write it into the paged cache (DESIGN.md format v1).

One routine, two input modes (reading A15), selected by strides exactly as in the C ABI:
  KV head h reads row t of its input at  k_in[t, h*k_head_stride : h*k_head_stride + d_in_k]
  dense-KV mode   k_head_stride = d_h, d_in_k = d_h          (north_star's "new K/V")
  hidden mode     k_head_stride = 0,   d_in_k = d_model       (the paper's x)
Latent = fp16_RNE( sum_j (double)x_j (double)A_jc ) -- one rounding, from the exact-in-double sum.
"""
from __future__ import annotations

import numpy as np

from .codec import write_token
from .layout import CacheDesc, page_layout


def project_latents(d: CacheDesc, k_in16: np.ndarray, k_head_stride: int, d_in_k: int,
                    v_in16: np.ndarray, ak16: np.ndarray, av16: np.ndarray):
    """fp16 latents (lk [n, sum r_h], lv [n, r_v]) of new tokens.
    k_in16 [n, row] fp16 (row >= (H_kv-1)*k_head_stride + d_in_k), v_in16 [n, d_in_v] fp16,
    ak16 [d_in_k, sum r_h], av16 [d_in_v, r_v]."""
    n = k_in16.shape[0]
    kin = k_in16.reshape(n, -1).astype(np.float64)
    ak = ak16.astype(np.float64)
    lk = np.zeros((n, d.sum_rank_k), np.float16)
    for h, (off, r) in enumerate(zip(d.k_offsets(), d.rank_k)):
        x = kin[:, h * k_head_stride: h * k_head_stride + d_in_k]
        lk[:, off:off + r] = (x @ ak[:, off:off + r]).astype(np.float16)
    lv = (v_in16.reshape(n, -1).astype(np.float64) @ av16.astype(np.float64)).astype(np.float16)
    return lk, lv


def append(d: CacheDesc, pool: np.ndarray, block_table: np.ndarray, seq_ids, positions,
           k_in16, k_head_stride: int, d_in_k: int, v_in16, ak16, av16) -> None:
    """Project, quantise and write n new tokens; token j goes to sequence seq_ids[j] at position
    positions[j] (page block_table[seq][pos // P], slot pos % P).  ``pool`` uint8
    [n_pool_pages, page_bytes] is modified in place."""
    lay = page_layout(d)
    lk, lv = project_latents(d, k_in16, k_head_stride, d_in_k, v_in16, ak16, av16)
    pool = pool.reshape(-1, lay.page_bytes)
    for j in range(lk.shape[0]):
        pos = int(positions[j])
        page = int(block_table[int(seq_ids[j]), pos // lay.page_tokens])
        assert page >= 0
        write_token(d, lay, pool[page], pos % lay.page_tokens, lk[j], lv[j])
