"""Byte map of one latent-cache page -- DESIGN.md "Cache page format v1" written out.

TEST INFRASTRUCTURE (see oracle/__init__.py).  Not from the paper (PAPER.md only cites
PagedAttention, L361); the format text in DESIGN.md is the common source for this file and for
the CUDA code, which share nothing else.

A page holds P consecutive tokens ("slots") of one sequence for one layer:

  for KV head h = 0..H_kv-1:   K_hi^h  P rows x r_hi^h channels   (token-major, bits_hi each)
                               K_lo^h  P rows x (r_h - r_hi^h)    (token-major, bits_lo each)
  K_scales  [H_kv][2][P] fp16  (quantised modes only; blk 0 = hi, 1 = lo)
  V_hi      r_v_hi rows x P slots     (channel-major, bits_hi each)
  V_lo      (r_v - r_v_hi) rows x P   (channel-major, bits_lo each)
  V_scales  [2][P] fp16        (quantised modes only)

Each block is padded to a multiple of 16 B, the page to a multiple of 128 B.  4-bit fields: two
per byte, low nibble = even index (channel for K rows, slot for V rows).  Code fields are
offset binary u = c + 2^(b-1).  fp16 mode (bits 16/16): one block per head / for V holding
IEEE fp16, no hi/lo split, no scales.
"""
from __future__ import annotations

import dataclasses
from typing import List


def _up(x: int, m: int) -> int:
    return (x + m - 1) // m * m


@dataclasses.dataclass
class CacheDesc:
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    rank_k: List[int]
    rank_k_hi: List[int]
    rank_v: int
    rank_v_hi: int
    bits_hi: int
    bits_lo: int
    page_tokens: int
    sm_scale: float

    @classmethod
    def from_config(cls, cfg) -> "CacheDesc":
        return cls(cfg.n_q_heads, cfg.n_kv_heads, cfg.head_dim, list(cfg.rank_k),
                   list(cfg.rank_k_hi), cfg.rank_v, cfg.rank_v_hi, cfg.bits_hi, cfg.bits_lo,
                   cfg.page_tokens, float(cfg.sm_scale))

    @property
    def quantized(self) -> bool:
        return self.bits_hi != 16

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def sum_rank_k(self) -> int:
        return sum(self.rank_k)

    def k_offsets(self) -> List[int]:
        out, off = [], 0
        for r in self.rank_k:
            out.append(off)
            off += r
        return out

    def validate(self) -> None:
        assert self.n_q_heads % self.n_kv_heads == 0
        assert (self.bits_hi, self.bits_lo) in ((16, 16), (8, 4), (8, 8), (4, 4))
        assert self.page_tokens % 16 == 0 and self.page_tokens > 0
        for r, rh in zip(self.rank_k, self.rank_k_hi):
            assert r % 8 == 0 and 0 < r <= self.head_dim and rh % 8 == 0 and 0 < rh <= r
        assert self.rank_v % 8 == 0 and self.rank_v_hi % 8 == 0 and 0 < self.rank_v_hi <= self.rank_v
        assert self.rank_v <= self.n_kv_heads * self.head_dim


@dataclasses.dataclass
class PageLayout:
    page_tokens: int
    page_bytes: int
    k_hi_off: List[int]
    k_hi_n: List[int]       # channels in the block
    k_lo_off: List[int]
    k_lo_n: List[int]
    k_scale_off: int        # -1 in fp16 mode
    v_hi_off: int
    v_hi_n: int
    v_lo_off: int
    v_lo_n: int
    v_scale_off: int        # -1 in fp16 mode
    bits_hi: int
    bits_lo: int


def page_layout(d: CacheDesc) -> PageLayout:
    d.validate()
    p = d.page_tokens
    off = 0
    k_hi_off, k_hi_n, k_lo_off, k_lo_n = [], [], [], []
    for r, rh in zip(d.rank_k, d.rank_k_hi):
        n_hi = r if not d.quantized else rh
        n_lo = 0 if not d.quantized else r - rh
        k_hi_off.append(off)
        k_hi_n.append(n_hi)
        off += _up(p * n_hi * d.bits_hi // 8, 16)
        k_lo_off.append(off)
        k_lo_n.append(n_lo)
        off += _up(p * n_lo * d.bits_lo // 8, 16)
    k_scale_off = -1
    if d.quantized:
        k_scale_off = off
        off += _up(d.n_kv_heads * 2 * p * 2, 16)
    v_hi_n = d.rank_v if not d.quantized else d.rank_v_hi
    v_lo_n = 0 if not d.quantized else d.rank_v - d.rank_v_hi
    v_hi_off = off
    off += _up(v_hi_n * p * d.bits_hi // 8, 16)
    v_lo_off = off
    off += _up(v_lo_n * p * d.bits_lo // 8, 16)
    v_scale_off = -1
    if d.quantized:
        v_scale_off = off
        off += _up(2 * p * 2, 16)
    return PageLayout(p, _up(off, 128), k_hi_off, k_hi_n, k_lo_off, k_lo_n, k_scale_off,
                      v_hi_off, v_hi_n, v_lo_off, v_lo_n, v_scale_off, d.bits_hi, d.bits_lo)
