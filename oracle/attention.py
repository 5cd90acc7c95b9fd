"""Decode attention over the latent cache by the plain definition, fp64.  TEST INFRASTRUCTURE.

What the fast path reaches exactly (up to rounding) has a plain definition, so the oracle is
that definition written out (no absorbed-form shortcut, no online softmax, no split-K):

  1. read the very bits the GPU reads (packed pages, fp16 scales/factors/q), dequantise
     L = code * scale                                         (Eq.12)
  2. reconstruct dense K^h = L_k^h B_k^h  and  V = L_v B_v    (§3.2:
     K = K' U_K^T, V = V' U_V^T; head-wise for K, joint for V: §4.3.1, §4.3.3)
  3. textbook attention per query head i with KV head g = floor(i/G):
     P = softmax(q_i K^gT * sm_scale), out_i = P V[:, g d_h:(g+1) d_h]   (§3.1)

One query token attends to positions [0, seq_len) and nothing else (decode; reading A3); there
is no RoPE on this path (reading A1: BASELINE.json's north_star scores in latent space).
seq_len = 0 gives zeros.  Summation over tokens is chunked only to bound memory.

``decode_attn_absorbed`` is a second, independent formulation (weight absorption / operation
reordering, §3.3) used only by identity tests; ``dense_attention`` is the
textbook routine on explicit K, V used by the full-rank pin.
"""
from __future__ import annotations

from typing import Optional, Sequence

import numpy as np

from .codec import read_sequence
from .layout import CacheDesc


def dense_attention(q: np.ndarray, K: np.ndarray, V: np.ndarray, sm_scale: float, group: int):
    """Textbook softmax attention, one query token.  q [H_q, d], K [l, H_kv, d], V [l, H_kv, d]
    -> out [H_q, d]."""
    hq = q.shape[0]
    out = np.zeros((hq, V.shape[2]))
    for i in range(hq):
        g = i // group
        s = (K[:, g, :] @ q[i]) * sm_scale
        p = np.exp(s - s.max())
        out[i] = (p @ V[:, g, :]) / p.sum()
    return out


def decode_attn(d: CacheDesc, q16: np.ndarray, pool: np.ndarray, block_table: np.ndarray,
                seq_lens: Sequence[int], bk16: np.ndarray, bv16: np.ndarray,
                heads: Optional[Sequence[int]] = None, chunk: int = 8192, diag: Optional[dict] = None):
    """out float64 [B, H_q, d_h] (rows of heads not in ``heads`` are left zero)."""
    B = q16.shape[0]
    dh, G = d.head_dim, d.group
    heads = list(range(d.n_q_heads)) if heads is None else [int(h) for h in heads]
    q = q16.astype(np.float64)
    bk = bk16.astype(np.float64)
    bv = bv16.astype(np.float64)
    koff = d.k_offsets()
    out = np.zeros((B, d.n_q_heads, dh))
    if diag is not None:
        diag["n_eff"] = np.zeros((B, d.n_q_heads))
    for b in range(B):
        l = int(seq_lens[b])
        if l == 0:
            continue
        Lk, Lv = read_sequence(d, pool, block_table[b], l)
        # scores: reconstruct the dense key of each needed KV head, then q . K
        s = {}
        for g in sorted({i // G for i in heads}):
            Kg = Lk[:, koff[g]:koff[g] + d.rank_k[g]] @ bk[koff[g]:koff[g] + d.rank_k[g]]   # [l, d_h]
            for i in heads:
                if i // G == g:
                    s[i] = (Kg @ q[b, i]) * d.sm_scale
        p = {i: np.exp(s[i] - s[i].max()) for i in heads}
        if diag is not None:
            for i in heads:
                w = p[i] / p[i].sum()
                diag["n_eff"][b, i] = 1.0 / np.sum(w * w)
        acc = {i: np.zeros(dh) for i in heads}
        for t0 in range(0, l, chunk):
            t1 = min(l, t0 + chunk)
            for g in sorted({i // G for i in heads}):
                Vg = Lv[t0:t1] @ bv[:, g * dh:(g + 1) * dh]                                  # [c, d_h]
                for i in heads:
                    if i // G == g:
                        acc[i] += p[i][t0:t1] @ Vg
        for i in heads:
            out[b, i] = acc[i] / p[i].sum()
    return out


def decode_attn_latent(d: CacheDesc, q16: np.ndarray, pool: np.ndarray, block_table: np.ndarray,
                       seq_lens: Sequence[int], bk16: np.ndarray, heads: Optional[Sequence[int]] = None):
    """NEXT-3, latent-output mode: the attention emits o~_i = softmax(s_i) . L_v, a row of r_v latent
    channels per query head, and leaves the up-projection to an output projection with U_V absorbed
    (section 3.3: "(p . V') . U_V", W'_out^i = W_out^i U_V^i).  Scores exactly as in decode_attn
    (dequantise, reconstruct K = L_k B_k, q . K, L58 / L62-68); softmax L54; then the weights times the dequantised
    joint value latents -- no B_v anywhere.  out float64 [B, H_q, r_v]; seq_len 0 gives a zero row (reading N2)."""
    B = q16.shape[0]
    G = d.group
    heads = list(range(d.n_q_heads)) if heads is None else [int(h) for h in heads]
    q = q16.astype(np.float64)
    bk = bk16.astype(np.float64)
    koff = d.k_offsets()
    out = np.zeros((B, d.n_q_heads, d.rank_v))
    for b in range(B):
        l = int(seq_lens[b])
        if l == 0:
            continue
        Lk, Lv = read_sequence(d, pool, block_table[b], l)
        for i in heads:
            g = i // G
            Kg = Lk[:, koff[g]:koff[g] + d.rank_k[g]] @ bk[koff[g]:koff[g] + d.rank_k[g]]   # [l, d_h]
            s = (Kg @ q[b, i]) * d.sm_scale
            p = np.exp(s - s.max())
            out[b, i] = (p / p.sum()) @ Lv
    return out


def rope_rotate(x: np.ndarray, positions: np.ndarray, theta: float) -> np.ndarray:
    """Rotary position embedding of rows x[t, :d_h] at integer positions[t] (Su et al. 2024; §3.3:
    "RoPE ... applied to the query and key states prior to computing attention scores").

    Channel pairing: HALF-SPLIT -- channel i is rotated together with channel i + d_h/2 by the angle
    positions[t] * theta^(-2i/d_h), i in [0, d_h/2) -- the convention of the LLaMA-family implementations the paper
    evaluates.  The paper does not state the pairing (interleaved pairs (2i, 2i+1) are the other common choice):
    DESIGN.md reading R1, parity with the authors' code UNPINNED."""
    x = np.asarray(x, np.float64)
    dh = x.shape[-1]
    half = dh // 2
    inv_freq = theta ** (-np.arange(half, dtype=np.float64) * 2.0 / dh)
    ang = np.asarray(positions, np.float64)[:, None] * inv_freq[None, :]
    c, sn = np.cos(ang), np.sin(ang)
    x1, x2 = x[..., :half], x[..., half:]
    return np.concatenate([x1 * c - x2 * sn, x2 * c + x1 * sn], axis=-1)


def decode_attn_rope(d: CacheDesc, q16: np.ndarray, pool: np.ndarray, block_table: np.ndarray,
                     seq_lens: Sequence[int], bk16: np.ndarray, bv16: np.ndarray, theta: float,
                     pos_offset: Optional[Sequence[int]] = None, pos_stride: int = 1,
                     heads: Optional[Sequence[int]] = None):
    """The paper's own key path (NEXT-1; §3.3, A.6 L619-627), step by step in the paper's order:
    latent keys are cached PRE-RoPE; per token: dequantise, reconstruct K = L_k B_k, apply RoPE at the token's position,
    then q . K; softmax; values as in ``decode_attn`` ((p V') U_V).  ``q16`` is the query AFTER its own rotation (the
    caller rotates q at the current position, as it does for dense attention; any float dtype).  Token t of sequence b
    sits at position pos_offset[b] + pos_stride * t (defaults 0 and 1; stride 0 puts every token at one position, which
    the pins use).  out float64 [B, H_q, d_h]."""
    B = q16.shape[0]
    dh, G = d.head_dim, d.group
    heads = list(range(d.n_q_heads)) if heads is None else [int(h) for h in heads]
    q = np.asarray(q16, np.float64)
    bk = bk16.astype(np.float64)
    bv = bv16.astype(np.float64)
    koff = d.k_offsets()
    out = np.zeros((B, d.n_q_heads, dh))
    for b in range(B):
        l = int(seq_lens[b])
        if l == 0:
            continue
        pos = pos_stride * np.arange(l) + (0 if pos_offset is None else int(pos_offset[b]))
        Lk, Lv = read_sequence(d, pool, block_table[b], l)
        for i in heads:
            g = i // G
            Kg = Lk[:, koff[g]:koff[g] + d.rank_k[g]] @ bk[koff[g]:koff[g] + d.rank_k[g]]   # reconstruct [l, d_h]
            Kg = rope_rotate(Kg, pos, theta)                                                   # RoPE at the token's position
            s = (Kg @ q[b, i]) * d.sm_scale
            p = np.exp(s - s.max())
            Vg = Lv @ bv[:, g * dh:(g + 1) * dh]
            out[b, i] = (p @ Vg) / p.sum()
    return out


def decode_attn_absorbed(d: CacheDesc, q16, pool, block_table, seq_lens, bk16, bv16):
    """Same result through the reordered products (§3.3): score =
    (q B_k^T) . L_k, out = ((p L_v) / sum p) B_v[:, slice].  Identity tests only."""
    B = q16.shape[0]
    dh, G = d.head_dim, d.group
    q = q16.astype(np.float64)
    bk = bk16.astype(np.float64)
    bv = bv16.astype(np.float64)
    koff = d.k_offsets()
    out = np.zeros((B, d.n_q_heads, dh))
    for b in range(B):
        l = int(seq_lens[b])
        if l == 0:
            continue
        Lk, Lv = read_sequence(d, pool, block_table[b], l)
        for i in range(d.n_q_heads):
            g = i // G
            qt = bk[koff[g]:koff[g] + d.rank_k[g]] @ q[b, i]                  # latent-space query
            s = (Lk[:, koff[g]:koff[g] + d.rank_k[g]] @ qt) * d.sm_scale
            p = np.exp(s - s.max())
            o_lat = (p @ Lv) / p.sum()                                        # [r_v]
            out[b, i] = o_lat @ bv[:, g * dh:(g + 1) * dh]
    return out


def partial_attn(d: CacheDesc, q16, Lk, Lv, bk16, bv16, b: int):
    """Un-normalised attention state of one token range: (m [H_q], l [H_q], acc [H_q, d_h]) with
    acc = sum_t exp(s_t - m) V_t.  Used with ``lse_merge`` by the split-combine pin."""
    dh, G = d.head_dim, d.group
    q = q16.astype(np.float64)
    bk, bv = bk16.astype(np.float64), bv16.astype(np.float64)
    koff = d.k_offsets()
    m = np.zeros(d.n_q_heads)
    ell = np.zeros(d.n_q_heads)
    acc = np.zeros((d.n_q_heads, dh))
    for i in range(d.n_q_heads):
        g = i // G
        Kg = Lk[:, koff[g]:koff[g] + d.rank_k[g]] @ bk[koff[g]:koff[g] + d.rank_k[g]]
        s = (Kg @ q[b, i]) * d.sm_scale
        m[i] = s.max()
        p = np.exp(s - m[i])
        ell[i] = p.sum()
        acc[i] = p @ (Lv @ bv[:, g * dh:(g + 1) * dh])
    return m, ell, acc


def lse_merge(parts):
    """Log-sum-exp merge of split partials: m* = max m_s, l* = sum l_s e^{m_s-m*},
    acc* = sum acc_s e^{m_s-m*}, out = acc*/l*."""
    ms = np.stack([p[0] for p in parts])
    mstar = ms.max(axis=0)
    w = np.exp(ms - mstar)
    ell = sum(w[k] * parts[k][1] for k in range(len(parts)))
    acc = sum(w[k][:, None] * parts[k][2] for k in range(len(parts)))
    return acc / ell[:, None]
