"""Low-rank-aware mixed-precision quantiser and page pack/unpack.  TEST INFRASTRUCTURE.

Follows PAPER.md §4.4 L204-210 and Eq.12:  Z_hat = [Q_{b_out}(Z_out) Q_{b_in}(Z_in)],
with the latent channels split into a leading "outlier" block (highest singular values, L206:
channels are ordered by singular value) kept at b_out bits and the trailing "inlier" block at
b_in < b_out bits, quantised per token (L206 "mixed-precision per-token quantization").  The
Hadamard factors H_out, H_in of Eq.12 are fused offline into the projection factors (L210), so
the runtime quantiser sees Z H already and applies only Q.

The paper does not define Q beyond "per-token" (readings A5, A6, A11).  Reading used,
for one token's one precision block z in fp16^n, b bits, qmax = 2^(b-1) - 1:

    a = max_j |z_j|            s = RN_fp16(a / qmax)
    s == 0  ->  all codes 0    else  c_j = clamp(RNE(z_j / s), -qmax, +qmax)
    dequantised value = c_j * s;  stored field u_j = c_j + 2^(b-1)  (offset binary)

All arithmetic here is exact or correctly rounded: z, s are fp16 values held in float64;
z/s in float64 then rint (ties to even).  tests/test_oracle_codec.py proves against exact
rational arithmetic that float64 (and float32) division + rint gives the exactly-rounded code.
"""
from __future__ import annotations

import numpy as np

from .layout import CacheDesc, PageLayout, page_layout


def qmax_of(bits: int) -> int:
    return (1 << (bits - 1)) - 1


def quantize_block(z16: np.ndarray, bits: int):
    """Quantise the last axis of ``z16`` (fp16, shape [..., n]) as ONE precision block per row.
    Returns (codes int8 [..., n], scale fp16 [...])."""
    assert z16.dtype == np.float16
    qmax = qmax_of(bits)
    lead = z16.shape[:-1]
    if z16.shape[-1] == 0:
        return np.zeros(z16.shape, np.int8), np.zeros(lead, np.float16)
    z = z16.astype(np.float64)
    a = np.max(np.abs(z), axis=-1)
    s16 = (a / qmax).astype(np.float16)                     # RN to fp16
    s = s16.astype(np.float64)[..., None]
    with np.errstate(divide="ignore", invalid="ignore"):
        c = np.rint(z / np.where(s == 0, 1.0, s))           # ties to even
    c = np.clip(c, -qmax, qmax)
    c = np.where(s == 0, 0.0, c)
    return c.astype(np.int8), s16


def dequantize(codes: np.ndarray, scale16: np.ndarray) -> np.ndarray:
    """c * s in float64 (exact: <= 7+11 significant bits)."""
    return codes.astype(np.float64) * scale16.astype(np.float64)[..., None]


def _pack_fields(u: np.ndarray, bits: int) -> np.ndarray:
    """Pack unsigned fields along the last axis; 4-bit: low nibble = even index."""
    u = u.astype(np.uint8)
    if bits == 8:
        return u
    assert bits == 4 and u.shape[-1] % 2 == 0
    return (u[..., 0::2] | (u[..., 1::2] << 4)).astype(np.uint8)


def _unpack_fields(b: np.ndarray, bits: int) -> np.ndarray:
    if bits == 8:
        return b.astype(np.uint8)
    out = np.empty(b.shape[:-1] + (b.shape[-1] * 2,), np.uint8)
    out[..., 0::2] = b & 0xF
    out[..., 1::2] = b >> 4
    return out


def _split_blocks(d: CacheDesc):
    """(start, n_hi, n_lo) of every K head block in the concatenated latent row."""
    out = []
    for off, r, rh in zip(d.k_offsets(), d.rank_k, d.rank_k_hi):
        out.append((off, rh, r - rh) if d.quantized else (off, r, 0))
    return out


def quantize_latents(d: CacheDesc, lk16: np.ndarray, lv16: np.ndarray):
    """Per-token, per-(head, precision block) quantisation of latent rows.
    Returns codes int8 [n, sum r_h + r_v] and scales fp16 [n, 2*H_kv + 2]
    (K: [h][blk], then V: [blk])."""
    n = lk16.shape[0]
    codes = np.zeros((n, d.sum_rank_k + d.rank_v), np.int8)
    scales = np.zeros((n, 2 * d.n_kv_heads + 2), np.float16)
    for h, (off, n_hi, n_lo) in enumerate(_split_blocks(d)):
        c, s = quantize_block(lk16[:, off:off + n_hi], d.bits_hi)
        codes[:, off:off + n_hi], scales[:, 2 * h] = c, s
        c, s = quantize_block(lk16[:, off + n_hi:off + n_hi + n_lo], d.bits_lo)
        codes[:, off + n_hi:off + n_hi + n_lo], scales[:, 2 * h + 1] = c, s
    vo, vh = d.sum_rank_k, d.rank_v_hi
    c, s = quantize_block(lv16[:, :vh], d.bits_hi)
    codes[:, vo:vo + vh], scales[:, 2 * d.n_kv_heads] = c, s
    c, s = quantize_block(lv16[:, vh:], d.bits_lo)
    codes[:, vo + vh:], scales[:, 2 * d.n_kv_heads + 1] = c, s
    return codes, scales


def pack_pages(d: CacheDesc, lk16: np.ndarray, lv16: np.ndarray) -> np.ndarray:
    """fp16 latents [n, sum r_h], [n, r_v] -> ceil(n/P) pages, uint8 [n_pages, page_bytes].
    Slots past n in the last page, and all padding bytes, are zero."""
    lay = page_layout(d)
    p = lay.page_tokens
    n = lk16.shape[0]
    assert lv16.shape[0] == n and lk16.shape[1] == d.sum_rank_k and lv16.shape[1] == d.rank_v
    n_pages = (n + p - 1) // p
    pages = np.zeros((n_pages, lay.page_bytes), np.uint8)
    if n == 0:
        return pages
    npad = n_pages * p
    valid = (np.arange(npad) < n).reshape(n_pages, p)

    def put_k(off, block_u8, rowbytes):
        # block: [npad, rowbytes] uint8, token-major rows
        pages[:, off:off + p * rowbytes] = block_u8.reshape(n_pages, p * rowbytes)

    def put_v(off, rows_u8):
        # rows_u8: [n_pages, ch, rowbytes]
        ch, rb = rows_u8.shape[1], rows_u8.shape[2]
        pages[:, off:off + ch * rb] = rows_u8.reshape(n_pages, ch * rb)

    if not d.quantized:
        lkp = np.zeros((npad, d.sum_rank_k), np.float16)
        lkp[:n] = lk16
        lvp = np.zeros((npad, d.rank_v), np.float16)
        lvp[:n] = lv16
        for h, (off, n_hi, _) in enumerate(_split_blocks(d)):
            put_k(lay.k_hi_off[h], np.ascontiguousarray(lkp[:, off:off + n_hi]).view(np.uint8), 2 * n_hi)
        vt = np.ascontiguousarray(lvp.reshape(n_pages, p, d.rank_v).transpose(0, 2, 1))  # [pg, ch, slot]
        put_v(lay.v_hi_off, vt.view(np.uint8).reshape(n_pages, d.rank_v, 2 * p))
        return pages

    codes, scales = quantize_latents(d, lk16, lv16)
    cp = np.zeros((npad, codes.shape[1]), np.int16)
    cp[:n] = codes
    sp = np.zeros((npad, scales.shape[1]), np.float16)
    sp[:n] = scales
    vmask = valid.reshape(npad, 1)

    def fields(c, bits):
        u = (c + (1 << (bits - 1))).astype(np.uint8)
        return np.where(vmask, u, 0).astype(np.uint8)          # unused slots -> field 0

    for h, (off, n_hi, n_lo) in enumerate(_split_blocks(d)):
        if n_hi:
            put_k(lay.k_hi_off[h], _pack_fields(fields(cp[:, off:off + n_hi], d.bits_hi), d.bits_hi),
                  n_hi * d.bits_hi // 8)
        if n_lo:
            put_k(lay.k_lo_off[h],
                  _pack_fields(fields(cp[:, off + n_hi:off + n_hi + n_lo], d.bits_lo), d.bits_lo),
                  n_lo * d.bits_lo // 8)
    # K scales [H][2][P]
    ks = sp[:, :2 * d.n_kv_heads].reshape(n_pages, p, d.n_kv_heads * 2).transpose(0, 2, 1)
    ks = np.ascontiguousarray(ks).view(np.uint8).reshape(n_pages, -1)
    pages[:, lay.k_scale_off:lay.k_scale_off + ks.shape[1]] = ks
    # V codes channel-major
    vo, vh = d.sum_rank_k, d.rank_v_hi
    for (c0, c1, off, bits) in ((vo, vo + vh, lay.v_hi_off, d.bits_hi),
                                (vo + vh, vo + d.rank_v, lay.v_lo_off, d.bits_lo)):
        if c1 == c0:
            continue
        u = fields(cp[:, c0:c1], bits).reshape(n_pages, p, c1 - c0).transpose(0, 2, 1)  # [pg, ch, slot]
        put_v(off, _pack_fields(np.ascontiguousarray(u), bits))
    vs = sp[:, 2 * d.n_kv_heads:].reshape(n_pages, p, 2).transpose(0, 2, 1)
    vs = np.ascontiguousarray(vs).view(np.uint8).reshape(n_pages, -1)
    pages[:, lay.v_scale_off:lay.v_scale_off + vs.shape[1]] = vs
    return pages


def unpack_pages(d: CacheDesc, pages: np.ndarray, n_tokens: int):
    """Inverse of pack_pages on the first n_tokens slots of consecutive pages.
    Returns dict(codes int8 [n, R] | None, scales uint16 [n, 2H+2] | None, dequant float64 [n, R])
    with R = sum r_h + r_v; dequant is exact (c*s, or the fp16 value)."""
    lay = page_layout(d)
    p = lay.page_tokens
    n_pages = (n_tokens + p - 1) // p
    pages = np.ascontiguousarray(pages[:n_pages]).reshape(n_pages, lay.page_bytes)
    R = d.sum_rank_k + d.rank_v
    npad = n_pages * p

    def get_k(off, rowbytes):
        return pages[:, off:off + p * rowbytes].reshape(npad, rowbytes)

    def get_v(off, ch, rowbytes):
        return pages[:, off:off + ch * rowbytes].reshape(n_pages, ch, rowbytes)

    if not d.quantized:
        deq = np.zeros((npad, R), np.float64)
        for h, (off, n_hi, _) in enumerate(_split_blocks(d)):
            deq[:, off:off + n_hi] = np.ascontiguousarray(get_k(lay.k_hi_off[h], 2 * n_hi)).view(np.float16)
        v = np.ascontiguousarray(get_v(lay.v_hi_off, d.rank_v, 2 * p)).view(np.float16)   # [pg, ch, slot]
        deq[:, d.sum_rank_k:] = v.transpose(0, 2, 1).reshape(npad, d.rank_v)
        return {"codes": None, "scales": None, "dequant": deq[:n_tokens]}

    codes = np.zeros((npad, R), np.int16)
    for h, (off, n_hi, n_lo) in enumerate(_split_blocks(d)):
        if n_hi:
            u = _unpack_fields(get_k(lay.k_hi_off[h], n_hi * d.bits_hi // 8), d.bits_hi)
            codes[:, off:off + n_hi] = u.astype(np.int16) - (1 << (d.bits_hi - 1))
        if n_lo:
            u = _unpack_fields(get_k(lay.k_lo_off[h], n_lo * d.bits_lo // 8), d.bits_lo)
            codes[:, off + n_hi:off + n_hi + n_lo] = u.astype(np.int16) - (1 << (d.bits_lo - 1))
    vo, vh = d.sum_rank_k, d.rank_v_hi
    for (c0, c1, off, bits) in ((vo, vo + vh, lay.v_hi_off, d.bits_hi),
                                (vo + vh, vo + d.rank_v, lay.v_lo_off, d.bits_lo)):
        if c1 == c0:
            continue
        u = _unpack_fields(get_v(off, c1 - c0, p * bits // 8), bits)            # [pg, ch, slot]
        codes[:, c0:c1] = u.transpose(0, 2, 1).reshape(npad, c1 - c0).astype(np.int16) - (1 << (bits - 1))
    nks = d.n_kv_heads * 2
    ks = np.ascontiguousarray(pages[:, lay.k_scale_off:lay.k_scale_off + nks * p * 2]).view(np.uint16)
    ks = ks.reshape(n_pages, nks, p).transpose(0, 2, 1).reshape(npad, nks)
    vs = np.ascontiguousarray(pages[:, lay.v_scale_off:lay.v_scale_off + 2 * p * 2]).view(np.uint16)
    vs = vs.reshape(n_pages, 2, p).transpose(0, 2, 1).reshape(npad, 2)
    scales = np.concatenate([ks, vs], axis=1)[:n_tokens].astype(np.uint16)
    codes = codes[:n_tokens]
    s = np.ascontiguousarray(scales).view(np.float16).astype(np.float64)
    # per-channel scale column
    col = np.zeros(R, np.int64)
    for h, (off, n_hi, n_lo) in enumerate(_split_blocks(d)):
        col[off:off + n_hi] = 2 * h
        col[off + n_hi:off + n_hi + n_lo] = 2 * h + 1
    col[vo:vo + vh] = nks
    col[vo + vh:] = nks + 1
    deq = codes.astype(np.float64) * s[:, col]
    return {"codes": codes.astype(np.int8), "scales": scales, "dequant": deq}


def write_token(d: CacheDesc, lay: PageLayout, page: np.ndarray, slot: int,
                zk16: np.ndarray, zv16: np.ndarray) -> None:
    """Quantise ONE token's fp16 latent rows and write them into ``page`` (uint8 view of one
    page, modified in place) at ``slot`` -- the append path's writer, written independently
    of pack_pages (tests check pack == repeated write_token)."""
    p = lay.page_tokens

    def put_nibble(byte_index, low, u):
        b = int(page[byte_index])
        page[byte_index] = (b & 0xF0) | u if low else (b & 0x0F) | (u << 4)

    def k_store(off, n, bits, z):
        if n == 0:
            return np.float16(0)
        if bits == 16:
            page[off + slot * 2 * n: off + (slot + 1) * 2 * n] = z.view(np.uint8)
            return None
        c, s = quantize_block(z[None, :], bits)
        u = (c[0].astype(np.int16) + (1 << (bits - 1))).astype(np.uint8)
        rb = n * bits // 8
        page[off + slot * rb: off + (slot + 1) * rb] = _pack_fields(u, bits)
        return s[0]

    def v_store(off, c0, n, bits):
        if n == 0:
            return np.float16(0)
        z = zv16[c0:c0 + n]
        if bits == 16:
            for ch in range(n):
                page[off + (ch * p + slot) * 2: off + (ch * p + slot) * 2 + 2] = z[ch:ch + 1].view(np.uint8)
            return None
        c, s = quantize_block(z[None, :], bits)
        u = (c[0].astype(np.int16) + (1 << (bits - 1))).astype(np.uint8)
        rb = p * bits // 8
        for ch in range(n):
            if bits == 8:
                page[off + ch * rb + slot] = u[ch]
            else:
                put_nibble(off + ch * rb + slot // 2, slot % 2 == 0, int(u[ch]))
        return s[0]

    for h, (off, n_hi, n_lo) in enumerate(_split_blocks(d)):
        s_hi = k_store(lay.k_hi_off[h], n_hi, d.bits_hi, zk16[off:off + n_hi])
        s_lo = k_store(lay.k_lo_off[h], n_lo, d.bits_lo, zk16[off + n_hi:off + n_hi + n_lo])
        if d.quantized:
            for blk, s in ((0, s_hi), (1, s_lo)):
                o = lay.k_scale_off + ((h * 2 + blk) * p + slot) * 2
                page[o:o + 2] = np.array([s], np.float16).view(np.uint8)
    if d.quantized:
        s_hi = v_store(lay.v_hi_off, 0, lay.v_hi_n, d.bits_hi)
        s_lo = v_store(lay.v_lo_off, lay.v_hi_n, lay.v_lo_n, d.bits_lo)
        for blk, s in ((0, s_hi), (1, s_lo)):
            o = lay.v_scale_off + (blk * p + slot) * 2
            page[o:o + 2] = np.array([s], np.float16).view(np.uint8)
    else:
        v_store(lay.v_hi_off, 0, lay.v_hi_n, 16)


def read_sequence(d: CacheDesc, pool: np.ndarray, table_row: np.ndarray, seq_len: int):
    """Gather one sequence's pages through its block-table row and dequantise:
    returns (L_k float64 [l, sum r_h], L_v float64 [l, r_v])."""
    lay = page_layout(d)
    n_pages = (seq_len + lay.page_tokens - 1) // lay.page_tokens
    if seq_len == 0:
        return np.zeros((0, d.sum_rank_k)), np.zeros((0, d.rank_v))
    idx = np.asarray(table_row[:n_pages], dtype=np.int64)
    assert (idx >= 0).all()
    deq = unpack_pages(d, pool.reshape(-1, lay.page_bytes)[idx], seq_len)["dequant"]
    return deq[:, :d.sum_rank_k], deq[:, d.sum_rank_k:]
