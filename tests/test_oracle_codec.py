"""Pins for oracle/codec.py and oracle/layout.py (CPU only).

P9  quantiser vs exact rational arithmetic (brute force), rounding lemma, invariants
P10 (part) byte accounting of the page layout
plus pack/unpack round trips and pack == repeated append-writer.
"""
from fractions import Fraction

import numpy as np
import pytest

import synth
from oracle import codec
from oracle.layout import CacheDesc, page_layout


def all_fp16_nonneg_finite():
    u = np.arange(0, 0x7C00, dtype=np.uint16)
    return u.view(np.float16)


def as_units(x16):
    """fp16 -> exact integer multiple of 2^-24 (int64)."""
    return np.round(x16.astype(np.float64) * 2.0 ** 24).astype(np.int64)


def rn_fp16_exact(num: int, den: int) -> np.float16:
    """Correctly rounded (RNE) fp16 of the rational num/den >= 0 by exact arithmetic."""
    if num == 0:
        return np.float16(0)
    q = Fraction(num, den)
    # find e with 2^e <= q < 2^(e+1)
    e = q.numerator.bit_length() - q.denominator.bit_length()
    if Fraction(2) ** e > q:
        e -= 1
    e = max(e, -14)                      # subnormal range shares the exponent of 2^-14
    ulp = Fraction(2) ** (e - 10)
    k = q / ulp
    f = k.numerator // k.denominator
    rem = k - f
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and f % 2 == 1):
        f += 1
    val = f * ulp
    if val >= 65520:
        return np.float16(np.inf)
    return np.float16(float(val))


@pytest.mark.parametrize("bits", [4, 8])
def test_scale_is_exactly_rounded(bits):
    """s = RN_fp16(a/qmax): the float64 route of the oracle equals exact-rational RN for every
    non-negative finite fp16 a (a sample of 4096 values through Fraction, all values through an
    integer-exact check)."""
    qmax = codec.qmax_of(bits)
    a = all_fp16_nonneg_finite()
    _, s = codec.quantize_block(a.reshape(-1, 1), bits)
    rng = np.random.default_rng(1)
    idx = np.concatenate([np.arange(0, 300), rng.choice(a.size, 3800, replace=False), [a.size - 1]])
    for i in idx:
        ka = int(as_units(a[i:i + 1])[0])
        want = rn_fp16_exact(ka, qmax * (1 << 24))
        assert s[i] == want, (float(a[i]), float(s[i]), float(want))
    # integer-exact check on ALL values: |a - qmax*s| must be <= qmax*ulp(s)/2
    ks = as_units(s)
    ka = as_units(a)
    sf = s.astype(np.float64)
    ulp = np.maximum(2.0 ** (np.floor(np.log2(np.maximum(sf, 2.0 ** -14))) - 10), 2.0 ** -24)
    assert np.all(np.abs(ka - qmax * ks) * 2 <= qmax * np.round(ulp * 2 ** 24).astype(np.int64))
    # s == 0 is reachable for small positive a (a/qmax below half the smallest subnormal)
    assert int(np.sum((s == 0) & (a > 0))) == {4: 3, 8: 63}[bits]


@pytest.mark.parametrize("bits", [4, 8])
def test_code_rounding_lemma(bits):
    """rint(z/s) in float64 AND in float32 equals the exactly-rounded (ties-to-even) quotient for
    every fp16 z with 0 <= z <= (qmax+1.5) s, over a few hundred scales s including all the
    smallest subnormals; reciprocal-multiply does NOT (so it is forbidden on the GPU side)."""
    qmax = codec.qmax_of(bits)
    vals = all_fp16_nonneg_finite()
    kall = as_units(vals)
    rng = np.random.default_rng(2)
    s_idx = np.unique(np.concatenate([np.arange(1, 130), rng.choice(np.arange(130, vals.size), 400, replace=False)]))
    n_pairs = n_ties = n_recip_bad = 0
    min_dist = 1.0
    for si in s_idx:
        ks = int(kall[si])
        zmask = kall <= int((qmax + 1.5) * ks)
        kz = kall[zmask]
        q, rem = kz // ks, kz % ks
        exact = q + ((2 * rem > ks) | ((2 * rem == ks) & (q % 2 == 1)))
        z64 = vals[zmask].astype(np.float64)
        s64 = np.float64(vals[si])
        got64 = np.rint(z64 / s64).astype(np.int64)
        got32 = np.rint(vals[zmask].astype(np.float32) / np.float32(vals[si])).astype(np.int64)
        assert np.array_equal(got64, exact)
        assert np.array_equal(got32, exact)
        rec = np.rint(vals[zmask].astype(np.float32) * (np.float32(1.0) / np.float32(vals[si]))).astype(np.int64)
        n_recip_bad += int(np.sum(rec != exact))
        n_pairs += kz.size
        n_ties += int(np.sum(2 * rem == ks))
        frac = rem.astype(np.float64) / ks
        dist = np.abs(frac - 0.5)
        dist = dist[dist > 0]
        if dist.size:
            min_dist = min(min_dist, float(dist.min()))
    assert n_pairs > 1e5
    assert n_ties > 0                 # exact .5 ties exist -> ties-to-even is load-bearing
    assert n_recip_bad > 0            # z * (1/s) is measurably wrong
    assert min_dist >= 2.0 ** -12     # never closer than 2^-12 to a half-integer unless it is one


def brute_force_codes(z16, s16, bits):
    """argmin_c |z - c s| over all codes in [-qmax, qmax], exact rationals, ties -> even c."""
    qmax = codec.qmax_of(bits)
    s = Fraction(float(s16))
    out = []
    for z in z16:
        zf = Fraction(float(z))
        best, bestd = None, None
        for c in range(-qmax, qmax + 1):
            dd = abs(zf - c * s)
            if bestd is None or dd < bestd or (dd == bestd and c % 2 == 0 and best % 2 != 0):
                best, bestd = c, dd
        out.append(best)
    return np.array(out, np.int8)


@pytest.mark.parametrize("bits", [4, 8])
def test_quantiser_matches_brute_force(bits):
    rng = np.random.default_rng(3 + bits)
    for trial in range(40):
        n = int(rng.choice([8, 16, 24]))
        scale = 10.0 ** rng.uniform(-6, 3)
        z = (rng.standard_normal(n) * scale).astype(np.float16)
        if trial % 5 == 0:                     # force exact ties: multiples of s/2
            z = (np.arange(n) - n // 2).astype(np.float16) * np.float16(0.5)
            z[0] = np.float16(codec.qmax_of(bits))   # absmax = qmax -> s = 1
        c, s = codec.quantize_block(z[None], bits)
        assert s[0] == rn_fp16_exact(int(as_units(np.abs(z)).max()), codec.qmax_of(bits) << 24)
        if s[0] == 0:
            assert not c.any()
            continue
        assert np.array_equal(c[0], brute_force_codes(z, s[0], bits))


@pytest.mark.parametrize("bits", [4, 8])
def test_quantiser_invariants(bits):
    qmax = codec.qmax_of(bits)
    rng = np.random.default_rng(5)
    z = (rng.standard_normal((500, 32)) * np.exp(rng.uniform(-8, 6, size=(500, 1)))).astype(np.float16)
    z = z[np.isfinite(z).all(axis=1)]
    c, s = codec.quantize_block(z, bits)
    zh = codec.dequantize(c, s)
    s64 = s.astype(np.float64)[:, None]
    z64 = z.astype(np.float64)
    clamped = np.abs(z64) > (qmax + 0.5) * s64
    assert np.all((np.abs(z64 - zh) <= s64 / 2 * (1 + 1e-12)) | clamped)
    # the absmax element maps to +-qmax whenever the scale is a normal fp16 number
    j = np.argmax(np.abs(z64), axis=1)
    normal = s64[:, 0] >= 2.0 ** -14
    assert np.all(np.abs(c[np.arange(len(j)), j])[normal] == qmax)
    assert np.all(np.abs(c.astype(np.int16)) <= qmax)
    # all-zero row and the s == 0 branch
    c0, s0 = codec.quantize_block(np.zeros((1, 8), np.float16), bits)
    assert s0[0] == 0 and not c0.any()
    tiny = np.full((1, 8), 2.0 ** -24, np.float16)
    c1, s1 = codec.quantize_block(tiny, bits)
    assert s1[0] == 0 and not c1.any()
    # clamp is reachable with subnormal scales: a = 10 * 2^-24 -> s = RN(10/7 * 2^-24) = 2^-24 (4-bit)
    if bits == 4:
        zc = np.array([[10 * 2.0 ** -24, 2.0 ** -24] + [0] * 6], np.float16)
        cc, sc = codec.quantize_block(zc, 4)
        assert float(sc[0]) == 2.0 ** -24 and cc[0, 0] == 7 and cc[0, 1] == 1
    # dequantised values are exactly representable in float32 (so GPU fp32 dequant is bit-comparable)
    assert np.array_equal(zh.astype(np.float32).astype(np.float64), zh)


def small_desc(bits, page_tokens=16):
    cfg = synth.custom_config("t", 1, 4, 2, 64, 100, [16, 40], 32, bits=bits, page_tokens=page_tokens,
                              outlier_frac=0.1)
    return cfg, CacheDesc.from_config(cfg)


@pytest.mark.parametrize("bits", [(16, 16), (8, 4), (8, 8), (4, 4)])
def test_layout_byte_accounting(bits):
    cfg, d = small_desc(bits, 32)
    lay = page_layout(d)
    per_tok = synth.algorithmic_bytes_per_token(cfg)["total"]
    # blocks are 16-B aligned and the page is the sum of blocks rounded to 128
    assert lay.page_bytes % 128 == 0
    assert lay.page_bytes >= per_tok * 32 and lay.page_bytes < per_tok * 32 + 128 + 16 * (2 * 2 + 4)
    offs = lay.k_hi_off + lay.k_lo_off + [lay.v_hi_off, lay.v_lo_off]
    if d.quantized:
        offs += [lay.k_scale_off, lay.v_scale_off]
    assert all(o % 16 == 0 for o in offs)
    # the C3 layer-0 page is exactly 64 x 348 B
    c3 = synth.make_config("C3")
    assert page_layout(CacheDesc.from_config(c3)).page_bytes == 64 * 348
    c2 = synth.make_config("C2")
    assert page_layout(CacheDesc.from_config(c2)).page_bytes == 64 * 1024


@pytest.mark.parametrize("bits", [(16, 16), (8, 4), (8, 8), (4, 4)])
@pytest.mark.parametrize("n", [1, 15, 16, 37, 100])
def test_pack_unpack_roundtrip(bits, n):
    cfg, d = small_desc(bits)
    lk, lv = synth.make_latents(cfg, n)
    pages = codec.pack_pages(d, lk, lv)
    un = codec.unpack_pages(d, pages, n)
    lat = np.concatenate([lk, lv], axis=1)
    if not d.quantized:
        assert np.array_equal(un["dequant"], lat.astype(np.float64))
        return
    codes, scales = codec.quantize_latents(d, lk, lv)
    assert np.array_equal(un["codes"], codes)
    assert np.array_equal(un["scales"], scales.view(np.uint16))
    # idempotence: pack(unpack(pack z)) == pack z
    deq16 = un["dequant"].astype(np.float16)
    re = codec.pack_pages(d, np.ascontiguousarray(deq16[:, :d.sum_rank_k]), np.ascontiguousarray(deq16[:, d.sum_rank_k:]))
    if np.array_equal(deq16.astype(np.float64), un["dequant"]):   # c*s representable in fp16
        assert np.array_equal(re, pages)
    # error bound per element: <= s/2 (no clamping happens when s is normal)
    s = scales.astype(np.float64)
    assert np.all(np.abs(un["dequant"] - lat.astype(np.float64)).max(axis=1) <= s.max(axis=1) / 2 + 1e-12)


@pytest.mark.parametrize("bits", [(16, 16), (8, 4), (4, 4)])
def test_pack_equals_repeated_token_writer(bits):
    cfg, d = small_desc(bits)
    lay = page_layout(d)
    n = 37
    lk, lv = synth.make_latents(cfg, n)
    pages = codec.pack_pages(d, lk, lv)
    pool = np.zeros_like(pages)
    for t in range(n):
        codec.write_token(d, lay, pool[t // lay.page_tokens], t % lay.page_tokens, lk[t], lv[t])
    assert np.array_equal(pool, pages)


def test_nibble_and_offset_binary_convention():
    """Hand-built page: one head r=8 (all hi), V r_v=8 (all hi), 4/4 bits, P=16."""
    cfg = synth.custom_config("t", 1, 1, 1, 64, 16, [8], 8, bits=(4, 4), page_tokens=16,
                              rank_k_hi=[8], rank_v_hi=8)
    d = CacheDesc.from_config(cfg)
    lay = page_layout(d)
    lk = np.zeros((2, 8), np.float16)
    lv = np.zeros((2, 8), np.float16)
    lk[0] = [7, -7, 1, 0, 2, -3, 0, 0]          # s = 1 -> codes as written
    lv[0, 0], lv[1, 0] = 7, -7                   # channel 0: slot0 = 7, slot1 = -7 (each s = 1)
    pg = codec.pack_pages(d, lk, lv)[0]
    assert list(pg[lay.k_hi_off[0]:lay.k_hi_off[0] + 4]) == [(7 + 8) | ((-7 + 8) << 4), (1 + 8) | (8 << 4),
                                                             (2 + 8) | ((-3 + 8) << 4), 8 | (8 << 4)]
    assert pg[lay.v_hi_off] == (7 + 8) | ((-7 + 8) << 4)          # low nibble = even slot
    assert pg[lay.v_hi_off + 8] == 8 | (8 << 4)                    # channel 1, slots 0,1: code 0 -> field 8
    assert pg[lay.v_hi_off + 1] == 0                               # slots 2,3 unused -> field 0
    ks = pg[lay.k_scale_off:lay.k_scale_off + 2].view(np.float16)[0]
    assert ks == np.float16(1.0)
    # lo block is empty (r_hi = r): its scale slot is written as 0
    assert not pg[lay.k_scale_off + 2 * 16: lay.k_scale_off + 2 * 16 + 4].any()
