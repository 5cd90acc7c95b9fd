"""Pins for oracle/attention.py, oracle/append.py (CPU only).  Pin numbers: DESIGN.md "Oracle pins".

Each test fixes the oracle against something other than itself: a closed form, a textbook
special case computed without the latent machinery, or an invariant the mathematics imposes.
"""
import numpy as np
import pytest

import synth
from oracle import analysis, append as oappend, attention as oattn, codec
from oracle.layout import CacheDesc, page_layout
from tests.util import build_cache, row_rel_err


def fullrank_case(seed=0, l=70, hq=4, hkv=2, dh=16, P=16):
    """Full-rank latent cache built from explicit dense projections: K = X M_k^T, V = X M_v^T."""
    rng = np.random.default_rng(seed)
    dmodel = 40
    X = rng.standard_normal((l, dmodel))
    Mk = [rng.standard_normal((dh, dmodel)) for _ in range(hkv)]          # W_K per head [d_out, d_in]
    Mv = rng.standard_normal((hkv * dh, dmodel))
    cfg = synth.custom_config("fr", 1, hq, hkv, dh, l, [dh] * hkv, hkv * dh, page_tokens=P)
    return rng, X, Mk, Mv, cfg


def test_P1_full_rank_equals_dense_attention():
    """Full rank + orthonormal SVD factors + no quantisation == textbook attention on K = X W_K^T,
    V = X W_V^T computed WITHOUT the factors.  The cache must hold fp16, so X and
    the factors are chosen such that the latents are exactly fp16-representable: we round the latent
    to fp16 and define the dense K, V from the rounded latent through the exact inverse."""
    rng, X, Mk, Mv, cfg = fullrank_case()
    d = CacheDesc.from_config(cfg)
    l, dh, hkv = X.shape[0], cfg.head_dim, cfg.n_kv_heads
    lk = np.zeros((l, d.sum_rank_k))
    bk = np.zeros((d.sum_rank_k, dh))
    Kdense = np.zeros((l, hkv, dh))
    for h in range(hkv):
        A, B, _ = analysis.svd_factors(Mk[h], dh)           # full rank: exact
        B16 = B.astype(np.float16).astype(np.float64)
        z = (X @ A).astype(np.float16).astype(np.float64)   # what the cache stores
        lk[:, h * dh:(h + 1) * dh] = z
        bk[h * dh:(h + 1) * dh] = B16
        # textbook K for these stored values, computed without the oracle: K = z B16
        Kdense[:, h] = np.einsum("tr,rd->td", z, B16)
    Av, Bv, _ = analysis.svd_factors(Mv, hkv * dh)
    Bv16 = Bv.astype(np.float16).astype(np.float64)
    zv = (X @ Av).astype(np.float16).astype(np.float64)
    Vdense = np.einsum("tr,rd->td", zv, Bv16).reshape(l, hkv, dh)
    q16 = rng.standard_normal((1, cfg.n_q_heads, dh)).astype(np.float16)
    c = build_cache(cfg, latents=[(lk.astype(np.float16), zv.astype(np.float16))])
    out = oattn.decode_attn(d, q16, c["pool"], c["table"], c["seq_lens"], bk.astype(np.float16), Bv.astype(np.float16))
    ref = oattn.dense_attention(q16[0].astype(np.float64), Kdense, Vdense, d.sm_scale, d.group)
    assert np.abs(out[0] - ref).max() <= 1e-12 * max(1.0, np.abs(ref).max())
    # and: with exact (fp64) factors the reconstruction really is X W^T (the factorisation is right)
    A, B, _ = analysis.svd_factors(Mk[0], dh)
    assert np.allclose((X @ A) @ B, X @ Mk[0].T, atol=1e-10)
    assert np.allclose((X @ Av) @ Bv, X @ Mv.T, atol=1e-10)


@pytest.mark.parametrize("bits", [(16, 16), (8, 4)])
def test_P2_absorbed_identity(bits):
    cfg = synth.custom_config("t", 2, 8, 2, 32, 150, [8, 24], 32, bits=bits, page_tokens=16, outlier_frac=0.1)
    c = build_cache(cfg, seq_lens=[150, 77])
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    a = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    b = oattn.decode_attn_absorbed(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    assert np.abs(a - b).max() <= 1e-12 * np.abs(a).max()


def test_P3_zero_query_gives_mean_value():
    cfg = synth.custom_config("t", 1, 4, 2, 32, 90, [16, 16], 32, page_tokens=16)
    c = build_cache(cfg)
    bk, bv = synth.make_factors(cfg)
    q = np.zeros((1, 4, 32), np.float16)
    out = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    lv = c["lat"][0][1].astype(np.float64)
    mean_v = lv.mean(axis=0) @ bv.astype(np.float64)              # [H_kv*d_h]
    for i in range(4):
        g = i // 2
        assert np.allclose(out[0, i], mean_v[g * 32:(g + 1) * 32], rtol=0, atol=1e-13)


def test_P4_dominant_score_selects_that_token():
    cfg = synth.custom_config("t", 1, 2, 1, 32, 64, [32], 32, page_tokens=16)
    bk, bv = synth.make_factors(cfg)
    lk, lv = synth.make_latents(cfg, 64)
    q = synth.make_q(cfg)
    # make token 17's key the (scaled) latent image of q for head 0: score_17 >> others
    qt = bk.astype(np.float64) @ q[0, 0].astype(np.float64)
    lk = (lk.astype(np.float64) * 0.01)
    lk[17] = 40.0 * qt / np.linalg.norm(qt)
    c = build_cache(cfg, latents=[(lk.astype(np.float16), lv)])
    out = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv, heads=[0])
    v17 = lv[17].astype(np.float64) @ bv.astype(np.float64)
    assert np.allclose(out[0, 0], v17[:32], atol=1e-9)


def test_P5_indexing_paging_and_head_permutation():
    cfg = synth.custom_config("t", 2, 4, 2, 32, 70, [8, 24], 32, bits=(8, 4), page_tokens=16)
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    c = build_cache(cfg, seq_lens=[70, 1], shuffle=True)
    d = c["desc"]
    out = oattn.decode_attn(d, q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    # seq_len = 1  =>  out = dequantised V row 0 (softmax over one token is 1)
    un = codec.unpack_pages(d, c["pool"][c["table"][1, :1]], 1)["dequant"][0]
    v0 = un[d.sum_rank_k:] @ bv.astype(np.float64)
    for i in range(4):
        assert np.allclose(out[1, i], v0[(i // 2) * 32:(i // 2 + 1) * 32], atol=1e-14)
    # physical page order is irrelevant
    c2 = build_cache(cfg, seq_lens=[70, 1], shuffle=False)
    out2 = oattn.decode_attn(d, q, c2["pool"], c2["table"], c2["seq_lens"], bk, bv)
    assert not np.array_equal(c["table"], c2["table"])
    assert np.array_equal(out, out2)
    # swapping the two KV heads (rank table, latents, B_k rows, B_v column blocks, q groups) swaps outputs
    cfgp = synth.custom_config("t", 2, 4, 2, 32, 70, [24, 8], 32, bits=(8, 4), page_tokens=16)
    latp = []
    for lk, lv in c["lat"]:
        latp.append((np.concatenate([lk[:, 8:], lk[:, :8]], axis=1), lv))
    cp = build_cache(cfgp, seq_lens=[70, 1], latents=latp)
    bkp = np.concatenate([bk[8:], bk[:8]], axis=0)
    bvp = np.concatenate([bv[:, 32:], bv[:, :32]], axis=1)
    qp = np.concatenate([q[:, 2:], q[:, :2]], axis=1)
    outp = oattn.decode_attn(cp["desc"], qp, cp["pool"], cp["table"], cp["seq_lens"], bkp, bvp)
    assert np.allclose(outp, np.concatenate([out[:, 2:], out[:, :2]], axis=1), atol=1e-13)


def test_P6_split_and_lse_merge_equals_single_pass():
    cfg = synth.custom_config("t", 1, 4, 2, 32, 200, [16, 32], 48, bits=(8, 4), page_tokens=16, outlier_frac=0.1)
    c = build_cache(cfg, regime="peaky")
    d = c["desc"]
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    ref = oattn.decode_attn(d, q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    Lk, Lv = codec.read_sequence(d, c["pool"], c["table"][0], 200)
    parts = [oattn.partial_attn(d, q, Lk[a:b], Lv[a:b], bk, bv, 0) for a, b in ((0, 64), (64, 65), (65, 200))]
    assert np.allclose(oattn.lse_merge(parts), ref[0], rtol=1e-12, atol=1e-14)


def test_P14_gqa_heads_with_identical_query_agree():
    cfg = synth.custom_config("t", 1, 8, 2, 32, 64, [16, 32], 32, page_tokens=16)
    c = build_cache(cfg)
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    q[0, 1] = q[0, 0]
    q[0, 3] = q[0, 0]
    q[0, 4] = q[0, 0]           # different group: must differ
    out = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    assert np.array_equal(out[0, 0], out[0, 1]) and np.array_equal(out[0, 0], out[0, 3])
    assert not np.allclose(out[0, 0], out[0, 4])


@pytest.mark.parametrize("N,D,vscale", [(4095, 10.0, 1e-3), (4095, 14.0, 1e-3),
                                        (131071, 10.0, 1e-3), (131071, 12.0, 3e-2), (131071, 14.0, 1e-3), (131071, 16.0, 3e-2)])
def test_P16_one_dominant_token_over_many_equal_ones(N, D, vscale):
    """Closed form: token 0 at score +D over N equal tokens of score 0, constant codes:
    out = (v0 + N e^-D v) / (1 + N e^-D).  N = 131071 with value scales 1e-3 and 3e-2 is SURVEY's P16 size (the
    128K underflow regime of the headline configuration)."""
    cfg = synth.custom_config("t", 1, 1, 1, 16, N + 1, [8], 8, bits=(8, 4), page_tokens=64,
                              rank_k_hi=[8], rank_v_hi=8)
    d = CacheDesc.from_config(cfg)
    bk = np.zeros((8, 16), np.float16)
    bk[np.arange(8), np.arange(8)] = 1
    bv = bk.copy()
    q = np.zeros((1, 1, 16), np.float16)
    q[0, 0, 0] = 4.0                                   # sm_scale = 1/4 -> score = latent channel 0
    lk = np.zeros((N + 1, 8), np.float16)
    lk[0, 0] = D                                       # exactly representable after 8-bit quant: absmax -> qmax
    lv = np.full((N + 1, 8), vscale, np.float16)
    lv[0] = 0.5
    c = build_cache(cfg, latents=[(lk, lv)])
    un = codec.unpack_pages(d, c["pool"][c["table"][0]], N + 1)["dequant"]
    Dq = un[0, 0]
    v0, v = un[0, 8:], un[1, 8:]
    want = (v0 + N * np.exp(-Dq) * v) / (1 + N * np.exp(-Dq))
    out = oattn.decode_attn(d, q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    assert np.allclose(out[0, 0, :8], want, rtol=1e-12)
    assert abs(Dq - D) < 0.05


def test_seq_len_zero_gives_zeros():
    cfg = synth.custom_config("t", 2, 2, 1, 16, 32, [8], 8, page_tokens=16)
    c = build_cache(cfg, seq_lens=[0, 20])
    bk, bv = synth.make_factors(cfg)
    out = oattn.decode_attn(c["desc"], synth.make_q(cfg), c["pool"], c["table"], c["seq_lens"], bk, bv)
    assert not out[0].any() and out[1].any()


# ------------------------------------------------------------------ append

def test_P17_hidden_state_and_dense_kv_modes_give_same_latent():
    """With W = U S V^T:  x (V S)_r  ==  (x W^T) U_r   (U^T U_r = [I;0])."""
    rng = np.random.default_rng(11)
    dh, dmodel, r = 16, 40, 8
    W = rng.standard_normal((dh, dmodel))
    x = rng.standard_normal((5, dmodel))
    A, B, _ = analysis.svd_factors(W, r)
    hidden_mode = x @ A
    dense_mode = (x @ W.T) @ B.T                       # dense K row times A_dense = U_r = B^T
    assert np.allclose(hidden_mode, dense_mode, atol=1e-12)


def test_append_hidden_state_mode_against_a_per_head_loop_and_the_dense_mode():
    """oracle.append.project_latents in HIDDEN-STATE mode (k_head_stride = 0, d_in = d_model; §3.2
    K' = x (Sigma V)_K): every KV head reads the SAME input row and its own columns of A_k.  Pinned (i) against an
    explicit scalar loop per head and column, and (ii) through W = U S V^T against the dense-KV mode of the same
    routine (k_head_stride = d_h), which must give the same latent: x (V S)_r == (x W^T) U_r.  A stride mistake in
    either mode fails one of the two."""
    rng = np.random.default_rng(23)
    dmodel, dh, n = 24, 16, 5
    cfg = synth.custom_config("t", 1, 4, 2, dh, 32, [8, 16], 16, page_tokens=16)
    d = CacheDesc.from_config(cfg)
    # dyadic-grid inputs so that every sum is exact in double and in fp16 after one rounding
    x = (rng.integers(-8, 9, size=(n, dmodel)) / 8.0).astype(np.float16)
    ak = (rng.integers(-16, 17, size=(dmodel, d.sum_rank_k)) / 16.0 * (rng.random((dmodel, d.sum_rank_k)) < 0.3)).astype(np.float16)
    av = (rng.integers(-16, 17, size=(dmodel, d.rank_v)) / 16.0 * (rng.random((dmodel, d.rank_v)) < 0.3)).astype(np.float16)
    lk, lv = oappend.project_latents(d, x, 0, dmodel, x, ak, av)
    for t in range(n):
        for h, (off, r) in enumerate(zip(d.k_offsets(), d.rank_k)):
            for c in range(r):
                acc = 0.0
                for j in range(dmodel):
                    acc += float(x[t, j]) * float(ak[j, off + c])
                assert np.float16(acc) == lk[t, off + c], (t, h, c)
        for c in range(d.rank_v):
            acc = sum(float(x[t, j]) * float(av[j, c]) for j in range(dmodel))
            assert np.float16(acc) == lv[t, c]
    # (ii) the two modes of the same routine agree through an SVD: head h projects x with W_h = U S V^T
    xs = rng.standard_normal((n, dmodel))
    lat_hidden = np.zeros((n, d.sum_rank_k))
    a_hidden = np.zeros((dmodel, d.sum_rank_k))
    a_dense = np.zeros((dh, d.sum_rank_k))
    kd = np.zeros((n, d.n_kv_heads, dh))
    for h, (off, r) in enumerate(zip(d.k_offsets(), d.rank_k)):
        W = rng.standard_normal((dh, dmodel))
        A, B, _ = analysis.svd_factors(W, r)          # A = (V S)_r [dmodel, r], B = U_r^T [r, dh]
        a_hidden[:, off:off + r] = A
        a_dense[:, off:off + r] = B.T
        kd[:, h] = xs @ W.T
        lat_hidden[:, off:off + r] = xs @ A
    # (fp16 storage of inputs and factors perturbs both sides by ~2^-11 per term)
    got_hidden, _ = oappend.project_latents(d, xs.astype(np.float16), 0, dmodel, xs.astype(np.float16), a_hidden.astype(np.float16), av)
    got_dense, _ = oappend.project_latents(d, kd.reshape(n, -1).astype(np.float16), dh, dh, xs.astype(np.float16), a_dense.astype(np.float16), av)
    scale = np.abs(lat_hidden).max()
    assert np.abs(got_hidden.astype(np.float64) - lat_hidden).max() <= 4e-3 * scale * np.sqrt(dmodel)
    assert np.abs(got_dense.astype(np.float64) - lat_hidden).max() <= 4e-3 * scale * np.sqrt(dmodel)
    # and a deliberately wrong stride is caught by (ii): dense inputs read with stride 0 give head 0's row to every head
    wrong, _ = oappend.project_latents(d, kd.reshape(n, -1).astype(np.float16), 0, dh, xs.astype(np.float16), a_dense.astype(np.float16), av)
    off1 = d.k_offsets()[1]
    assert np.abs(wrong.astype(np.float64)[:, off1:] - lat_hidden[:, off1:]).max() > 0.1 * scale


def test_append_projection_is_plain_matmul_and_rounds_once():
    cfg = synth.custom_config("t", 1, 4, 2, 16, 32, [8, 16], 16, page_tokens=16)
    d = CacheDesc.from_config(cfg)
    k, v, ak, av = synth.dyadic_append_case(cfg, 6, 16, 32)
    lk, lv = oappend.project_latents(d, k.reshape(6, -1), 16, 16, v, ak, av)
    # dyadic inputs: the sum is exact in float32 in any order -> compare with a float32 loop in reverse order
    for t in range(6):
        for h, (off, r) in enumerate(zip(d.k_offsets(), d.rank_k)):
            for c in range(r):
                acc = np.float32(0)
                for j in reversed(range(16)):
                    acc += np.float32(k[t, h, j]) * np.float32(ak[j, off + c])
                assert np.float16(acc) == lk[t, off + c]
    assert np.array_equal(lv, (v.astype(np.float32) @ av.astype(np.float32)).astype(np.float16))


@pytest.mark.parametrize("bits", [(16, 16), (8, 4)])
def test_append_then_decode_equals_pack_then_decode(bits):
    """Appending tokens one call at a time (out of order, two sequences) produces the same pages as
    packing the projected latents."""
    cfg = synth.custom_config("t", 2, 4, 2, 16, 40, [8, 16], 16, bits=bits, page_tokens=16)
    d = CacheDesc.from_config(cfg)
    lay = page_layout(d)
    ak, av = synth.make_append_factors(cfg, 16, 32)
    seq_lens = np.array([40, 23], np.int32)
    table, n_pool = synth.make_block_table(cfg, seq_lens)
    pool = np.zeros((n_pool, lay.page_bytes), np.uint8)
    k, v = synth.make_append_inputs(cfg, 63)
    seq_ids = np.array([0] * 40 + [1] * 23)
    pos = np.concatenate([np.arange(40), np.arange(23)])
    order = np.random.default_rng(0).permutation(63)
    oappend.append(d, pool, table, seq_ids[order], pos[order], k.reshape(63, -1)[order], 16, 16, v[order], ak, av)
    lk, lv = oappend.project_latents(d, k.reshape(63, -1), 16, 16, v, ak, av)
    want = np.zeros_like(pool)
    want[table[0, :3]] = codec.pack_pages(d, lk[:40], lv[:40])
    want[table[1, :2]] = codec.pack_pages(d, lk[40:], lv[40:])
    assert np.array_equal(pool, want)


# ------------------------------------------------------------------ synthetic-input regimes

def test_regimes_are_what_design_md_says():
    """diffuse: many tokens attended; peaky: few.  (n_eff = 1/sum p^2, oracle diagnostic.)"""
    cfg = synth.make_config("C3", context=4096)
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    for regime in ("diffuse", "peaky"):
        c = build_cache(cfg, regime=regime)
        diag = {}
        oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv, diag=diag)
        ne = diag["n_eff"][0]
        if regime == "diffuse":
            assert np.median(ne) >= 4096 / 16 and ne.min() >= 4096 / 256, ne
        else:
            assert np.median(ne) <= 200, ne


# ------------------------------------------------------------------ NEXT-1: the paper's RoPE key path (oracle only)

ROPE_THETA = 10000.0


def _rope_case(l=37):
    cfg = synth.custom_config("t", 2, 4, 2, 16, l, [8, 16], 16, bits=(8, 4), page_tokens=16)
    c = build_cache(cfg, seq_lens=[l, l - 9])
    bk, bv = synth.make_factors(cfg)
    return cfg, c, bk, bv, synth.make_q(cfg)


def test_rope_is_a_rotation():
    """Position 0 is the identity, norms are preserved, and the inner product of two rotated vectors depends on the
    position difference only (Su et al. 2024, the property PAPER.md §3.3 L62-68 relies on)."""
    rng = np.random.default_rng(5)
    x, y = rng.standard_normal((7, 16)), rng.standard_normal((7, 16))
    assert np.array_equal(oattn.rope_rotate(x, np.zeros(7), ROPE_THETA), x)
    pos = np.arange(7) * 13
    rx = oattn.rope_rotate(x, pos, ROPE_THETA)
    assert np.allclose(np.linalg.norm(rx, axis=1), np.linalg.norm(x, axis=1), rtol=1e-13)
    a = np.sum(oattn.rope_rotate(x, pos + 5, ROPE_THETA) * oattn.rope_rotate(y, pos, ROPE_THETA), axis=1)
    b = np.sum(oattn.rope_rotate(x, pos + 905, ROPE_THETA) * oattn.rope_rotate(y, pos + 900, ROPE_THETA), axis=1)
    assert np.allclose(a, b, rtol=1e-10)


def test_rope_all_tokens_at_one_position_is_the_position_free_path():
    """Every key AND the query at the same position (pos_stride = 0): all relative positions are 0, so the RoPE path
    must equal decode_attn -- it pins the reconstruct / rotate / score order and the value side against the pinned
    position-free oracle."""
    cfg, c, bk, bv, q = _rope_case()
    want = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    for p in (0, 123):
        qr = np.stack([oattn.rope_rotate(q[b].astype(np.float64), np.full(cfg.n_q_heads, p), ROPE_THETA) for b in range(2)])
        got = oattn.decode_attn_rope(c["desc"], qr, c["pool"], c["table"], c["seq_lens"], bk, bv, ROPE_THETA,
                                     pos_offset=[p, p], pos_stride=0)
        assert np.allclose(got, want, rtol=1e-10, atol=1e-13)


def test_rope_output_is_invariant_to_a_common_position_offset():
    cfg, c, bk, bv, q = _rope_case()
    lens = c["seq_lens"]
    outs = []
    for off in (0, 1000):
        qr = np.stack([oattn.rope_rotate(q[b].astype(np.float64), np.full(cfg.n_q_heads, lens[b] - 1 + off), ROPE_THETA)
                       for b in range(2)])
        outs.append(oattn.decode_attn_rope(c["desc"], qr, c["pool"], c["table"], lens, bk, bv, ROPE_THETA, pos_offset=[off, off]))
    assert np.allclose(outs[0], outs[1], rtol=1e-9, atol=1e-12)
    # and it is NOT the position-free result (the rotation does something)
    plain = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], lens, bk, bv)
    assert np.abs(outs[0] - plain).max() > 1e-3


def test_rope_hand_computed_two_token_case():
    """Full rank, identity factors, fp16 latents, d_h = 16: both keys are e_0 before RoPE; channel 0 pairs with channel 8
    at frequency theta^0 = 1, so RoPE(k, position 1) = cos(1) e_0 + sin(1) e_8.  With q = 2 e_0 and sm_scale = 1/sqrt 2:
    s0 = sqrt 2, s1 = sqrt 2 cos 1; values v0 = e_0, v1 = e_1."""
    d = CacheDesc(n_q_heads=1, n_kv_heads=1, head_dim=16, rank_k=[16], rank_k_hi=[16], rank_v=16, rank_v_hi=16,
                  bits_hi=16, bits_lo=16, page_tokens=16, sm_scale=1.0 / np.sqrt(2.0))
    lk = np.zeros((2, 16), np.float16)
    lk[:, 0] = 1.0
    lv = np.zeros((2, 16), np.float16)
    lv[0, 0] = 1.0
    lv[1, 1] = 1.0
    pages = codec.pack_pages(d, lk, lv)
    eye = np.eye(16, dtype=np.float16)
    q = np.zeros((1, 1, 16), np.float16)
    q[0, 0, 0] = 2.0
    out = oattn.decode_attn_rope(d, q, pages, np.array([[0]], np.int32), [2], eye, eye, theta=ROPE_THETA)
    s0, s1 = np.sqrt(2.0), np.sqrt(2.0) * np.cos(1.0)
    w1 = np.exp(s1 - s0) / (1 + np.exp(s1 - s0))
    want = np.zeros(16)
    want[0], want[1] = 1 - w1, w1
    assert np.allclose(out[0, 0], want, rtol=1e-13, atol=1e-15)


# ---- NEXT-3 (latent-output mode): decode_attn_latent --------------------------------------------
@pytest.mark.parametrize("bits", [(16, 16), (8, 4)], ids=str)
def test_latent_output_up_projected_is_the_dense_output(bits):
    """PAPER.md section 3.3: (p . V') . U_V = p . (V' U_V).  The latent rows times each head's slice of B_v must be the
    output of the (pinned) decode_attn, which multiplies in the other order -- ragged lengths, quantised cache, GQA."""
    cfg = synth.custom_config("t", 2, 8, 4, 32, 150, [8, 16, 24, 32], 48, bits=bits, page_tokens=16, outlier_frac=0.1)
    c = build_cache(cfg, seq_lens=[150, 67])
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg)
    lat = oattn.decode_attn_latent(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk)
    want = oattn.decode_attn(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, bv)
    assert lat.shape == (2, 8, 48)
    bvf = bv.astype(np.float64)
    for i in range(8):
        g = i // 2
        assert np.allclose(lat[:, i] @ bvf[:, g * 32:(g + 1) * 32], want[:, i], rtol=1e-11, atol=1e-13)


def test_latent_output_of_a_zero_query_is_the_mean_latent_row():
    """Closed form: equal scores -> uniform weights -> the mean of the cached value latents, the same row for every head."""
    cfg = synth.custom_config("t", 1, 4, 2, 32, 90, [16, 16], 32, page_tokens=16)
    c = build_cache(cfg)
    bk, _ = synth.make_factors(cfg)
    out = oattn.decode_attn_latent(c["desc"], np.zeros((1, 4, 32), np.float16), c["pool"], c["table"], c["seq_lens"], bk)
    mean_l = c["lat"][0][1].astype(np.float64).mean(axis=0)
    for i in range(4):
        assert np.allclose(out[0, i], mean_l, rtol=0, atol=1e-13)


def test_latent_output_of_a_dominant_token_is_its_latent_row_and_empty_sequences_give_zeros():
    cfg = synth.custom_config("t", 2, 2, 1, 32, 64, [32], 32, page_tokens=16)
    bk, _ = synth.make_factors(cfg)
    lk, lv = synth.make_latents(cfg, 64)
    q = synth.make_q(cfg)
    qt = bk.astype(np.float64) @ q[0, 0].astype(np.float64)
    lk = lk.astype(np.float64) * 0.01
    lk[17] = 40.0 * qt / np.linalg.norm(qt)
    c = build_cache(cfg, seq_lens=[64, 0], latents=[(lk.astype(np.float16), lv), (lk.astype(np.float16)[:0], lv[:0])])
    out = oattn.decode_attn_latent(c["desc"], q, c["pool"], c["table"], c["seq_lens"], bk, heads=[0])
    assert np.allclose(out[0, 0], lv[17].astype(np.float64), atol=1e-9)
    assert not out[1].any()
