"""GPU parity, codec and append: starkv_pack / starkv_unpack / starkv_append through the C ABI against
the CPU oracle, bit-exact (page bytes, codes, scale bits; append on dyadic-grid inputs -- pin P15)."""
import numpy as np
import pytest
import torch

import synth
from oracle import append as oappend
from oracle import codec as ocodec
from oracle.layout import CacheDesc, page_layout
from tests.gpu_util import dev, f16

pytestmark = pytest.mark.gpu
sk = pytest.importorskip("paper_2606_08382_b200")


def cfgs():
    out = [synth.make_config("C1")]
    out.append(synth.make_config("C3", context=300, batch=1))
    out.append(synth.make_config("C4", context=200, batch=1))
    out.append(synth.make_config("C2", context=130, batch=1))
    # r_hi == r (empty trailing block), 8/8 and 4/4 pairs, other page sizes
    out.append(synth.custom_config("e88", 1, 8, 2, 64, 100, [8, 40], 48, bits=(8, 8)))
    out.append(synth.custom_config("e44", 1, 8, 4, 128, 77, [8, 16, 96, 128], 80, bits=(4, 4), outlier_frac=0.2))
    out.append(synth.custom_config("p32", 1, 4, 4, 64, 70, [16, 24, 32, 64], 40, bits=(8, 4), page_tokens=32,
                                   rank_v_hi=8))
    out.append(synth.custom_config("p128", 1, 4, 2, 64, 300, [16, 24], 64, bits=(8, 4), page_tokens=128))
    return out


@pytest.mark.parametrize("cfg", cfgs(), ids=lambda c: c.name)
def test_pack_bit_exact_and_unpack(cfg):
    d = CacheDesc.from_config(cfg)
    lay = page_layout(d)
    n = cfg.context
    lk, lv = synth.make_latents(cfg, n, regime="peaky")
    lk[3] = 0          # an all-zero token: scale 0, codes 0
    lv[5] = 0
    lk[7, :] = np.float16(6.0e-8)   # subnormal row: tiny scale, clamp reachable
    ref = ocodec.pack_pages(d, lk, lv)
    ctx = sk.create_from_config(cfg)
    assert sk.starkv_page_bytes(ctx) == lay.page_bytes
    pages = torch.full((ref.shape[0], lay.page_bytes), 0xAB, dtype=torch.uint8, device="cuda")
    sk.starkv_pack(ctx, f16(lk), f16(lv), n, pages)
    torch.cuda.synchronize()
    got = pages.cpu().numpy()
    bad = np.nonzero(got != ref)
    assert bad[0].size == 0, f"{bad[0].size} bytes differ, first at page {bad[0][:3]} byte {bad[1][:3]}"

    R = d.sum_rank_k + d.rank_v
    deq = torch.empty((n, R), dtype=torch.float32, device="cuda")
    codes = torch.empty((n, R), dtype=torch.int8, device="cuda")
    scales = torch.empty((n, 2 * d.n_kv_heads + 2), dtype=torch.int16, device="cuda")
    sk.starkv_unpack(ctx, pages, n, codes if d.quantized else None, scales if d.quantized else None, deq)
    torch.cuda.synchronize()
    want = ocodec.unpack_pages(d, ref, n)
    assert np.array_equal(deq.cpu().numpy().astype(np.float64), want["dequant"])
    if d.quantized:
        assert np.array_equal(codes.cpu().numpy(), want["codes"])
        assert np.array_equal(scales.cpu().numpy().view(np.uint16), want["scales"])


def test_pack_empty_is_a_no_op():
    cfg = synth.make_config("C1")
    ctx = sk.create_from_config(cfg)
    sk.starkv_pack(ctx, None, None, 0, None)
    sk.starkv_unpack(ctx, None, 0)


def _append_case(cfg, mode, n_new, dyadic, pad=0, tc5=True, ordered=False):
    d = CacheDesc.from_config(cfg)
    lay = page_layout(d)
    rng = np.random.default_rng(5)
    B = 3
    lens = np.array([70, 0, 129], np.int32)                       # existing tokens per sequence
    tot = lens + np.array([n_new, n_new // 2, n_new // 3 + 1])
    cfgb = synth.custom_config("x", B, 1, 1, 16, int(tot.max()), [8], 8, page_tokens=cfg.page_tokens)
    table, n_pool = synth.make_block_table(cfgb, tot)
    pool = rng.integers(0, 256, size=(n_pool, lay.page_bytes), dtype=np.uint8)  # pre-existing bytes must survive
    seq_ids, positions = [], []
    for b in range(B):
        for p in range(int(lens[b]), int(tot[b])):
            seq_ids.append(b)
            positions.append(p)
    order = np.arange(len(seq_ids)) if ordered else rng.permutation(len(seq_ids))
    seq_ids = np.array(seq_ids, np.int32)[order]
    positions = np.array(positions, np.int32)[order]
    n = len(seq_ids)
    if mode == "dense":
        d_in_k, d_in_v, khs = cfg.head_dim, cfg.n_kv_heads * cfg.head_dim, cfg.head_dim
    else:
        d_in_k = d_in_v = cfg.d_model
        khs = 0
    if dyadic:
        k, v, ak, av = synth.dyadic_append_case(cfg, n, d_in_k, d_in_v)
        if mode == "hidden":
            k = k[:, 0, :]
            v = k
    else:
        ak, av = synth.make_append_factors(cfg, d_in_k, d_in_v)
        k, v = synth.make_append_inputs(cfg, n, mode)
        if v is None:
            v = k
    k2 = np.ascontiguousarray(k.reshape(n, -1))
    v2 = np.ascontiguousarray(v.reshape(n, -1))
    ref = pool.copy()
    kw, vw = k2.shape[1], v2.shape[1]
    oappend.append(d, ref, table, seq_ids, positions, k2, khs, d_in_k, v2, ak, av)
    ctx = sk.create_from_config(cfg)
    sk.starkv_set_option(ctx, "append_tc5", 1 if tc5 else 0)
    dpool = dev(pool)
    wsb = sk.starkv_append_workspace_bytes(ctx, n)
    ws = torch.empty(max(wsb, 16), dtype=torch.uint8, device="cuda")
    if pad:   # row strides that are not a multiple of 8 elements: the tensor-core kernel's alignment rule fails
        k2 = np.ascontiguousarray(np.pad(k2, ((0, 0), (0, pad))))
        v2 = np.ascontiguousarray(np.pad(v2, ((0, 0), (0, pad))))
    kd, vd = f16(k2), f16(v2)
    sk.starkv_append(ctx, dpool, dev(table.astype(np.int32)), table.shape[1], dev(seq_ids), dev(positions), n,
                     kd, kw + pad, khs, d_in_k, vd, vw + pad, d_in_v, f16(ak), f16(av), ws, wsb)
    torch.cuda.synchronize()
    want = ("append_small_kernel" if n <= 16 else "append_project_kernel" if pad else
            "append_gemm_kernel" if (tc5 and n >= 64) else "append_project_mma_kernel")
    assert sk.starkv_last_append_kernel_name(ctx) == want   # the path under test really ran (no silent fallback)
    return d, lay, dpool.cpu().numpy(), ref, n


@pytest.mark.parametrize("n_new", [-80, 80, 37, 8, 1], ids=["n80-tcgen05", "n80-mma", "n37-mma", "n8-small", "n1-small"])
@pytest.mark.parametrize("name,mode", [("C1", "dense"), ("C3", "dense"), ("C3", "hidden"), ("C4", "dense")])
def test_append_bit_exact_on_dyadic_inputs(name, mode, n_new):
    """n_new 80 -> 134 tokens (two token tiles with a ragged tail) on the mma.sync projection and, opted in through
    starkv_set_option "append_tc5", on the tcgen05 projection; 37 -> 62 tokens; 8 -> 15 and 1 -> 2 tokens (split-K
    small-n kernel)."""
    tc5 = n_new < 0
    n_new = abs(n_new)
    cfg = synth.make_config(name, context=256, batch=3)
    d, lay, got, ref, n = _append_case(cfg, mode, n_new, dyadic=True, tc5=tc5)
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} bytes differ of {got.size}"


@pytest.mark.parametrize("name,mode", [("C1", "dense"), ("C3", "dense"), ("C4", "hidden"), ("C2", "dense")])
def test_append_prefill_chunk_in_position_order(name, mode):
    """Tokens in (sequence, position) order, the first sequence starting mid-octet (position 70): append_write_kernel maps
    whole slot octets of a page to CTAs and writes the channel-major value fields as whole words (no atomics); the other
    sequences start at other offsets and take the per-field path.  Pre-existing bytes of the pages must survive."""
    cfg = synth.make_config(name, context=256, batch=3)
    d, lay, got, ref, n = _append_case(cfg, mode, 80, dyadic=True, ordered=True)
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} bytes differ of {got.size}"


@pytest.mark.parametrize("n_new", [80, 8], ids=["prefill", "decode-time"])
def test_append_at_the_paper_sized_value_rank(n_new):
    """Joint value rank 1024 (Fig.11): the low-precision value block has more than 512 columns, so the
    prefill GEMM runs without its fused epilogue and append_write_kernel quantises; the decode-time path takes the
    one-launch kernel's projection.  Bit-exact on dyadic inputs like every other shape."""
    cfg = synth.custom_config("rv1024", 3, 32, 32, 128, 256, [32] * 32, 1024, bits=(8, 4))
    d, lay, got, ref, n = _append_case(cfg, "dense", n_new, dyadic=True, ordered=(n_new == 80))
    assert np.array_equal(got, ref), f"{int((got != ref).sum())} bytes differ of {got.size}"


def test_append_unaligned_rows_take_the_scalar_kernel():
    cfg = synth.make_config("C3", context=256, batch=3)
    d, lay, got, ref, n = _append_case(cfg, "dense", 37, dyadic=True, pad=2)
    assert np.array_equal(got, ref)


@pytest.mark.parametrize("n_new", [120, 40, 8])
def test_append_gaussian_inputs_close(n_new):
    """Gaussian activations: fp32 summation order differs from the oracle's exact sum, so the fp16
    latent may differ in the last bit on a few entries; scales within 1 ulp, codes within 1 step."""
    cfg = synth.make_config("C3", context=256, batch=3)
    d, lay, got, ref, n = _append_case(cfg, "dense", n_new, dyadic=False)
    frac = float((got != ref).mean())
    assert frac < 1e-3, frac   # SURVEY pin P15: code mismatches on <= 1e-3 of the entries
    # compare decoded values of the touched pages
    n_pages = got.shape[0]
    a = ocodec.unpack_pages(d, got, n_pages * lay.page_tokens)
    b = ocodec.unpack_pages(d, ref, n_pages * lay.page_tokens)
    dc = np.abs(a["codes"].astype(np.int32) - b["codes"].astype(np.int32))
    assert dc.max() <= 1 and (dc > 0).mean() < 2e-3
    ds = np.abs(a["scales"].astype(np.int32) - b["scales"].astype(np.int32))
    assert ds.max() <= 1
