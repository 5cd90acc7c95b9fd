"""GPU test of starkv_decode_attn_static, the entry point that allocates nothing: its decode scratch is a file-scope
device array of the library (csrc/decode_static.cu) instead of a caller workspace.  It must give what the existing
path (starkv_decode_attn with a caller workspace) gives, on calls made IN A ROW -- every call shares the array and
finds the previous call's bytes in it -- and must refuse a call whose scratch need exceeds the array.

Named test_zz_* so that pytest collects it last (the suite runs with `pytest -x`: a failure here hides nothing).
It passes alone in a fresh process (the first call resolves the array's device address) and after the other tests."""
import numpy as np
import pytest
import torch

import synth
from tests.gpu_util import dev, f16, run_decode
from tests.util import build_cache, row_rel_err

pytestmark = pytest.mark.gpu
sk = pytest.importorskip("paper_2606_08382_b200")

TOL = 2e-3   # the parity bar of tests/test_gpu_decode.py (BASELINE.json north_star), row-relative error


def _case(name, ctxlen, batch, lens):
    cfg = synth.make_config(name, context=ctxlen, batch=batch)
    cache = build_cache(cfg, seq_lens=lens)
    bk, bv = synth.make_factors(cfg)
    q = synth.make_q(cfg, batch=batch)
    ctx = sk.create_from_config(cfg)
    ref = run_decode(cfg, cache, q, bk, bv, ctx=ctx)            # existing path: caller-owned workspace
    table = dev(cache["table"].astype(np.int32))
    args = dict(ctx=ctx, q=f16(q), pool=dev(cache["pool"]), table=table, max_pages=table.shape[1],
                lens=dev(np.asarray(cache["seq_lens"], np.int32)), batch=batch, bk=f16(bk), bv=f16(bv),
                out=torch.full((batch, cfg.n_q_heads, cfg.head_dim), float("nan"), dtype=torch.float16, device="cuda"))
    assert sk.starkv_workspace_bytes(ctx, batch, table.shape[1]) <= sk.STATIC_SCRATCH_BYTES
    return args, ref


def _call_static(a):
    sk.starkv_decode_attn_static(a["ctx"], a["q"], a["pool"], a["table"], a["max_pages"], a["lens"], a["batch"], a["bk"],
                                 a["bv"], a["out"])


def test_static_scratch_decode_equals_the_workspace_path_on_calls_in_a_row():
    """Three shapes on three kernels (C3: TMEM-operand kernel, int8/int4; C2: mma.sync kernel, fp16; C1: 4 heads), called
    back to back on one stream with no synchronisation in between, then the first shape again: every call starts from
    the scratch contents another shape left behind."""
    cases = [_case("C3", 3000, 2, [3000, 1777]), _case("C2", 1500, 3, [1500, 64, 999]), _case("C1", 512, 1, [512])]
    cases.append(_case("C3", 3000, 2, [2999, 1]))
    torch.cuda.synchronize()
    for a, _ in cases:          # in a row: same stream, nothing between the calls
        _call_static(a)
    torch.cuda.synchronize()
    for i, (a, ref) in enumerate(cases):
        out = a["out"].double().cpu().numpy()
        assert np.isfinite(out).all(), i
        err = row_rel_err(out, ref)
        assert err <= TOL, f"call {i}: row rel err {err:.3e} against the workspace path"
        assert sk.starkv_last_launches(a["ctx"]) == 3
    # and the same call twice in a row gives the same bits (the array's previous contents do not leak into a result)
    a, _ = cases[0]
    first = a["out"].clone()
    a["out"].fill_(float("nan"))
    _call_static(a)
    torch.cuda.synchronize()
    assert torch.equal(a["out"].view(torch.int16), first.view(torch.int16))


def test_static_scratch_refuses_a_call_beyond_its_size():
    """148 splits x 32 heads x (512 + 4) fp32 = 9.8 MB of partials do not fit the 8 MiB array: STARKV_ERR_WORKSPACE with
    both sizes in the text, before anything is launched (out untouched).  With fewer splits the same call fits."""
    cfg = synth.custom_config("wide", 1, 32, 8, 128, 16384, [32] * 8, 512, bits=(8, 4))
    ctx = sk.create_from_config(cfg)
    max_pages = 256
    need = sk.starkv_workspace_bytes(ctx, 1, max_pages)
    assert need > sk.STATIC_SCRATCH_BYTES
    pool = torch.zeros((1, sk.starkv_page_bytes(ctx)), dtype=torch.uint8, device="cuda")
    table = torch.zeros((1, max_pages), dtype=torch.int32, device="cuda")
    lens = torch.zeros((1,), dtype=torch.int32, device="cuda")
    bk, bv = synth.make_factors(cfg)
    q = f16(synth.make_q(cfg, batch=1))
    out = torch.full((1, 32, 128), float("nan"), dtype=torch.float16, device="cuda")
    with pytest.raises(sk.StarkvError) as e:
        sk.starkv_decode_attn_static(ctx, q, pool, table, max_pages, lens, 1, f16(bk), f16(bv), out)
    assert e.value.code == sk.STARKV_ERR_WORKSPACE
    assert str(need) in str(e.value) and str(sk.STATIC_SCRATCH_BYTES) in str(e.value)
    torch.cuda.synchronize()
    assert torch.isnan(out).all()
    sk.starkv_set_splits(ctx, 64)
    assert sk.starkv_workspace_bytes(ctx, 1, max_pages) <= sk.STATIC_SCRATCH_BYTES
    sk.starkv_decode_attn_static(ctx, q, pool, table, max_pages, lens, 1, f16(bk), f16(bv), out)   # seq_len 0: a zero row
    torch.cuda.synchronize()
    assert (out == 0).all()
