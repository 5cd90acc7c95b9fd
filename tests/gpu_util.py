"""Helpers for the -m gpu parity tests: move an oracle-built cache to the device and call the C ABI."""
import numpy as np
import torch

import paper_2606_08382_b200 as sk


def dev(a, dtype=None):
    t = torch.from_numpy(np.ascontiguousarray(a))
    if dtype is not None:
        t = t.view(dtype)
    return t.cuda()


def f16(a):
    return dev(np.ascontiguousarray(a).view(np.uint16), torch.int16).view(torch.float16)


def run_decode(cfg, cache, q16, bk16, bv16, generic=False, splits=0, ctx=None):
    """cache: tests.util.build_cache dict.  Returns out float64 [B, H_q, d_h] (from the fp16 result)."""
    ctx = ctx or sk.create_from_config(cfg)
    assert sk.starkv_page_bytes(ctx) == cache["layout"].page_bytes
    pool = dev(cache["pool"])
    table = dev(cache["table"].astype(np.int32))
    lens = dev(np.asarray(cache["seq_lens"], np.int32))
    B, max_pages = table.shape
    q, bk, bv = f16(q16), f16(bk16), f16(bv16)
    sk.starkv_set_splits(ctx, splits)
    wsb = sk.starkv_workspace_bytes(ctx, B, max_pages)
    ws = torch.empty(wsb, dtype=torch.uint8, device="cuda")
    out = torch.full((B, cfg.n_q_heads, cfg.head_dim), float("nan"), dtype=torch.float16, device="cuda")
    fn = sk.starkv_decode_attn_generic if generic else sk.starkv_decode_attn
    fn(ctx, q, pool, table, max_pages, lens, B, bk, bv, ws, wsb, out)
    torch.cuda.synchronize()
    return out.double().cpu().numpy()
