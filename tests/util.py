"""Test helpers: build a paged cache for a synth.Config with the ORACLE's codec."""
import numpy as np

import synth
from oracle import codec as ocodec
from oracle.layout import CacheDesc, page_layout


def build_cache(cfg, seq_lens=None, regime="diffuse", shuffle=True, latents=None, clip=synth.KEY_OUTLIER_CLIP):
    """Returns dict(desc, layout, pool uint8 [n_pool, page_bytes], table, seq_lens, lat=[(lk, lv)...])."""
    d = CacheDesc.from_config(cfg)
    lay = page_layout(d)
    seq_lens = synth.make_seq_lens(cfg) if seq_lens is None else np.asarray(seq_lens, np.int32)
    table, n_pool = synth.make_block_table(cfg, seq_lens, shuffle=shuffle)
    pool = np.zeros((n_pool, lay.page_bytes), np.uint8)
    lat = []
    for b, l in enumerate(seq_lens):
        l = int(l)
        lk, lv = latents[b] if latents is not None else synth.make_latents(cfg, l, seq=b, regime=regime, clip=clip)
        lat.append((lk, lv))
        if l == 0:
            continue
        pages = ocodec.pack_pages(d, lk[:l], lv[:l])
        pool[table[b, :pages.shape[0]]] = pages
    return dict(desc=d, layout=lay, pool=pool, table=table, seq_lens=seq_lens, lat=lat)


def row_rel_err(out, ref):
    """max over (b, head) rows of ||out-ref||_inf / ||ref||_inf  (DESIGN.md error metric)."""
    out = np.asarray(out, np.float64)
    ref = np.asarray(ref, np.float64)
    num = np.abs(out - ref).max(axis=-1)
    den = np.abs(ref).max(axis=-1)
    den = np.where(den == 0, 1.0, den)
    return float((num / den).max())
