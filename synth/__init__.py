"""Seeded synthetic inputs for the STAR-KV decode/append hot path.

This module is the ONLY code shared by the CPU oracle's tests and the CUDA path's
tests/bench.  It produces inputs (shapes, rank tables, fp16 factors, fp16 latents,
queries, block tables) and holds none of the method's arithmetic: no quantiser, no
page codec, no attention, no projection of activations.  Packing latents into cache
pages is done by whichever side is under test (oracle codec in the parity tests,
``starkv_pack`` in the bench).

Recipe and citations: DESIGN.md "Synthetic inputs"; configs follow BASELINE.json
``configs[0..4]`` (called C1..C5 here); value structure follows PAPER.md L206
(latent channels scaled by ordered singular values -> decaying channel magnitude)
and Fig.10/11 L408-412 (ragged per-head key ranks, one joint value rank).

Every array comes from ``numpy.random.Generator(PCG64(BASE_SEED + stream))`` with a
fixed stream id per array kind, so oracle and GPU see bit-identical inputs.
"""
from __future__ import annotations

import dataclasses
import math
from typing import List, Optional, Sequence

import numpy as np

BASE_SEED = 8382

# fixed stream ids (added to the seed) per array kind
_S_RANKS, _S_FACT_K, _S_FACT_V, _S_LAT_K, _S_LAT_V, _S_Q, _S_TABLE, _S_LENS = range(1, 9)
_S_APP_X, _S_APP_AK, _S_APP_AV, _S_OUTLIER = range(9, 13)


def _rng(seed: int, stream: int, sub: int = 0) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64([BASE_SEED + seed, stream, sub]))


@dataclasses.dataclass
class Config:
    """Static description of one workload (one layer)."""
    name: str
    batch: int
    n_q_heads: int
    n_kv_heads: int
    head_dim: int
    d_model: int
    context: int
    rank_k: List[int]            # per KV head r_h
    rank_k_hi: List[int]         # leading high-precision channels per KV head
    rank_v: int
    rank_v_hi: int
    bits_hi: int                 # 16 => fp16 latents (bits_lo must be 16 too)
    bits_lo: int
    page_tokens: int = 64
    outlier_frac: float = 0.0    # fraction of heavy-tailed tokens (Student-t df=3)
    layer: int = 0
    seed: int = 0

    @property
    def group(self) -> int:
        return self.n_q_heads // self.n_kv_heads

    @property
    def sum_rank_k(self) -> int:
        return int(sum(self.rank_k))

    @property
    def sm_scale(self) -> float:
        return 1.0 / math.sqrt(self.head_dim)     # 1/sqrt(d_h), full head dim

    @property
    def quantized(self) -> bool:
        return self.bits_hi != 16

    def k_offsets(self) -> List[int]:
        off, out = 0, []
        for r in self.rank_k:
            out.append(off)
            off += r
        return out


def rank_hi(r: int) -> int:
    """Channel count of the leading ("outlier") precision block: 20% of r (PAPER.md L210,
    L270) rounded to a multiple of 8, at least 8 (reading A8)."""
    return int(min(r, max(8, 8 * int(math.floor(0.2 * r / 8 + 0.5)))))


def rank_profile(n_layers: int, n_kv_heads: int, target: int, head_dim: int,
                 seed: int = 0, lo: int = 8, hi: int = 96) -> np.ndarray:
    """"Soft-threshold-like" ragged key-rank table [n_layers, n_kv_heads].

    Per (layer, head): decay length tau ~ LogNormal(ln(target/2), 0.5); spectrum
    sigma_c = exp(-c/tau); one hard threshold alpha per layer (Eq.1)
    found by bisection so the layer's mean rank hits ``target``; ranks rounded to a
    multiple of 8, clamped to [lo, hi], then fixed up by +-8 in seeded head order until
    the layer sum is exactly n_kv_heads*target.
    """
    out = np.zeros((n_layers, n_kv_heads), dtype=np.int64)
    for layer in range(n_layers):
        g = _rng(seed, _S_RANKS, layer)
        tau = np.exp(g.normal(math.log(target / 2.0), 0.5, size=n_kv_heads))
        # rank_h(x) = #{c : exp(-c/tau_h) >= alpha} with x = -ln(alpha)
        def ranks_at(x):
            return np.minimum(head_dim, np.floor(tau * x) + 1.0)
        a, b = 0.0, 64.0
        for _ in range(80):
            m = 0.5 * (a + b)
            if ranks_at(m).mean() < target:
                a = m
            else:
                b = m
        r = ranks_at(b)
        r = np.clip(8 * np.floor(r / 8 + 0.5), lo, hi).astype(np.int64)
        order = g.permutation(n_kv_heads)
        want = n_kv_heads * target
        i = 0
        while r.sum() != want:
            h = order[i % n_kv_heads]
            if r.sum() < want and r[h] + 8 <= hi:
                r[h] += 8
            elif r.sum() > want and r[h] - 8 >= lo:
                r[h] -= 8
            i += 1
            if i > 100000:
                raise RuntimeError("rank fix-up did not converge")
        out[layer] = r
    return out


def make_config(name: str, *, context: Optional[int] = None, batch: Optional[int] = None,
                layer: int = 0, page_tokens: int = 64, seed: int = 0,
                bits: Optional[Sequence[int]] = None) -> Config:
    """BASELINE.json configs C1..C5 (one layer of C5 per call). ``context``/``batch``
    override the size for reduced parity copies; the rank tables do not change."""
    name = name.upper()
    if name == "C1":
        g = _rng(seed, _S_RANKS, 1000)
        rk = [int(x) for x in g.choice([16, 32, 48, 64], size=2)]
        cfg = Config("C1", 1, 4, 2, 64, 256, 512, rk, [rank_hi(r) for r in rk], 64, rank_hi(64),
                     16, 16)
    elif name == "C2":
        rk = [int(x) for x in rank_profile(32, 8, 32, 128, seed)[layer]]
        cfg = Config("C2", 4, 32, 8, 128, 4096, 32768, rk, [rank_hi(r) for r in rk], 256,
                     rank_hi(256), 16, 16)
    elif name in ("C3", "C5"):
        rk = [int(x) for x in rank_profile(32, 8, 32, 128, seed)[layer]]
        cfg = Config(name, 1 if name == "C3" else 4, 32, 8, 128, 4096,
                     131072 if name == "C3" else 65536, rk, [rank_hi(r) for r in rk], 256,
                     rank_hi(256), 8, 4, outlier_frac=0.10)
    elif name == "C4":
        rk = [int(x) for x in rank_profile(32, 32, 48, 128, seed + 1)[layer]]
        cfg = Config("C4", 8, 32, 32, 128, 4096, 16384, rk, [rank_hi(r) for r in rk], 384,
                     rank_hi(384), 8, 4, outlier_frac=0.10)
    else:
        raise ValueError(f"unknown config {name}")
    if context is not None:
        cfg.context = int(context)
    if batch is not None:
        cfg.batch = int(batch)
    if bits is not None:
        cfg.bits_hi, cfg.bits_lo = int(bits[0]), int(bits[1])
    cfg.layer, cfg.page_tokens, cfg.seed = layer, page_tokens, seed
    return cfg


def custom_config(name, batch, n_q_heads, n_kv_heads, head_dim, context, rank_k, rank_v,
                  bits=(16, 16), page_tokens=64, outlier_frac=0.0, rank_k_hi=None,
                  rank_v_hi=None, d_model=0, seed=0) -> Config:
    rk = [int(r) for r in rank_k]
    return Config(name, batch, n_q_heads, n_kv_heads, head_dim, d_model or n_q_heads * head_dim,
                  context, rk,
                  [int(x) for x in (rank_k_hi if rank_k_hi is not None else [rank_hi(r) for r in rk])],
                  int(rank_v), int(rank_v_hi if rank_v_hi is not None else rank_hi(rank_v)),
                  int(bits[0]), int(bits[1]), page_tokens, outlier_frac, 0, seed)


# ----------------------------------------------------------------------------------------
# factors
# ----------------------------------------------------------------------------------------

def _orthonormal_rows(g: np.random.Generator, r: int, d: int) -> np.ndarray:
    """r orthonormal rows in R^d (Haar): left singular vectors of a seeded Gaussian d x d
    for d <= 1024 (BASELINE.json recipe), reduced QR of a Gaussian d x r above that (same
    distribution, far cheaper)."""
    if d <= 1024:
        m = g.standard_normal((d, d))
        u, _, _ = np.linalg.svd(m)
        return np.ascontiguousarray(u[:, :r].T)
    m = g.standard_normal((d, r))
    qm, _ = np.linalg.qr(m)
    return np.ascontiguousarray(qm.T)


def make_factors(cfg: Config):
    """Reconstruction factors, fp16: B_k [sum r_h, d_h] (head h = rows koff[h]..+r_h, orthonormal
    rows) and B_v [r_v, H_kv*d_h] (orthonormal rows)."""
    d_h, dv = cfg.head_dim, cfg.n_kv_heads * cfg.head_dim
    bk = np.zeros((cfg.sum_rank_k, d_h), dtype=np.float64)
    for h, (off, r) in enumerate(zip(cfg.k_offsets(), cfg.rank_k)):
        bk[off:off + r] = _orthonormal_rows(_rng(cfg.seed, _S_FACT_K, cfg.layer * 4096 + h), r, d_h)
    bv = _orthonormal_rows(_rng(cfg.seed, _S_FACT_V, cfg.layer), cfg.rank_v, dv)
    return bk.astype(np.float16), bv.astype(np.float16)


def make_svd_projection_factors(cfg: Config):
    """C1 recipe (BASELINE.json configs[0]): per KV head a seeded Gaussian d_h x d_h projection
    M_h = U S V^T and one joint (H_kv d_h)^2 projection M_v; returns fp64
    (M_k list, M_v, A_k [d_h, sum r_h] = (V S)_r per head, B_k = U_r^T, A_v, B_v) so that
    X A B ~= X M^T."""
    d_h, dv = cfg.head_dim, cfg.n_kv_heads * cfg.head_dim
    mk, ak, bk = [], np.zeros((d_h, cfg.sum_rank_k)), np.zeros((cfg.sum_rank_k, d_h))
    for h, (off, r) in enumerate(zip(cfg.k_offsets(), cfg.rank_k)):
        m = _rng(cfg.seed, _S_FACT_K, 100000 + cfg.layer * 4096 + h).standard_normal((d_h, d_h)) / math.sqrt(d_h)
        u, s, vt = np.linalg.svd(m)
        mk.append(m)
        ak[:, off:off + r] = vt[:r].T * s[:r]
        bk[off:off + r] = u[:, :r].T
    m = _rng(cfg.seed, _S_FACT_V, 100000 + cfg.layer).standard_normal((dv, dv)) / math.sqrt(dv)
    u, s, vt = np.linalg.svd(m)
    r = cfg.rank_v
    return mk, m, ak, bk, vt[:r].T * s[:r], u[:, :r].T


def make_append_factors(cfg: Config, d_in_k: int, d_in_v: int):
    """Down-projections for the append kernel, fp16: A_k [d_in_k, sum r_h], A_v [d_in_v, r_v];
    seeded Gaussian with column c of each head scaled by sigma_c/sqrt(d_in),
    sigma_c = exp(-c/(r/2)) (singular values folded in)."""
    ak = np.zeros((d_in_k, cfg.sum_rank_k), dtype=np.float32)
    for h, (off, r) in enumerate(zip(cfg.k_offsets(), cfg.rank_k)):
        g = _rng(cfg.seed, _S_APP_AK, cfg.layer * 4096 + h)
        sig = np.exp(-np.arange(r) / (r / 2.0))
        ak[:, off:off + r] = g.standard_normal((d_in_k, r), dtype=np.float32) * (sig / math.sqrt(d_in_k)).astype(np.float32)
    g = _rng(cfg.seed, _S_APP_AV, cfg.layer)
    sig = np.exp(-np.arange(cfg.rank_v) / (cfg.rank_v / 2.0))
    av = g.standard_normal((d_in_v, cfg.rank_v), dtype=np.float32) * (sig / math.sqrt(d_in_v)).astype(np.float32)
    return ak.astype(np.float16), av.astype(np.float16)


def make_append_inputs(cfg: Config, n_new: int, mode: str = "dense"):
    """New-token activations for append, fp16. mode "dense": K [n, H_kv, d_h], V [n, H_kv*d_h]
    (north_star's "new K/V"); mode "hidden": x [n, d_model] used for both."""
    g = _rng(cfg.seed, _S_APP_X, cfg.layer)
    if mode == "dense":
        k = g.standard_normal((n_new, cfg.n_kv_heads, cfg.head_dim), dtype=np.float32)
        v = g.standard_normal((n_new, cfg.n_kv_heads * cfg.head_dim), dtype=np.float32)
        return k.astype(np.float16), v.astype(np.float16)
    x = g.standard_normal((n_new, cfg.d_model), dtype=np.float32)
    return x.astype(np.float16), None


def dyadic_append_case(cfg: Config, n_new: int, d_in_k: int, d_in_v: int):
    """Inputs on a dyadic grid (X in {-8..8}/8, A in integers/16, |A| <= 2) so every partial sum
    over d_in <= 4096 is exact in fp32 in any order: append parity is then bit-exact
    (DESIGN.md pin P15)."""
    g = _rng(cfg.seed, _S_APP_X, 7777 + cfg.layer)
    k = g.integers(-8, 9, size=(n_new, cfg.n_kv_heads, d_in_k)).astype(np.float32) / 8.0
    v = g.integers(-8, 9, size=(n_new, d_in_v)).astype(np.float32) / 8.0
    ak = g.integers(-32, 33, size=(d_in_k, cfg.sum_rank_k)).astype(np.float32) / 16.0
    av = g.integers(-32, 33, size=(d_in_v, cfg.rank_v)).astype(np.float32) / 16.0
    # sparsify so |sum| stays well inside fp16 range and has few significant bits
    ak *= (g.random(ak.shape) < 0.25)
    av *= (g.random(av.shape) < 0.05)
    return k.astype(np.float16), v.astype(np.float16), ak.astype(np.float16), av.astype(np.float16)


# ----------------------------------------------------------------------------------------
# latents, queries, paging
# ----------------------------------------------------------------------------------------

#: closed-form score spread per regime: scores ~ N(0, tau^2) for Gaussian tokens gives
#: n_eff = 1/sum p^2 ~= l * exp(-tau^2) (log-normal weights).
REGIME_TAU = {"diffuse": 0.8, "peaky": 3.0}
#: Student-t draws of KEY latents are clipped to +-KEY_OUTLIER_CLIP so a single outlier token
#: cannot capture the whole softmax in the "diffuse" regime (value latents are not clipped).
KEY_OUTLIER_CLIP = 6.0


def _latent_block(g: np.random.Generator, n: int, r: int, kappa: float,
                  outlier: Optional[np.ndarray], clip: Optional[float] = None) -> np.ndarray:
    sig = (kappa * np.exp(-np.arange(r) / (r / 2.0))).astype(np.float32)
    z = g.standard_normal((n, r), dtype=np.float32)
    if outlier is not None and outlier.any():
        idx = np.nonzero(outlier)[0]
        t = g.standard_t(3.0, size=(idx.size, r)).astype(np.float32)
        z[idx] = t if clip is None else np.clip(t, -clip, clip)
    return (z * sig).astype(np.float16)


def make_latents(cfg: Config, n_tokens: int, seq: int = 0, regime: str = "diffuse",
                 clip: Optional[float] = KEY_OUTLIER_CLIP):
    """Latent cache contents for one sequence, fp16: L_k [n, sum r_h], L_v [n, r_v].

    z[t,c] = kappa * sigma_c * g,  sigma_c = exp(-c/(r/2)),  g ~ N(0,1); a seeded
    ``outlier_frac`` of tokens draws g from Student-t(df=3) instead.  Key latents use
    kappa_h = tau / (sm_scale * sqrt(sum_c sigma_c^2)) so that, for unit-variance projected
    queries, scores have standard deviation ~tau (REGIME_TAU); value latents use kappa = 1.
    ``clip`` bounds the Student-t draws of the KEY latents (default +-KEY_OUTLIER_CLIP; ``None`` = unclipped, as
    BASELINE.json words the workload -- parity tests run both).
    """
    tau = REGIME_TAU[regime]
    outlier = None
    if cfg.outlier_frac > 0:
        outlier = _rng(cfg.seed, _S_OUTLIER, cfg.layer * 65536 + seq).random(n_tokens) < cfg.outlier_frac
    lk = np.zeros((n_tokens, cfg.sum_rank_k), dtype=np.float16)
    for h, (off, r) in enumerate(zip(cfg.k_offsets(), cfg.rank_k)):
        sig2 = float(np.sum(np.exp(-np.arange(r) / (r / 2.0)) ** 2))
        kappa = tau / (cfg.sm_scale * math.sqrt(sig2))
        g = _rng(cfg.seed, _S_LAT_K, (cfg.layer * 65536 + seq) * 256 + h)
        lk[:, off:off + r] = _latent_block(g, n_tokens, r, kappa, outlier, clip)
    g = _rng(cfg.seed, _S_LAT_V, cfg.layer * 65536 + seq)
    lv = _latent_block(g, n_tokens, cfg.rank_v, 1.0, outlier)
    return lk, lv


def make_q(cfg: Config, batch: Optional[int] = None) -> np.ndarray:
    """Query, fp16 [B, H_q, d_h], N(0,1)."""
    b = cfg.batch if batch is None else batch
    return _rng(cfg.seed, _S_Q, cfg.layer).standard_normal((b, cfg.n_q_heads, cfg.head_dim)).astype(np.float16)


def make_seq_lens(cfg: Config, ragged: bool = False) -> np.ndarray:
    if not ragged:
        return np.full(cfg.batch, cfg.context, dtype=np.int32)
    g = _rng(cfg.seed, _S_LENS, cfg.layer)
    return g.integers(max(1, cfg.context // 2), cfg.context + 1, size=cfg.batch).astype(np.int32)


def make_block_table(cfg: Config, seq_lens: np.ndarray, shuffle: bool = True, extra_pages: int = 0):
    """Paged-cache block table int32 [B, max_pages] (unused entries -1) over a pool of
    ``n_pool`` physical pages; a seeded random permutation makes pages non-contiguous."""
    p = cfg.page_tokens
    need = [(int(l) + p - 1) // p for l in seq_lens]
    max_pages = max(1, max(need) if need else 1)
    n_pool = int(sum(need)) + extra_pages
    perm = np.arange(n_pool, dtype=np.int32)
    if shuffle:
        perm = _rng(cfg.seed, _S_TABLE, cfg.layer).permutation(n_pool).astype(np.int32)
    table = np.full((len(seq_lens), max_pages), -1, dtype=np.int32)
    k = 0
    for b, n in enumerate(need):
        table[b, :n] = perm[k:k + n]
        k += n
    return table, max(n_pool, 1)


def algorithmic_bytes_per_token(cfg: Config) -> dict:
    """Bytes of latent cache one cached token occupies (what decode must read), split as in
    SURVEY.md 8(d): key codes, value codes, scales."""
    if not cfg.quantized:
        kb, vb, sb = 2 * cfg.sum_rank_k, 2 * cfg.rank_v, 0
    else:
        kb = sum(rh * cfg.bits_hi // 8 + (r - rh) * cfg.bits_lo // 8
                 for r, rh in zip(cfg.rank_k, cfg.rank_k_hi))
        vb = cfg.rank_v_hi * cfg.bits_hi // 8 + (cfg.rank_v - cfg.rank_v_hi) * cfg.bits_lo // 8
        sb = 2 * (2 * cfg.n_kv_heads + 2)
    return {"key": kb, "value": vb, "scale": sb, "total": kb + vb + sb}


def factor_bytes(cfg: Config) -> int:
    """Per-step bytes that are not per-token: B_k, B_v, q, out (fp16)."""
    return 2 * (cfg.sum_rank_k * cfg.head_dim + cfg.rank_v * cfg.n_kv_heads * cfg.head_dim
                + 2 * cfg.batch * cfg.n_q_heads * cfg.head_dim)
