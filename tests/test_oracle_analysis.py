"""Pins P7, P8, P10, P11, P12, P13 for oracle/analysis.py (CPU only)."""
import os

import numpy as np

from oracle import analysis

GOLD = os.path.join(os.path.dirname(__file__), "golden", "paper_accounting.txt")


def golden():
    out = {}
    for line in open(GOLD):
        line = line.split("#")[0].strip()
        if "=" in line:
            k, v = line.split("=")
            out[k.strip()] = float(v)
    return out


def test_P7_truncation_error_is_next_singular_value_and_channels_are_ordered():
    """Lemma 4.1 / Eq.6: ||W - A B||_2 = sigma_{r+1}; and the latent channels
    (columns of A = V_r Sigma_r) have norms sigma_1 >= sigma_2 >= ... (L206: ordered channels)."""
    rng = np.random.default_rng(0)
    W = rng.standard_normal((24, 40))
    for r in (1, 5, 16, 23):
        A, B, s = analysis.svd_factors(W, r)
        err = np.linalg.norm(W - (A @ B).T, 2)
        assert abs(err - s[r]) <= 1e-12 * s[0]
        assert np.allclose(np.linalg.norm(A, axis=0), s[:r], atol=1e-12)
        assert np.all(np.diff(np.linalg.norm(A, axis=0)) <= 1e-12)
        assert np.allclose(B @ B.T, np.eye(r), atol=1e-12)            # orthonormal reconstruction rows
    # hard threshold (Eq.1): rank = number of singular values >= alpha
    _, _, s = analysis.svd_factors(W, 4)
    assert analysis.hard_threshold_rank(s, s[6]) == 7
    assert analysis.hard_threshold_rank(s, s[6] * (1 + 1e-9)) == 6


def test_P8_joint_error_not_larger_than_headwise():
    """Lemma 4.2 / Eq.10 on random matrices, R = h r."""
    rng = np.random.default_rng(1)
    for h, dh, r in ((4, 8, 2), (8, 16, 4), (2, 32, 8)):
        W = rng.standard_normal((48, h * dh)) @ np.diag(np.exp(-np.arange(h * dh) / 10.0))
        ej = np.linalg.norm(W - analysis.joint_approx(W, h * r))
        eh = np.linalg.norm(W - analysis.headwise_approx(W, h, r))
        assert ej <= eh * (1 + 1e-12)
        assert np.linalg.matrix_rank(analysis.headwise_approx(W, h, r)) <= h * r


def test_P10_bit_and_compression_accounting_matches_paper_tables():
    g = golden()
    assert abs(analysis.average_bits(0.2, 4, 3) - g["avg_bits_20_80"]) < 1e-12
    assert abs(analysis.compression_factor(0.75, 3.2) - g["comp_75_3p2"]) < 1e-9
    assert abs(analysis.compression_factor(0.60, 3.2) - g["comp_60_3p2"]) < 1e-9
    assert abs(analysis.compression_factor(0.50, 4.0) - g["comp_palu50_4bit"]) < 1e-9
    assert round(analysis.compression_factor(0.0, 3.16), 1) == g["comp_kivi_3p16"]
    assert round(analysis.compression_factor(0.0, 2.33), 1) == g["comp_kvquant_2p33"]
    for hi in (10, 20, 30, 40):
        bits = analysis.average_bits(hi / 100.0, 4, 3)
        assert abs(bits - g[f"split_{hi}_{100 - hi}_bits"]) < 1e-12
        assert abs(analysis.compression_factor(0.75, bits) - g[f"split_{hi}_{100 - hi}_comp"]) < 0.006


def test_P11_dense_cache_footprint_example():
    """LLaMA-3.1-8B (32 layers, 8 KV heads x 128), 128K x batch 4, fp16: KV = 81% of 85 GB."""
    g = golden()
    kv = analysis.dense_kv_bytes(32, 8, 128, 131072, 4)
    assert kv == 32 * 2 * 8 * 128 * 2 * 131072 * 4 == 68719476736
    weights = g["total_footprint_gb"] * 1e9 - kv
    assert 15e9 < weights < 17e9                      # ~8 B params in fp16
    assert round(100 * kv / (g["total_footprint_gb"] * 1e9)) == g["kv_share_percent"]


def test_P12_flop_models():
    """Observation 1 (L145-147): JD/HD reconstruction = h.  Value reordering (L68, reading A13):
    saving approaches d_h for long sequences."""
    for h, dh in ((32, 128), (8, 64)):
        assert analysis.recon_flops_jd(1000, 0.25, h, dh) / analysis.recon_flops_hd(1000, 0.25, h, dh) == h
        rv = 256
        ratio = analysis.value_flops_before(10 ** 7, rv, h, dh) / analysis.value_flops_after(10 ** 7, rv, h, dh)
        assert abs(ratio - dh * (1 + 1 / rv)) / dh < 1e-2


def test_P13_fused_block_hadamard_leaves_reconstruction_unchanged():
    """L206-210: (V Sigma) H and H^T U^T with independent H_out / H_in; no quantisation -> identity."""
    rng = np.random.default_rng(2)
    W = (rng.standard_normal((32, 32)) * np.exp(-np.arange(32) / 4.0)) @ rng.standard_normal((32, 48))
    for r, r_hi in ((24, 8), (32, 8), (16, 16), (32, 24)):
        A, B, _ = analysis.svd_factors(W, r)
        Ah, Bh = analysis.fuse_hadamard(A, B, r_hi)
        assert np.allclose(Ah @ Bh, A @ B, atol=1e-12)
        H = analysis.block_hadamard(r_hi)
        assert np.allclose(H @ H.T, np.eye(r_hi), atol=1e-12)
        # the rotation spreads the leading channel's energy across its block (Fig.8)
        x = rng.standard_normal((200, 48))
        z, zh = x @ A, x @ Ah
        assert zh[:, :r_hi].std(axis=0).max() / zh[:, :r_hi].std(axis=0).min() < z[:, :r_hi].std(axis=0).max() / z[:, :r_hi].std(axis=0).min() + 1e-9
