"""Factor construction and the paper's accounting formulas, fp64.  TEST INFRASTRUCTURE.

These are the off-hot-path definitions the hot path's inputs come from; the oracle states them so
its pins can check the hot-path oracle against what the paper fixes.
"""
from __future__ import annotations

import numpy as np


# --- PAPER.md §3.2: W ~= U_r (Sigma V)_r^T; cache K' = x (Sigma V)_r, K = K' U_r^T ------------

def svd_factors(W: np.ndarray, r: int):
    """W [d_out, d_in] -> (A [d_in, r] = V_r Sigma_r  (down-projection, singular values folded in),
    B [r, d_out] = U_r^T (reconstruction), sigma [min(d_out, d_in)])  so that x A B ~= x W^T."""
    u, s, vt = np.linalg.svd(W, full_matrices=False)
    return vt[:r].T * s[:r], u[:, :r].T.copy(), s


def hard_threshold_rank(sigma: np.ndarray, alpha: float) -> int:
    """PAPER.md Eq.1: sigma~_i = sigma_i 1{sigma_i >= alpha}; effective rank = #kept."""
    return int(np.sum(np.asarray(sigma) >= alpha))


# --- PAPER.md §4.3: joint vs head-wise decomposition -------------------------------------

def joint_approx(W: np.ndarray, R: int) -> np.ndarray:
    """Best rank-R approximation of W [m, d] (Eq.8)."""
    u, s, vt = np.linalg.svd(W, full_matrices=False)
    return (u[:, :R] * s[:R]) @ vt[:R]


def headwise_approx(W: np.ndarray, h: int, r: int) -> np.ndarray:
    """Best approximation with rank <= r per head, heads = column blocks of W [m, h*d_h] (Eq.9)."""
    dh = W.shape[1] // h
    return np.concatenate([joint_approx(W[:, i * dh:(i + 1) * dh], r) for i in range(h)], axis=1)


def recon_flops_jd(l, c, h, dh):
    """L145: l * r_j * d with r_j = c d, d = h d_h."""
    return l * (c * h * dh) * (h * dh)


def recon_flops_hd(l, c, h, dh):
    """L145: h * l * r_h * d_h with r_h = c d_h."""
    return h * l * (c * dh) * dh


def value_flops_before(l, rv, h, dh):
    """DESIGN.md reading A13 of L68 (printed formula garbled): reconstruct V^i = V' U_V^iT per head
    (h l r_v d_h) then p^i V^i (h l d_h)."""
    return h * l * rv * dh + h * l * dh


def value_flops_after(l, rv, h, dh):
    """Reordered (p^i V') U_V^iT: h l r_v + h r_v d_h."""
    return h * l * rv + h * rv * dh


# --- PAPER.md §4.4 / Table 4 / Table 11: bit accounting (scale bytes NOT counted, as in the paper) --

def average_bits(frac_hi: float, b_hi: float, b_lo: float) -> float:
    return frac_hi * b_hi + (1.0 - frac_hi) * b_lo


def compression_factor(lowrank_compression: float, avg_bits: float, base_bits: float = 16.0) -> float:
    """Overall KV reduction = (1 / (1 - low-rank compression)) * (base_bits / avg_bits)."""
    return (1.0 / (1.0 - lowrank_compression)) * (base_bits / avg_bits)


def dense_kv_bytes(n_layers, n_kv_heads, head_dim, context, batch, bytes_per=2) -> int:
    """Dense fp16 KV cache bytes (L15): layers x {K,V} x H_kv x d_h x bytes x tokens x batch."""
    return n_layers * 2 * n_kv_heads * head_dim * bytes_per * context * batch


# --- block-wise Hadamard fused into the factors --------------------------------

def hadamard(n: int) -> np.ndarray:
    """Orthonormal Sylvester Hadamard H/sqrt(n), n a power of two."""
    assert n & (n - 1) == 0 and n > 0
    H = np.ones((1, 1))
    while H.shape[0] < n:
        H = np.block([[H, H], [H, -H]])
    return H / np.sqrt(n)


def block_hadamard(n: int) -> np.ndarray:
    """Orthogonal n x n: block diagonal of orthonormal Hadamards over n split into descending
    powers of two (reading A12; the paper is silent on non-power-of-two blocks)."""
    out = np.zeros((n, n))
    o = 0
    while o < n:
        b = 1 << ((n - o).bit_length() - 1)
        out[o:o + b, o:o + b] = hadamard(b)
        o += b
    return out


def fuse_hadamard(A: np.ndarray, B: np.ndarray, r_hi: int):
    """L210: independent H_out on the leading r_hi channels and H_in on the rest, fused offline as
    (V Sigma) H  and  H^T U^T.  A [d_in, r], B [r, d_out]."""
    r = A.shape[1]
    H = np.zeros((r, r))
    H[:r_hi, :r_hi] = block_hadamard(r_hi)
    if r > r_hi:
        H[r_hi:, r_hi:] = block_hadamard(r - r_hi)
    return A @ H, H.T @ B
