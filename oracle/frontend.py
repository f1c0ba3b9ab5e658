"""CPU ORACLE for the front end of the GDN block: feature map, gates, output gate (App. G.2, G.3, G.5).

THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT (same rules as gdn_oracle.c: only tests/, __graft_entry__.smoke() and
the cpu_baseline / --impl reference legs of bench.py may import it; it shares nothing with the CUDA path).

Plain numpy, fp64, one formula per line, in the paper's order and notation (row-token convention: a token is a row).

  feature_map   Eq. 12 (L552) + the key rescale of L554:
                    x^ = rho_3D( ReLU( RMSNorm(x) ) ),   K and K^ additionally * 1/sqrt(D N)
                returns the un-rotated features (used by the normaliser, Eq. 20-22) and the rotated ones
                (used by the KV memory, Eq. 18-19, 22).
  gates         Eq. 13-15 (L562-L572): x_bar_f = mean_n x_{f,n};  Delta_f = softplus(W_alpha . x_bar_f + b_alpha);
                    alpha_f = exp(-e^{A_log} Delta_f);   beta_n = sigmoid(W_beta . x_n + b_beta)
  output_gate   Eq. 23 (L626), the element-wise part: O = G (.) Y  (W_o is a GEMM outside this path)

Readings of the paper (items 23-26):
  * RMSNorm is taken over the D channels of one head, with a per-head-channel weight w[H, D]
    (App. G writes every equation per head; RMSNorm(x)_i = x_i / sqrt(mean_j x_j^2 + eps_rms) * w_i, [40]);
    eps_rms is an argument (the paper does not state it).
  * rho_3D rotates ADJACENT channel pairs (2i, 2i+1) by the angle theta_i(position): the caller supplies
    cos / sin tables [T, D/2] (Alg. 1 "Require: ... RoPE tables", L325); how the 3-D position maps to angles is the
    table's business, not this function's.
  * N in 1/sqrt(D N) is the number of tokens per frame, D the (un-padded) head dimension (L554).
  * the output gate G_f = SiLU(W_g X_f + b_g) (Eq. 16) arrives evaluated; only the Hadamard product is here.

Pins: tests/test_oracle_frontend.py (hand-worked example in tests/golden/frontend_d4.txt, norm preservation and the
relative-position property of the rotation, zero-angle reduction, scale invariance of RMSNorm, closed forms of the
gates at zero weights, permutation invariance of alpha inside a frame, limits).  Nothing here is "parity unpinned".
"""
from __future__ import annotations

import numpy as np


def _f64(x):
    import torch
    if isinstance(x, torch.Tensor):
        return x.detach().to(torch.float64).cpu().numpy()
    return np.asarray(x, dtype=np.float64)


def rms_norm(x, w, eps_rms):
    """RMSNorm over the last axis: x_i / sqrt(mean_j x_j^2 + eps) * w_i.  x [..., H, D], w [H, D]."""
    x, w = _f64(x), _f64(w)
    ms = np.mean(x * x, axis=-1, keepdims=True)
    return x / np.sqrt(ms + eps_rms) * w


def rope_pairs(x, cos, sin):
    """Rotate adjacent pairs: (x_{2i}, x_{2i+1}) -> (x_{2i} c_i - x_{2i+1} s_i, x_{2i} s_i + x_{2i+1} c_i).
    x [B, T, H, D], cos / sin [T, D/2]."""
    x, cos, sin = _f64(x), _f64(cos), _f64(sin)
    c = cos[None, :, None, :]
    s = sin[None, :, None, :]
    xe, xo = x[..., 0::2], x[..., 1::2]
    out = np.empty_like(x)
    out[..., 0::2] = xe * c - xo * s
    out[..., 1::2] = xe * s + xo * c
    return out


def feature_map(q, k, w_q, w_k, cos, sin, *, group: int, eps_rms: float = 1e-6):
    """q, k [B, T, H, D] raw projections (Eq. 11) -> (q_rot, k_rot, q_raw, k_raw), all fp64 [B, T, H, D].
    group = N = tokens per frame (enters the key rescale 1/sqrt(D N), L554)."""
    q, k = _f64(q), _f64(k)
    D = q.shape[-1]
    q_raw = np.maximum(rms_norm(q, w_q, eps_rms), 0.0)                      # ReLU(RMSNorm(Q))
    k_raw = np.maximum(rms_norm(k, w_k, eps_rms), 0.0)
    q_rot = rope_pairs(q_raw, cos, sin)                                     # rho_3D(.)
    k_rot = rope_pairs(k_raw, cos, sin)
    ks = 1.0 / np.sqrt(float(D) * float(group))                             # both K and K^ (L554)
    return q_rot, k_rot * ks, q_raw, k_raw * ks


def softplus(x):
    x = _f64(x)
    return np.maximum(x, 0.0) + np.log1p(np.exp(-np.abs(x)))


def gates(x, w_alpha, b_alpha, a_log, w_beta, b_beta, *, group: int):
    """x [B, T, H, D] per-head latent features; w_alpha, w_beta [H, D]; b_alpha, a_log, b_beta [H].
    -> (alpha [B, H, T/group], log_alpha [B, H, T/group], beta [B, H, T]), fp64."""
    x = _f64(x)
    w_alpha, b_alpha, a_log, w_beta, b_beta = map(_f64, (w_alpha, b_alpha, a_log, w_beta, b_beta))
    B, T, H, D = x.shape
    F = T // group
    x_bar = x.reshape(B, F, group, H, D).mean(axis=2)                       # Eq. 13
    delta = softplus(np.einsum("bfhd,hd->bfh", x_bar, w_alpha) + b_alpha)   # Eq. 14
    log_alpha = -np.exp(a_log)[None, None, :] * delta
    alpha = np.exp(log_alpha)
    beta = 1.0 / (1.0 + np.exp(-(np.einsum("bthd,hd->bth", x, w_beta) + b_beta)))   # Eq. 15
    return alpha.transpose(0, 2, 1).copy(), log_alpha.transpose(0, 2, 1).copy(), beta.transpose(0, 2, 1).copy()


def output_gate(y, g):
    """Eq. 23, element-wise part: G (.) Y."""
    return _f64(g) * _f64(y)
