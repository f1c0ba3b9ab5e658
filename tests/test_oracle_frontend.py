"""Pins for oracle/frontend.py (feature map, gates, output gate: PAPER.md Eq. 12-15, 23, L554).  CPU only."""
from pathlib import Path

import numpy as np
import pytest

from oracle import frontend as fe

GOLD = Path(__file__).parent / "golden" / "frontend_d4.txt"


def _gold():
    d = {}
    for line in GOLD.read_text().splitlines():
        if not line or line.startswith("#"):
            continue
        k, *v = line.split()
        d[k] = np.array([float(x) for x in v])
    return d


def test_handworked_feature_map():
    g = _gold()
    x = g["x"].reshape(1, 2, 1, 4)
    w = g["w"].reshape(1, 4)
    cos, sin = g["cos"].reshape(2, 2), g["sin"].reshape(2, 2)
    q_rot, k_rot, q_raw, k_raw = fe.feature_map(x, x, w, w, cos, sin, group=2, eps_rms=0.0)
    for name, got in (("q_rot", q_rot), ("k_rot", k_rot), ("q_raw", q_raw), ("k_raw", k_raw)):
        np.testing.assert_allclose(got.reshape(-1), g[name], rtol=0, atol=1e-15, err_msg=name)


def test_handworked_gates():
    g = _gold()
    x = g["gx"].reshape(1, 2, 1, 2)
    alpha, log_alpha, beta = fe.gates(x, np.array([[0.5, -0.5]]), np.zeros(1), np.zeros(1), np.array([[1.0, -1.0]]), np.zeros(1), group=2)
    np.testing.assert_allclose(alpha.reshape(-1), g["alpha"], atol=1e-15)
    np.testing.assert_allclose(np.exp(log_alpha), alpha, atol=1e-15)
    np.testing.assert_allclose(beta.reshape(-1), g["beta"], atol=1e-15)


def _rand(seed, B=2, T=12, H=3, D=8):
    r = np.random.default_rng(seed)
    ang = r.uniform(-3, 3, size=(T, D // 2))
    return r.standard_normal((B, T, H, D)), r.standard_normal((B, T, H, D)), r.uniform(0.5, 1.5, (H, D)), r.uniform(0.5, 1.5, (H, D)), ang


def test_rotation_preserves_pair_norms_and_zero_angle_is_identity():
    q, k, wq, wk, ang = _rand(0)
    q_rot, k_rot, q_raw, k_raw = fe.feature_map(q, k, wq, wk, np.cos(ang), np.sin(ang), group=4)
    for rot, raw in ((q_rot, q_raw), (k_rot, k_raw)):
        n_rot = rot[..., 0::2] ** 2 + rot[..., 1::2] ** 2
        n_raw = raw[..., 0::2] ** 2 + raw[..., 1::2] ** 2
        np.testing.assert_allclose(n_rot, n_raw, atol=1e-13)
    z = np.zeros_like(ang)
    q_rot0, k_rot0, q_raw0, k_raw0 = fe.feature_map(q, k, wq, wk, np.cos(z), np.sin(z), group=4)
    np.testing.assert_array_equal(q_rot0, q_raw0)
    np.testing.assert_array_equal(k_rot0, k_raw0)
    assert np.abs(q_rot - q_raw).max() > 0.1                 # negative control: the rotation does something


def test_relative_position_property():
    """With angles theta_i(t) = t * w_i the rotated dot product depends on positions only through t_q - t_k:
    <rho_t(a), rho_s(b)> = <rho_{t-s}(a), b>  (the defining property of RoPE [22])."""
    r = np.random.default_rng(1)
    D = 8
    a, b = r.standard_normal((1, 1, 1, D)), r.standard_normal((1, 1, 1, D))
    freq = r.uniform(0.1, 1.0, D // 2)
    def rot(x, t):
        ang = (t * freq)[None, :]
        return fe.rope_pairs(x, np.cos(ang), np.sin(ang))
    for t, s in ((5, 2), (7, 7), (1, 9)):
        lhs = np.sum(rot(a, t) * rot(b, s))
        rhs = np.sum(rot(a, t - s) * b)
        assert abs(lhs - rhs) < 1e-12


def test_rmsnorm_scale_invariance_relu_and_key_scale():
    q, k, wq, wk, ang = _rand(2)
    c, s = np.cos(ang), np.sin(ang)
    base = fe.feature_map(q, k, wq, wk, c, s, group=4, eps_rms=0.0)
    scaled = fe.feature_map(3.7 * q, 0.2 * k, wq, wk, c, s, group=4, eps_rms=0.0)
    for x, y in zip(base, scaled):
        np.testing.assert_allclose(x, y, atol=1e-13)          # RMSNorm removes a positive scale of the input
    assert base[2].min() >= 0 and base[3].min() >= 0            # un-rotated features are non-negative (ReLU)
    # unit weights: ReLU(RMSNorm(x)) has mean square <= 1 per token; the key carries exactly 1/sqrt(D N)
    ones = np.ones_like(wq)
    q_rot, k_rot, q_raw, k_raw = fe.feature_map(q, q, ones, ones, c, s, group=4, eps_rms=0.0)
    np.testing.assert_allclose(k_raw, q_raw / np.sqrt(8 * 4), atol=1e-15)
    np.testing.assert_allclose(k_rot, q_rot / np.sqrt(8 * 4), atol=1e-15)
    assert (np.mean(q_raw ** 2, axis=-1) <= 1 + 1e-12).all()
    # the other frame length changes only the key scale
    k_rot8 = fe.feature_map(q, q, ones, ones, c, s, group=6, eps_rms=0.0)[1]
    np.testing.assert_allclose(k_rot8 * np.sqrt(6), k_rot * np.sqrt(4), atol=1e-14)


def test_gate_closed_forms_and_invariants():
    r = np.random.default_rng(3)
    B, T, H, D, N = 2, 12, 3, 8, 4
    x = r.standard_normal((B, T, H, D))
    wa, wb = r.standard_normal((H, D)), r.standard_normal((H, D))
    ba, bb, al = r.standard_normal(H), r.standard_normal(H), r.standard_normal(H)
    alpha, log_alpha, beta = fe.gates(x, wa, ba, al, wb, bb, group=N)
    assert alpha.shape == (B, H, T // N) and beta.shape == (B, H, T)
    assert (alpha > 0).all() and (alpha <= 1).all() and (beta > 0).all() and (beta < 1).all()
    # zero weights: alpha = exp(-e^{A_log} softplus(b_alpha)), beta = sigmoid(b_beta), whatever x is
    a0, _, b0 = fe.gates(x, 0 * wa, ba, al, 0 * wb, bb, group=N)
    np.testing.assert_allclose(a0, np.broadcast_to(np.exp(-np.exp(al) * np.log1p(np.exp(ba)))[None, :, None], a0.shape), atol=1e-14)
    np.testing.assert_allclose(b0, np.broadcast_to((1 / (1 + np.exp(-bb)))[None, :, None], b0.shape), atol=1e-15)
    # alpha is a function of the frame MEAN: permuting tokens inside a frame leaves it unchanged and permutes beta
    perm = np.concatenate([f * N + r.permutation(N) for f in range(T // N)])
    a1, _, b1 = fe.gates(x[:, perm], wa, ba, al, wb, bb, group=N)
    np.testing.assert_allclose(a1, alpha, atol=1e-13)
    np.testing.assert_allclose(b1, beta[:, :, perm], atol=1e-15)
    # written out with loops for one (b, h, f) / token
    b_, h_, f_ = 1, 2, 1
    xb = sum(x[b_, f_ * N + n, h_] for n in range(N)) / N
    pre = sum(wa[h_, d] * xb[d] for d in range(D)) + ba[h_]
    delta = np.log(1 + np.exp(pre))
    assert abs(alpha[b_, h_, f_] - np.exp(-np.exp(al[h_]) * delta)) < 1e-14
    t_ = 7
    pre_b = sum(wb[h_, d] * x[b_, t_, h_, d] for d in range(D)) + bb[h_]
    assert abs(beta[b_, h_, t_] - 1 / (1 + np.exp(-pre_b))) < 1e-15
    # limits: a very negative pre-activation gives alpha -> 1 (no decay), a very positive one alpha -> 0
    a_hi, _, _ = fe.gates(x, 0 * wa, np.full(H, -50.0), al, wb, bb, group=N)
    a_lo, _, _ = fe.gates(x, 0 * wa, np.full(H, 60.0), np.full(H, 2.0), wb, bb, group=N)
    assert np.all(a_hi > 1 - 1e-12) and np.all(a_lo < 1e-100)


def test_softplus_is_stable_and_output_gate_is_hadamard():
    assert abs(fe.softplus(np.array(0.0)) - np.log(2)) < 1e-16
    assert fe.softplus(np.array(800.0)) == 800.0 and fe.softplus(np.array(-800.0)) == 0.0
    y, g = np.arange(6.0).reshape(2, 3), np.array([[1.0, 0.0, -2.0], [0.5, 2.0, 1.0]])
    np.testing.assert_array_equal(fe.output_gate(y, g), np.array([[0.0, 0.0, -4.0], [1.5, 8.0, 5.0]]))
