"""Pins for the CPU oracle (oracle/gdn_oracle.c): every test checks it against something OTHER than
itself -- a hand-worked example, brute force, closed forms, textbook/library reductions, invariants.
CPU only (-m "not gpu").  Pin numbers follow DESIGN.md "Oracle pins"."""
from pathlib import Path

import numpy as np
import pytest

import oracle
from tests import np_forms

GOLD = Path(__file__).parent / "golden"


def rnd(seed):
    return np.random.default_rng(seed)


def unit(x):
    return x / np.linalg.norm(x, axis=-1, keepdims=True)


def make(seed, T, dk, dv, G=1, B=1, H=1, key_scale=None, amin=0.3):
    r = rnd(seed)
    q = unit(r.standard_normal((B, T, H, dk))).astype(np.float32)
    k = unit(r.standard_normal((B, T, H, dk)))
    k = (k * (key_scale if key_scale is not None else (1.0 / np.sqrt(G) if G > 1 else 1.0))).astype(np.float32)
    v = r.standard_normal((B, T, H, dv)).astype(np.float32)
    alpha = r.uniform(amin, 1.0, (B, H, T // G)).astype(np.float32)
    beta = r.uniform(0.05, 0.95, (B, H, T)).astype(np.float32)
    S0 = (0.5 * r.standard_normal((B, H, dk, dv))).astype(np.float64)
    return q, k, v, alpha, beta, S0


def stream(x, b=0, h=0):
    """[B,T,H,d] -> [T,d] fp64 of one stream."""
    return np.asarray(x[b, :, h, :], dtype=np.float64)


# ---- pin 0: hand-worked example (tests/golden/handworked_d2.txt) ---------------------------------
def _golden():
    vals = {}
    for line in (GOLD / "handworked_d2.txt").read_text().splitlines():
        if line and not line.startswith("#"):
            name, *xs = line.split()
            vals[name] = np.array([float(x) for x in xs])
    return vals


@pytest.mark.parametrize("G", [1, 2])
def test_handworked_example(G):
    gold = _golden()
    q = np.array([[1, 1], [0.6, 0.8]], dtype=np.float32).reshape(1, 2, 1, 2)
    k = np.array([[1, 0], [0.6, 0.8]], dtype=np.float32).reshape(1, 2, 1, 2)
    v = np.array([[3], [1]], dtype=np.float32).reshape(1, 2, 1, 1)
    alpha = np.array([0.5, 1.0] if G == 1 else [0.5], dtype=np.float32).reshape(1, 1, -1)
    beta = np.array([0.5, 1.0], dtype=np.float32).reshape(1, 1, 2)
    S0 = np.array([[1.0], [2.0]]).reshape(1, 1, 2, 1)
    out, S = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=G)
    np.testing.assert_allclose(out.ravel(), gold[f"G{G}_out"], rtol=0, atol=2e-7)
    np.testing.assert_allclose(S.ravel(), gold[f"G{G}_state"], rtol=0, atol=2e-7)


# ---- pin 1: brute force product formula on tiny inputs -------------------------------------------
@pytest.mark.parametrize("T,dk,dv,G", [(8, 4, 3, 1), (6, 3, 4, 1), (8, 4, 4, 2), (8, 2, 3, 4), (6, 4, 2, 3)])
def test_brute_force_products(T, dk, dv, G):
    q, k, v, a, b, S0 = make(1, T, dk, dv, G, key_scale=0.9)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, group=G, scale=0.7)
    o2, S2 = np_forms.brute_force_products(stream(q), stream(k), stream(v), a[0, 0].astype(np.float64),
                                           b[0, 0].astype(np.float64), S0[0, 0], G, 0.7)
    np.testing.assert_allclose(out[0, :, 0], o2, rtol=0, atol=1e-13)
    np.testing.assert_allclose(S[0, 0], S2, rtol=0, atol=1e-13)


# ---- pin 2: three algebraic forms agree (Eq. 17-18 vs Eq. 19 vs Eq. 4-5) -------------------------
@pytest.mark.parametrize("G", [1, 4, 16])
def test_three_forms_agree(G):
    T, dk, dv = 64, 8, 6
    q, k, v, a, b, S0 = make(2, T, dk, dv, G)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    args = (stream(q), stream(k), stream(v), a[0, 0].astype(np.float64), b[0, 0].astype(np.float64), S0[0, 0])
    o2, S2 = np_forms.compact_form(*args, G)
    o3, S3 = np_forms.summaries_scan_readout(*args, G)
    for o, s in ((o2, S2), (o3, S3)):
        np.testing.assert_allclose(out[0, :, 0], o, rtol=0, atol=1e-13)
        np.testing.assert_allclose(S[0, 0], s, rtol=0, atol=1e-13)


# ---- pin 3: beta == 0 closed form: S_t = (prod alpha) S_in, o_t = (prod alpha) q_t S_in ----------
@pytest.mark.parametrize("G", [1, 4])
def test_beta_zero_closed_form(G):
    T, dk, dv = 32, 8, 8
    q, k, v, a, b, S0 = make(3, T, dk, dv, G)
    b[:] = 0
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    cum = np.cumprod(a[0, 0].astype(np.float64))
    exp_o = np.repeat(cum, G)[:, None] * (stream(q) @ S0[0, 0])
    np.testing.assert_allclose(out[0, :, 0], exp_o, rtol=0, atol=1e-14)
    np.testing.assert_allclose(S[0, 0], cum[-1] * S0[0, 0], rtol=0, atol=1e-14)


# ---- pin 4: orthonormal keys, S_in=0, T<=dk: gated linear attention with values beta*v -----------
def test_orthonormal_keys_reduce_to_gated_linear_attention():
    T = dk = 16
    dv = 8
    r = rnd(4)
    Qm, _ = np.linalg.qr(r.standard_normal((dk, dk)))
    q, k, v, a, b, _ = make(4, T, dk, dv)
    k[0, :, 0, :] = Qm[:T].astype(np.float32)
    kk = stream(k)
    out, S = oracle.gdn_forward(q, k, v, a, b, None)
    Gam = np.cumsum(np.log(a[0, 0].astype(np.float64)))
    M = np.tril(np.exp(Gam[:, None] - Gam[None, :]))              # diagonal included
    exp_o = (M * (stream(q) @ kk.T)) @ (b[0, 0][:, None].astype(np.float64) * stream(v))
    # k rows are orthonormal only up to fp32 rounding of the stored keys: tolerance 1e-6
    np.testing.assert_allclose(out[0, :, 0], exp_o, rtol=0, atol=5e-6)


# ---- pin 5: alpha=1, beta=1, orthonormal keys: plain causal linear attention; negative control ---
def test_reduces_to_causal_linear_attention_and_negative_control():
    T = dk = 12
    dv = 5
    r = rnd(5)
    Qm, _ = np.linalg.qr(r.standard_normal((dk, dk)))
    q, k, v, a, b, _ = make(5, T, dk, dv)
    a[:] = 1
    b[:] = 1
    k_orth = k.copy()
    k_orth[0, :, 0, :] = Qm.astype(np.float32)
    out, _ = oracle.gdn_forward(q, k_orth, v, a, b, None)
    exp_o = np.tril(stream(q) @ stream(k_orth).T) @ stream(v)
    np.testing.assert_allclose(out[0, :, 0], exp_o, rtol=0, atol=5e-6)
    # general (non-orthogonal) keys: the delta rule is NOT linear attention
    out2, _ = oracle.gdn_forward(q, k, v, a, b, None)
    exp2 = np.tril(stream(q) @ stream(k).T) @ stream(v)
    assert np.abs(out2[0, :, 0] - exp2).max() > 1e-2


# ---- pin 6: overwrite property: |k_t|=1, beta_t=1 => k_t S_t = v_t -------------------------------
def test_overwrite_property():
    T, dk, dv = 10, 6, 4
    q, k, v, a, b, S0 = make(6, T, dk, dv)
    b[:] = 1
    qk = k.copy()                                                  # read back with the key itself
    out, _ = oracle.gdn_forward(qk, k, v, a, b, S0)
    kn = np.linalg.norm(stream(k), axis=-1) ** 2                   # fp32-stored keys: |k|^2 = 1 + O(1e-7)
    np.testing.assert_allclose(out[0, :, 0], stream(v), rtol=0, atol=1e-5)
    assert np.abs(kn - 1).max() < 1e-6


# ---- pin 7: split invariance (streaming carry, App. G.6) -------------------------------
@pytest.mark.parametrize("G,T1", [(1, 7), (1, 20), (4, 8), (8, 24)])
def test_split_invariance(G, T1):
    T, dk, dv = 32, 8, 8
    q, k, v, a, b, S0 = make(7, T, dk, dv, G, B=2, H=2)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    o1, S1 = oracle.gdn_forward(q[:, :T1], k[:, :T1], v[:, :T1], a[..., :T1 // G], b[..., :T1], S0, group=G)
    o2, S2 = oracle.gdn_forward(q[:, T1:], k[:, T1:], v[:, T1:], a[..., T1 // G:], b[..., T1:], S1, group=G)
    assert np.array_equal(np.concatenate([o1, o2], axis=1), out)   # exact: same operations in the same order
    assert np.array_equal(S2, S)


# ---- pin 8/9: tile-size independence of the token-wise form via the chunkwise WY identities ------
@pytest.mark.parametrize("C", [16, 64, 100, 128])
def test_chunkwise_wy_matches_token_loop(C):
    T, dk, dv = 300, 16, 12
    q, k, v, a, b, S0 = make(9, T, dk, dv, amin=0.05)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0)
    o2, S2 = np_forms.chunkwise_wy(stream(q), stream(k), stream(v), a[0, 0].astype(np.float64),
                                   b[0, 0].astype(np.float64), S0[0, 0], C)
    np.testing.assert_allclose(out[0, :, 0], o2, rtol=0, atol=1e-12)
    np.testing.assert_allclose(S[0, 0], S2, rtol=0, atol=1e-12)


def test_affine_chunk_summaries_reproduce_state():
    T, dk, dv, C = 256, 16, 8, 64
    q, k, v, a, b, S0 = make(10, T, dk, dv)
    _, S = oracle.gdn_forward(q, k, v, a, b, S0)
    Ms, Ns = np_forms.affine_chunk_summaries(stream(k), stream(v), a[0, 0].astype(np.float64),
                                             b[0, 0].astype(np.float64), C)
    Sc = S0[0, 0]
    for M, N in zip(Ms, Ns):
        Sc = M @ Sc + N
    np.testing.assert_allclose(S[0, 0], Sc, rtol=0, atol=1e-12)


@pytest.mark.parametrize("C,NS,T", [(16, 1, 100), (16, 2, 100), (16, 4, 250), (8, 3, 64), (32, 4, 40)])
def test_two_level_segment_scan_matches_token_loop(C, NS, T):
    """SURVEY 8f NEXT-4 (Eq. 5): scanning segments from the identity map, composing the segment maps
    and fixing the outputs up afterwards gives the token loop (associativity of the affine maps), including a ragged
    last chunk, a shorter last segment and fewer chunks than segments."""
    dk, dv = 12, 10
    q, k, v, a, b, S0 = make(40 + NS, T, dk, dv, amin=0.1)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, scale=0.7)
    o2, S2 = np_forms.segment_scan(stream(q), stream(k), stream(v), a[0, 0].astype(np.float64), b[0, 0].astype(np.float64),
                                   S0[0, 0], C, NS, scale=0.7)
    np.testing.assert_allclose(out[0, :, 0], o2, rtol=0, atol=1e-12)
    np.testing.assert_allclose(S[0, 0], S2, rtol=0, atol=1e-12)


# ---- pin 10: joint linearity in (V, S_in) (L122) -------------------------------------------------
@pytest.mark.parametrize("G", [1, 8])
def test_linearity_in_v_and_state(G):
    T, dk, dv = 32, 8, 8
    q, k, v, a, b, S0 = make(11, T, dk, dv, G)
    _, _, v2, _, _, S02 = make(12, T, dk, dv, G)
    o1, s1 = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    o2, s2 = oracle.gdn_forward(q, k, v2, a, b, S02, group=G)
    # 2*v - 3*v2 is formed in fp64 then stored fp32: use exactly representable combos (x2, x-0.5 sums of fp32 are not exact) -> compare with fp32-rounded combo
    vc = (2.0 * v.astype(np.float64) - 0.5 * v2.astype(np.float64)).astype(np.float32)
    oc, sc = oracle.gdn_forward(q, k, vc, a, b, 2.0 * S0 - 0.5 * S02, group=G)
    np.testing.assert_allclose(oc, 2.0 * o1 - 0.5 * o2, rtol=0, atol=2e-6)
    np.testing.assert_allclose(sc, 2.0 * s1 - 0.5 * s2, rtol=0, atol=2e-6)


# ---- pin 11: column independence (L419-L423) -----------------------------------------------------
@pytest.mark.parametrize("G", [1, 8])
def test_column_independence(G):
    T, dk, dv = 32, 8, 8
    q, k, v, a, b, S0 = make(13, T, dk, dv, G)
    o1, s1 = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    v2, S02 = v.copy(), S0.copy()
    J = [1, 5]
    v2[..., J] += 1.0
    S02[..., J] -= 2.0
    o2, s2 = oracle.gdn_forward(q, k, v2, a, b, S02, group=G)
    keep = [j for j in range(dv) if j not in J]
    assert np.array_equal(o1[..., keep], o2[..., keep]) and np.array_equal(s1[..., keep], s2[..., keep])
    assert np.abs(o1[..., J] - o2[..., J]).max() > 1e-3


# ---- pin 12: permutation invariance inside a frame (mode F only) ---------------------------------
def test_permutation_inside_frame():
    T, dk, dv, G = 32, 8, 8, 8
    q, k, v, a, b, S0 = make(14, T, dk, dv, G)
    perm = np.concatenate([g * G + rnd(g).permutation(G) for g in range(T // G)])
    o1, s1 = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    o2, s2 = oracle.gdn_forward(q[:, perm], k[:, perm], v[:, perm], a, b[..., perm], S0, group=G)
    np.testing.assert_allclose(o2, o1[:, perm], rtol=0, atol=1e-13)
    np.testing.assert_allclose(s2, s1, rtol=0, atol=1e-13)
    # negative control: the token-wise recurrence is order dependent
    a1 = np.repeat(a, G, axis=-1)
    o3, s3 = oracle.gdn_forward(q, k * np.sqrt(G), v, a1, b, S0, group=1)
    o4, s4 = oracle.gdn_forward(q[:, perm], (k * np.sqrt(G))[:, perm], v[:, perm], a1[..., perm], b[..., perm], S0, group=1)
    assert np.abs(s3 - s4).max() > 1e-3


# ---- pin 13: normaliser path = matrix path with v == 1; mass conservation (L554, Eq. 20-22) ------
def test_normalizer_is_gdn_with_unit_values_and_mass_conservation():
    T, dk, dv, G = 24, 8, 4, 8
    r = rnd(15)
    q, k, v, a, b, S0 = make(15, T, dk, dv, G)
    q_raw = np.abs(q)
    k_raw = np.abs(k)
    z0 = r.uniform(0, 1, (1, 1, dk))
    out, S, z = oracle.gdn_forward(q, k, v, a, b, S0, group=G, q_raw=q_raw, k_raw=k_raw, z_in=z0, normalizer=True)
    # (a) z-path == matrix path on (q_raw,k_raw) with d_v = 1, v == 1
    ones = np.ones((1, T, 1, 1), dtype=np.float32)
    den, zS = oracle.gdn_forward(q_raw, k_raw, ones, a, b, z0[..., None], group=G)
    assert np.array_equal(zS[..., 0], z)
    num, S_plain = oracle.gdn_forward(q, k, v, a, b, S0, group=G)
    assert np.array_equal(S_plain, S)
    np.testing.assert_allclose(out, num / (den + 1e-6), rtol=1e-14, atol=0)
    # (b) mass conservation: rotated == raw, V == c, S_in = c z_in 1^T  =>  Y = c den/(den+eps)
    c = 1.5
    vc = np.full((1, T, 1, dv), c, dtype=np.float32)
    Sc = c * z0[..., None] * np.ones((1, 1, 1, dv))
    y, _, _ = oracle.gdn_forward(q_raw, k_raw, vc, a, b, Sc, group=G, q_raw=q_raw, k_raw=k_raw, z_in=z0, normalizer=True)
    np.testing.assert_allclose(y, c * (den / (den + 1e-6)) * np.ones((1, 1, 1, dv)), rtol=1e-12, atol=1e-14)


# ---- pin 14: scale equivariance ------------------------------------------------------------------
def test_scale_equivariance():
    T, dk, dv = 16, 8, 8
    q, k, v, a, b, S0 = make(16, T, dk, dv)
    o1, s1 = oracle.gdn_forward(q, k, v, a, b, S0, scale=1.0)
    o2, s2 = oracle.gdn_forward(q, k, v, a, b, S0, scale=0.25)
    assert np.array_equal(o2, 0.25 * o1) and np.array_equal(s1, s2)


# ---- strides / multi-stream plumbing: a sliced head view gives the same numbers ------------------
def test_strided_stream_views_and_threads():
    T, dk, dv = 16, 8, 8
    q, k, v, a, b, S0 = make(17, T, dk, dv, B=2, H=3)
    out, S = oracle.gdn_forward(q, k, v, a, b, S0, nthreads=3)
    for bi in range(2):
        for h in range(3):
            o1, s1 = oracle.gdn_forward(q[bi:bi + 1, :, h:h + 1], k[bi:bi + 1, :, h:h + 1], v[bi:bi + 1, :, h:h + 1],
                                        a[bi:bi + 1, h:h + 1], b[bi:bi + 1, h:h + 1], S0[bi:bi + 1, h:h + 1], nthreads=1)
            assert np.array_equal(o1[0, :, 0], out[bi, :, h]) and np.array_equal(s1[0, 0], S[bi, h])


def test_state_none_equals_zeros():
    T, dk, dv = 16, 8, 8
    q, k, v, a, b, S0 = make(18, T, dk, dv)
    o1, s1 = oracle.gdn_forward(q, k, v, a, b, None)
    o2, s2 = oracle.gdn_forward(q, k, v, a, b, np.zeros_like(S0))
    assert np.array_equal(o1, o2) and np.array_equal(s1, s2)


# ---- bidirectional in-chunk scan (Alg. 1 lines 8-22, L337-L359; L122, L145) ----------------------
def _dense_alg1(q, k, v, alpha, beta, S0, G, q_raw=None, k_raw=None, z0=None, eps=1e-6, scale=1.0):
    """Alg. 1 written with explicit frame summaries (Eq. 4-5): P_f = I - K^T diag(beta) K, A_f = K^T diag(beta) V,
    forward / reverse recursions on the matrices, one readout on the summed histories.  One stream, fp64."""
    T, dk = q.shape
    F = T // G
    P, A, Pz, bz = [], [], [], []
    for f in range(F):
        sl = slice(f * G, (f + 1) * G)
        Bm = np.diag(beta[sl])
        P.append(np.eye(dk) - k[sl].T @ Bm @ k[sl])
        A.append(k[sl].T @ Bm @ v[sl])
        if k_raw is not None:
            Pz.append(np.eye(dk) - k_raw[sl].T @ Bm @ k_raw[sl])
            bz.append(k_raw[sl].T @ beta[sl])
    fwd, S = [], S0.copy()
    for f in range(F):
        S = alpha[f] * P[f] @ S + A[f]
        fwd.append(S)
    rev = [None] * F
    rev[F - 1] = np.zeros_like(S0)
    for f in range(F - 1, 0, -1):
        rev[f - 1] = alpha[f] * P[f] @ rev[f] + A[f]
    if k_raw is not None:
        zf, z = [], z0.copy()
        for f in range(F):
            z = alpha[f] * Pz[f] @ z + bz[f]
            zf.append(z)
        zr = [None] * F
        zr[F - 1] = np.zeros_like(z0)
        for f in range(F - 1, 0, -1):
            zr[f - 1] = alpha[f] * Pz[f] @ zr[f] + bz[f]
    out = np.empty((T, v.shape[1]))
    for f in range(F):
        sl = slice(f * G, (f + 1) * G)
        num = scale * q[sl] @ (fwd[f] + rev[f])
        if k_raw is not None:
            num = num / (q_raw[sl] @ (zf[f] + zr[f]) + eps)[:, None]
        out[sl] = num
    return out, fwd[-1], (zf[-1] if k_raw is not None else None)


@pytest.mark.parametrize("G,F", [(1, 5), (3, 4), (8, 3)])
def test_bidir_matches_dense_algorithm_1(G, F):
    q, k, v, alpha, beta, S0 = make(40 + G, G * F, 5, 4, G=G, H=2)
    out, S = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=G, scale=0.7, bidir=True)
    for h in range(2):
        o_ref, S_ref, _ = _dense_alg1(stream(q, 0, h), stream(k, 0, h), stream(v, 0, h), alpha[0, h].astype(np.float64),
                                      beta[0, h].astype(np.float64), S0[0, h], G, scale=0.7)
        assert np.abs(out[0, :, h] - o_ref).max() < 1e-12 and np.abs(S[0, h] - S_ref).max() < 1e-12


def test_bidir_with_normaliser_matches_dense_algorithm_1():
    G, F, dk = 4, 3, 6
    r = rnd(77)
    q, k, v, alpha, beta, S0 = make(41, G * F, dk, 3, G=G)
    q_raw = np.abs(r.standard_normal(q.shape)).astype(np.float32)
    k_raw = (np.abs(r.standard_normal(k.shape)) / np.sqrt(dk * G)).astype(np.float32)
    z0 = np.abs(r.standard_normal((1, 1, dk)))
    out, S, z = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=G, q_raw=q_raw, k_raw=k_raw, z_in=z0, normalizer=True, bidir=True)
    o_ref, S_ref, z_ref = _dense_alg1(stream(q), stream(k), stream(v), alpha[0, 0].astype(np.float64), beta[0, 0].astype(np.float64),
                                      S0[0, 0], G, q_raw=stream(q_raw), k_raw=stream(k_raw), z0=z0[0, 0])
    assert np.abs(out[0, :, 0] - o_ref).max() < 1e-12 and np.abs(S[0, 0] - S_ref).max() < 1e-12 and np.abs(z[0, 0] - z_ref).max() < 1e-12


def test_bidir_single_frame_is_the_forward_scan_and_last_frame_never_changes():
    q, k, v, alpha, beta, S0 = make(42, 12, 4, 4, G=12)
    o1, s1 = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=12)
    o2, s2 = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=12, bidir=True)
    assert np.array_equal(o1, o2) and np.array_equal(s1, s2)                    # F = 1: S<_0 = 0
    q, k, v, alpha, beta, S0 = make(43, 12, 4, 4, G=4)
    o1, s1 = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=4)
    o2, s2 = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=4, bidir=True)
    assert np.array_equal(s1, s2) and np.array_equal(o1[:, 8:], o2[:, 8:])      # the cache and the last frame are forward-only
    assert np.abs(o1[:, :8] - o2[:, :8]).max() > 1e-2                           # negative control: earlier frames see the future


def test_bidir_two_frames_closed_form():
    """F = 2: S<_0 = alpha_1 P_1 0 + A_1 = K_1^T diag(beta_1) V_1, so frame 0 reads S>_0 + A_1."""
    G = 5
    q, k, v, alpha, beta, S0 = make(44, 2 * G, 4, 3, G=G)
    out, _ = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=G, bidir=True)
    _, S_f0 = oracle.gdn_forward(q[:, :G], k[:, :G], v[:, :G], alpha[:, :, :1], beta[:, :, :G], S0, group=G)   # forward state after frame 0
    K1, V1 = stream(k)[G:], stream(v)[G:]
    A1 = K1.T @ np.diag(beta[0, 0, G:].astype(np.float64)) @ V1
    assert np.abs(out[0, :G, 0] - stream(q)[:G] @ (S_f0[0, 0] + A1)).max() < 1e-12


def test_bidir_reverse_history_is_the_forward_scan_of_the_reversed_chunk():
    """S<_f is what a forward scan from zero over the frames F-1, F-2, ..., f+1 (in that order) leaves behind, so with
    the unidirectional oracle (pinned above) run on prefixes of the chunk and of the frame-reversed chunk:
    out_f = q_f (S>_f + S'>_{F-2-f})."""
    G, F, dk = 3, 4, 4
    q, k, v, alpha, beta, S0 = make(45, G * F, dk, 5, G=G)
    out, _ = oracle.gdn_forward(q, k, v, alpha, beta, S0, group=G, bidir=True)
    def rev_frames(x, axis):
        idx = np.concatenate([np.arange(f * G, (f + 1) * G) for f in range(F - 1, -1, -1)])
        return np.take(x, idx, axis=axis)
    kr, vr, br, ar = rev_frames(k, 1), rev_frames(v, 1), rev_frames(beta, 2), alpha[:, :, ::-1].copy()
    for f in range(F):
        _, Sf = oracle.gdn_forward(q[:, :(f + 1) * G], k[:, :(f + 1) * G], v[:, :(f + 1) * G], alpha[:, :, :f + 1], beta[:, :, :(f + 1) * G], S0, group=G)
        n = F - 1 - f                                                           # frames after f, scanned from the far end
        Sb = np.zeros_like(S0)
        if n > 0:
            _, Sb = oracle.gdn_forward(q[:, :n * G], kr[:, :n * G], vr[:, :n * G], ar[:, :, :n], br[:, :, :n * G], None, group=G)
        ref = stream(q)[f * G:(f + 1) * G] @ (Sf[0, 0] + Sb[0, 0])
        assert np.abs(out[0, f * G:(f + 1) * G, 0] - ref).max() < 1e-12
