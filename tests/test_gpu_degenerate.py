"""Degenerate-gate inputs pushed through the CUDA paths (tensor-core token path at C = 64 / 128 and the frame
path, d = 64 / 128) and compared with the oracle: SURVEY.md section 8(c) pins 3-6 "again on the GPU path", plus
the decay edge cases of T0-T2 (Eq. 17-19): alpha == 1, beta == 0, beta == 1 with unit keys
(overwrite), orthonormal keys from a zero state, a run of alpha ~ 1e-30 (the in-tile cumulative decay underflows
fp32), alpha at the fp32 denormal edge, and an alpha of exactly 1.0f in the middle of a tile.

The inputs come from the seeded generator; only the gates (and, where a pin needs it, the keys) are overwritten here.
Tolerances are north_star's (tests/gpu_util.py), untouched."""
import numpy as np
import pytest
import torch

import oracle
import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import inputs as gin
from tests.gpu_util import TOL_BF16, rel_err, run_cuda, run_oracle

pytestmark = pytest.mark.gpu

T_TOK = 3 * 128 + 72          # three full 128-token tiles and a ragged tail (also ragged for C = 64)


def _check(inp, **kw):
    out, S, info = run_cuda(inp, **kw)
    o_ref, S_ref = run_oracle(inp, **{k: v for k, v in kw.items() if k in ("state_in", "scale")})
    eo, es = rel_err(out, o_ref), rel_err(S, S_ref)
    assert eo <= TOL_BF16 and es <= TOL_BF16, f"{inp.wl.name}: err_o={eo:.3e} err_S={es:.3e} path={info}"
    return out, S, o_ref, S_ref, info


def _tok(name, d, C, seed, T=T_TOK, H=3, B=2):
    return gin.make_inputs(gin.GdnWorkload(name, B, H, T, d, d, seed=seed, chunk=C))


def _frm(name, d, seed, G=352, F=4, H=3, B=2):
    return gin.make_inputs(gin.GdnWorkload(name, B, H, G * F, d, d, group=G, seed=seed))


def _hadamard(n):
    h = np.array([[1.0]])
    while h.shape[0] < n:
        h = np.block([[h, h], [h, -h]])
    return h


def _orthonormal_rows(T, d):
    """T <= d exactly orthonormal rows that are exact in bf16: rows of block-diagonal 64x64 Hadamard matrices / 8."""
    blk = _hadamard(64) / 8.0
    m = np.zeros((d, d))
    for i in range(d // 64):
        m[64 * i:64 * (i + 1), 64 * i:64 * (i + 1)] = blk
    return torch.tensor(m[:T], dtype=torch.float32)


# ---------------------------------------------------------------------------------------- token path
TOK = [(64, 64), (64, 128), (128, 64), (128, 128)]


@pytest.mark.parametrize("d,C", TOK)
def test_token_alpha_identically_one(d, C):
    inp = _tok("a1", d, C, 901)
    inp.alpha = torch.ones_like(inp.alpha)            # log alpha = 0, gamma == 1 everywhere
    *_, info = _check(inp)
    assert info[0] == 1 and info[1] == C


@pytest.mark.parametrize("d,C", TOK)
def test_token_beta_identically_zero_state_only_decays(d, C):
    """Pin 3: L = 0, Tm = I, no write: S_T = (prod alpha) S_in and o_t = (prod_{s<=t} alpha_s) q_t S_in."""
    inp = _tok("b0", d, C, 902)
    inp.beta = torch.zeros_like(inp.beta)
    out, S, o_ref, S_ref, info = _check(inp)
    assert info[0] == 1
    g = torch.cumprod(inp.alpha.double(), dim=-1)                                   # [B,H,T]
    o_closed = torch.einsum("bthk,bhkv->bthv", inp.q.double(), inp.state.double()) * g.permute(0, 2, 1)[..., None]
    S_closed = inp.state.double() * g[..., -1, None, None]
    assert rel_err(out, o_closed.numpy()) <= TOL_BF16 and rel_err(S, S_closed.numpy()) <= TOL_BF16


@pytest.mark.parametrize("d,C", TOK)
def test_token_beta_one_unit_keys_overwrite(d, C):
    """Pin 6: beta == 1 and unit-norm keys: k_t S_t = v_t.  With q = k the output IS that product.  bf16 keys are unit
    norm to 2^-8, so the property holds to that (well inside the bar); the oracle comparison is the bar proper."""
    inp = _tok("b1", d, C, 903)
    inp.beta = torch.ones_like(inp.beta)
    inp.q = inp.k.clone()
    out, S, o_ref, S_ref, info = _check(inp)
    assert info[0] == 1
    assert rel_err(out, inp.v.double().numpy()) <= TOL_BF16


@pytest.mark.parametrize("d,C", TOK)
def test_token_orthonormal_keys_zero_state_is_gated_linear_attention(d, C):
    """Pins 4-5: orthonormal keys, S_in = 0, T <= d: the erase term vanishes and o = (M o QK^T)(beta o V),
    M_ij = prod_{r=j+1..i} alpha_r (j <= i).  Second run with alpha == beta == 1: plain causal linear attention."""
    T = d
    wl = gin.GdnWorkload("ortho", 2, 3, T, d, d, seed=904, chunk=C)
    inp = gin.make_inputs(wl)
    inp.k = _orthonormal_rows(T, d)[None, :, None, :].expand(2, T, 3, d).contiguous().to(torch.bfloat16)
    for plain in (False, True):
        if plain:
            inp.alpha, inp.beta = torch.ones_like(inp.alpha), torch.ones_like(inp.beta)
        out, S, info = run_cuda(inp, state_in=None)
        o_ref, S_ref = run_oracle(inp, state_in=None)
        assert info[0] == 1
        assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S, S_ref) <= TOL_BF16
        lg = torch.cumsum(torch.log(inp.alpha.double()), dim=-1)                    # [B,H,T]
        M = torch.tril(torch.exp(lg[..., :, None] - lg[..., None, :]))
        qk = torch.einsum("bihk,bjhk->bhij", inp.q.double(), inp.k.double())
        dense = torch.einsum("bhij,bjhv->bihv", M * qk, inp.beta.double().permute(0, 2, 1)[..., None] * inp.v.double())
        assert rel_err(out, dense.numpy()) <= TOL_BF16


@pytest.mark.parametrize("d,C", TOK)
def test_token_decay_underflow_denormal_edge_and_exact_one_mid_tile(d, C):
    """T0-T2 edge cases in ONE stream each: a run of alpha ~ 1e-30 inside a tile (its cumulative product underflows fp32
    after two tokens: every exponent the kernel forms must stay a difference <= 0 and flush to 0, not to NaN / inf),
    alpha at the fp32 denormal edge (1.2e-38, and a true denormal 1e-41), and alpha = 1.0f exactly in mid tile."""
    inp = _tok("edge", d, C, 905)
    a = inp.alpha.clone()
    a[0, 0, 40:56] = 1e-30                       # run inside the first tile
    a[0, 0, 200:203] = 1e-30                     # and across nothing special, second tile
    a[0, 1, 130] = 1.17549435e-38                # smallest normal
    a[0, 1, 300] = 1e-41                         # denormal
    a[0, 2, 60:70] = 1.0                         # exactly 1 across the C = 64 chunk boundary
    a[1, 0, 127] = 1e-30                         # last row of a tile
    a[1, 1, 128] = 1e-30                         # first row of a tile
    a[1, 2, T_TOK - 1] = 1e-30                   # last token of the ragged tail
    inp.alpha = a
    out, S, o_ref, S_ref, info = _check(inp)
    assert info[0] == 1
    assert torch.isfinite(out.float()).all() and torch.isfinite(S).all()


# ---------------------------------------------------------------------------------------- frame path
@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("case", ["alpha1", "beta0", "beta1", "tiny_alpha", "denormal_alpha", "one_mid"])
def test_frame_degenerate_gates(d, case):
    inp = _frm(f"F_{case}", d, 910)
    if case == "alpha1":
        inp.alpha = torch.ones_like(inp.alpha)
    elif case == "beta0":
        inp.beta = torch.zeros_like(inp.beta)
    elif case == "beta1":
        inp.beta = torch.ones_like(inp.beta)
    elif case == "tiny_alpha":
        inp.alpha[:, :, 1] = 1e-30
        inp.alpha[0, 0, :] = 1e-30               # the cumulative product over the call underflows fp32
    elif case == "denormal_alpha":
        inp.alpha[0, 1, 2] = 1e-41
        inp.alpha[1, 0, 0] = 1.17549435e-38
    elif case == "one_mid":
        inp.alpha[:, :, 2] = 1.0
    out, S, o_ref, S_ref, info = _check(inp)
    assert info[0] == 2
    assert torch.isfinite(out.float()).all() and torch.isfinite(S).all()
    if case == "beta0":                          # pin 3 on the frame path: the state only decays
        g = torch.cumprod(inp.alpha.double(), dim=-1)
        S_closed = inp.state.double() * g[..., -1, None, None]
        assert rel_err(S, S_closed.numpy()) <= TOL_BF16


@pytest.mark.parametrize("d", [64, 128])
def test_frame_bidirectional_degenerate_gates(d):
    """The reverse scan of Alg. 1 l.14-17 under the same edge gates (alpha == 1 on one frame, ~1e-30 on another, beta == 0
    on a whole frame)."""
    G, F = 352, 4
    inp = _frm("F_bidir_edge", d, 911, G=G, F=F)
    inp.alpha[:, :, 1] = 1.0
    inp.alpha[:, :, 2] = 1e-30
    inp.beta[:, :, 3 * G:4 * G] = 0.0
    out, S, info = run_cuda(inp, flags=gdn.GDN_FLAG_BIDIR)
    o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, bidir=True)
    assert info[0] == 2
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S, S_ref) <= TOL_BF16
