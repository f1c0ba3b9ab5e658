"""Parity of the CUDA path (through the C ABI) against the CPU oracle, element by element, on the
same seeded inputs.  Bars (north_star): max|o - o_ref| <= 2e-2 * max|o_ref| for bf16 inputs with fp32
state, <= 1e-4 in the fp32-input mode; same rule for state_out (reading 16)."""
import numpy as np
import pytest
import torch

import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import inputs as gin
from tests.gpu_util import TOL_BF16, TOL_FP32, rel_err, run_cuda, run_oracle, tol_for

pytestmark = pytest.mark.gpu


def check(inp, **kw):
    out, S, info = run_cuda(inp, **kw)
    okw = {k: v for k, v in kw.items() if k in ("state_in", "scale")}
    o_ref, S_ref = run_oracle(inp, **okw)
    tol = tol_for(inp.wl.dtype)
    eo, es = rel_err(out, o_ref), rel_err(S, S_ref)
    assert eo <= tol and es <= tol, f"{inp.wl.name}: err_o={eo:.3e} err_S={es:.3e} tol={tol} path={info}"
    return eo, es, info


# ---- config 1 (fp32-input mode, tolerance 1e-4), token-wise and frame-wise ------------------------
@pytest.mark.parametrize("frame", [False, True])
def test_config1_fp32(frame):
    inp = gin.make_inputs(gin.config(1, frame=frame))
    eo, es, info = check(inp)
    assert info[0] == 0            # fp32 io always takes the fp32 CUDA-core kernel
    assert eo < TOL_FP32


def test_config1_fp32_with_state_and_scale():
    wl = gin.config(1).with_(state_std=0.5, seed=11)
    check(gin.make_inputs(wl), scale=0.5)


# ---- the fp32 CUDA-core kernel on bf16 inputs, all head dims, ragged lengths ----------------------
@pytest.mark.parametrize("d", [32, 64, 128])
@pytest.mark.parametrize("T,G", [(1, 1), (67, 1), (200, 1), (192, 48), (96, 96)])
def test_simt_kernel_bf16(d, T, G):
    wl = gin.GdnWorkload("simt", 2, 3, T, d, d, group=G, seed=100 + d + T)
    check(gin.make_inputs(wl), flags=gdn.GDN_FLAG_FORCE_SIMT)


def test_simt_rectangular_state():
    wl = gin.GdnWorkload("rect", 1, 2, 130, 64, 128, seed=5)
    check(gin.make_inputs(wl), flags=gdn.GDN_FLAG_FORCE_SIMT)
    wl = gin.GdnWorkload("rect", 1, 2, 130, 128, 32, seed=6)
    check(gin.make_inputs(wl), flags=gdn.GDN_FLAG_FORCE_SIMT)


# ---- degenerate cases ------------------------------------------------------------------------------
def test_empty_chunk_passes_state_through():
    dev = torch.device("cuda:0")
    S = torch.randn(1, 2, 32, 32, device=dev)
    S_out = torch.zeros_like(S)
    with gdn.GdnPlan(B=1, H=2, T=0, d_k=32, d_v=32) as p:
        p.forward(None, None, None, None, None, S, None, S_out)
        torch.cuda.synchronize()
        assert torch.equal(S, S_out)
        p.forward(None, None, None, None, None, None, None, S_out)
        torch.cuda.synchronize()
        assert float(S_out.abs().max()) == 0.0
    with gdn.GdnPlan(B=0, H=2, T=64, d_k=32, d_v=32) as p:
        p.forward(None, None, None, None, None, None, None, None)


def test_state_none_equals_zero_state_and_inplace_state():
    wl = gin.GdnWorkload("st", 1, 2, 96, 32, 32, dtype=torch.float32, seed=3)
    inp = gin.make_inputs(wl)
    o1, s1, _ = run_cuda(inp, state_in=None)
    o2, s2, _ = run_cuda(inp, state_in=torch.zeros(1, 2, 32, 32))
    assert torch.equal(o1, o2) and torch.equal(s1, s2)
    # state_out aliasing state_in (streaming use)
    dev = torch.device("cuda:0")
    st = inp.state.to(dev)
    out = torch.empty(1, 96, 2, 32, device=dev)
    with gdn.GdnPlan(B=1, H=2, T=96, d_k=32, d_v=32, io_dtype=gdn.GDN_FP32) as p:
        p.forward(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), inp.alpha.to(dev), inp.beta.to(dev), st, out, st)
        torch.cuda.synchronize()
    o3, s3, _ = run_cuda(inp)
    assert torch.equal(out.cpu(), o3) and torch.equal(st.cpu(), s3)


def test_alignment_and_alias_errors():
    dev = torch.device("cuda:0")
    x = torch.zeros(1 * 64 * 1 * 32 + 8, dtype=torch.bfloat16, device=dev)
    a = torch.zeros(64, device=dev)
    S = torch.zeros(32 * 32, device=dev)
    with gdn.GdnPlan(B=1, H=1, T=64, d_k=32, d_v=32) as p:
        with pytest.raises(gdn.GdnError) as ei:
            p.forward(x.data_ptr() + 2, x, x, a, a, None, torch.empty_like(x), S)
        assert ei.value.status == gdn.GDN_ERR_ALIGNMENT
        with pytest.raises(gdn.GdnError) as ei:
            p.forward(x, x, x, a, a, None, x, S)
        assert ei.value.status == gdn.GDN_ERR_INVALID_ARG


# ---- options: log-alpha, packed qkv strides, host entry point -------------------------------------
def test_log_alpha_flag():
    wl = gin.GdnWorkload("la", 1, 2, 128, 32, 32, dtype=torch.float32, seed=8)
    inp = gin.make_inputs(wl)
    o1, s1, _ = run_cuda(inp)
    inp2 = gin.make_inputs(wl)
    inp2.alpha = torch.log(inp.alpha)
    o2, s2, _ = run_cuda(inp2, flags=gdn.GDN_FLAG_LOG_ALPHA)
    assert rel_err(o2, o1.double().numpy()) < 1e-5 and rel_err(s2, s1.double().numpy()) < 1e-5


@pytest.mark.parametrize("force_simt", [True, False])
def test_packed_qkv_token_stride(force_simt):
    B, H, T, d = 1, 4, 256, 64
    wl = gin.GdnWorkload("packed", B, H, T, d, d, seed=9)
    inp = gin.make_inputs(wl)
    dev = torch.device("cuda:0")
    qkv = torch.stack([inp.q, inp.k, inp.v], dim=2).contiguous().to(dev)      # [B,T,3,H,d]
    out = torch.empty(B, T, H, d, dtype=torch.bfloat16, device=dev)
    S_out = torch.empty(B, H, d, d, device=dev)
    ts = 3 * H * d
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, q_token_stride=ts, k_token_stride=ts, v_token_stride=ts,
                     flags=gdn.GDN_FLAG_FORCE_SIMT if force_simt else 0) as p:
        p.forward(qkv[:, :, 0], qkv[:, :, 1], qkv[:, :, 2], inp.alpha.to(dev), inp.beta.to(dev),
                  inp.state.to(dev), out, S_out)
        torch.cuda.synchronize()
    o_ref, S_ref = run_oracle(inp)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16 and rel_err(S_out.cpu(), S_ref) <= TOL_BF16


def test_host_entry_point_matches_device_call():
    wl = gin.GdnWorkload("host", 1, 2, 192, 64, 64, seed=10)
    inp = gin.make_inputs(wl)
    o_dev, s_dev, _ = run_cuda(inp)
    pin = lambda t: t.contiguous().pin_memory()
    q, k, v, a, b, st = map(pin, (inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state))
    out = torch.empty_like(inp.v).pin_memory()
    S_out = torch.empty_like(inp.state).pin_memory()
    with gdn.GdnPlan(B=1, H=2, T=192, d_k=64, d_v=64) as p:
        p.forward_host(q, k, v, a, b, st, out, S_out)
        torch.cuda.synchronize()
    assert torch.equal(out, o_dev) and torch.equal(S_out, s_dev)


# ---- normaliser path (paper Eq. 20-22) --------------------------------------------------------------
@pytest.mark.parametrize("G", [1, 64])
def test_normalizer_readout(G):
    import oracle
    wl = gin.GdnWorkload("norm", 1, 2, 256, 64, 64, group=G, seed=12, dtype=torch.float32)
    inp = gin.make_normalizer_inputs(wl)
    dev = torch.device("cuda:0")
    ex = inp.extras
    out = torch.empty(1, 256, 2, 64, device=dev)
    S_out = torch.empty(1, 2, 64, 64, device=dev)
    z = ex["z_in"].to(dev)
    with gdn.GdnPlan(B=1, H=2, T=256, d_k=64, d_v=64, group=G, io_dtype=gdn.GDN_FP32, flags=gdn.GDN_FLAG_NORMALIZER) as p:
        p.forward_norm(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev),
                       inp.alpha.to(dev), inp.beta.to(dev), inp.state.to(dev), z, out, S_out, z)   # z in place
        torch.cuda.synchronize()
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G,
                                             q_raw=ex["q_raw"], k_raw=ex["k_raw"], z_in=ex["z_in"], normalizer=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_FP32
    assert rel_err(S_out.cpu(), S_ref) <= TOL_FP32 and rel_err(z.cpu(), z_ref) <= TOL_FP32


# ---- streaming carry: split invariance on the device path -------------------------------------------
@pytest.mark.parametrize("G", [1, 32])
def test_split_invariance_device(G):
    wl = gin.GdnWorkload("split", 1, 2, 256, 32, 32, dtype=torch.float32, group=G, seed=13)
    inp = gin.make_inputs(wl)
    o_full, s_full, _ = run_cuda(inp)
    T1 = 96
    def part(lo, hi, st):
        w = wl.with_(T=hi - lo)
        i2 = gin.GdnInputs(w, inp.q[:, lo:hi].contiguous(), inp.k[:, lo:hi].contiguous(), inp.v[:, lo:hi].contiguous(),
                           inp.alpha[..., lo // G:hi // G].contiguous(), inp.beta[..., lo:hi].contiguous(), st)
        return run_cuda(i2)
    o1, s1, _ = part(0, T1, inp.state)
    o2, s2, _ = part(T1, 256, s1)
    assert torch.equal(torch.cat([o1, o2], dim=1), o_full) and torch.equal(s2, s_full)
