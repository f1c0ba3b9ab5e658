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


@pytest.mark.parametrize("B,H,T,d,G", [(2, 16, 4096, 128, 1), (1, 16, 6144, 128, 2048), (2, 8, 4000, 128, 1)])
def test_host_entry_point_pipelined_segments(B, H, T, d, G):
    """Large enough for the host entry point to cut the call into token segments (copy-in | compute | copy-out
    pipeline, incl. a shorter tail segment and B > 1 strided segment copies): same result as one device call."""
    wl = gin.GdnWorkload("host_seg", B, H, T, d, d, group=G, seed=77)
    inp = gin.make_inputs(wl)
    o_dev, s_dev, _ = run_cuda(inp)
    pin = lambda t: t.contiguous().pin_memory()
    q, k, v, a, b, st = map(pin, (inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state))
    out = torch.full_like(inp.v, float("nan")).pin_memory()
    S_out = torch.full_like(inp.state, float("nan")).pin_memory()
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, group=G) as p:
        for _ in range(2):                                   # second call reuses the pipeline (events, staging)
            p.forward_host(q, k, v, a, b, st, out, S_out)
            torch.cuda.synchronize()
    o_ref, S_ref = run_oracle(inp)
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S_out, S_ref) <= TOL_BF16
    # one device call vs segments: the state crosses a segment boundary as fp32 S_out/S_in instead of staying in
    # registers, so single bf16 roundings of out may flip (one ulp of bf16 = 3.9e-3 relative)
    assert rel_err(out, o_dev.double().numpy()) <= 1e-2 and rel_err(S_out, s_dev.double().numpy()) <= 1e-3


def test_host_entry_point_bidirectional_is_never_segmented():
    """The paper's production chunk (3 x 880 tokens, 20 heads, d = 128: ~40 MB of input, above the segmentation
    threshold) through the HOST entry point with GDN_FLAG_BIDIR: the reverse scan of Alg. 1 l.14-17 spans all frames
    of the call, so the host path must not cut the call into token segments."""
    import oracle
    wl = gin.paper_shape(3)
    inp = gin.make_inputs(wl)
    pin = lambda t: t.contiguous().pin_memory()
    q, k, v, a, b, st = map(pin, (inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state))
    out = torch.full_like(inp.v, float("nan")).pin_memory()
    S_out = torch.full_like(inp.state, float("nan")).pin_memory()
    with gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=wl.group, flags=gdn.GDN_FLAG_BIDIR) as p:
        p.forward_host(q, k, v, a, b, st, out, S_out)
        torch.cuda.synchronize()
    o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=wl.group, bidir=True)
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S_out, S_ref) <= TOL_BF16


def test_host_entry_point_segment_gate_slots_stay_aligned():
    """Frame mode with B*H*F_seg not a multiple of 4 (H = 6, one frame per segment): every segment's alpha slot in the
    staging buffer must still be 16-byte aligned."""
    B, H, G, F, d = 1, 6, 4096, 4, 128
    wl = gin.GdnWorkload("host_align", B, H, G * F, d, d, group=G, seed=78)
    inp = gin.make_inputs(wl)
    pin = lambda t: t.contiguous().pin_memory()
    q, k, v, a, b, st = map(pin, (inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state))
    out = torch.full_like(inp.v, float("nan")).pin_memory()
    S_out = torch.full_like(inp.state, float("nan")).pin_memory()
    with gdn.GdnPlan(B=B, H=H, T=G * F, d_k=d, d_v=d, group=G) as p:
        p.forward_host(q, k, v, a, b, st, out, S_out)
        torch.cuda.synchronize()
    o_ref, S_ref = run_oracle(inp)
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S_out, S_ref) <= TOL_BF16


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


@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("B,H,G,F", [(1, 2, 352, 2), (2, 3, 880, 3), (1, 20, 256, 1),
                                     (1, 20, 880, 3)])      # 420 tiles on 148 readout CTAs: several tiles and frame changes per CTA
def test_normalizer_readout_tensor_core_frame_path(d, B, H, G, F):
    """Paper Eq. 20-22 on the tcgen05 frame path (bf16): the z recurrence runs through the same three kernels as
    column 0 of a matrix state; out = scale q S / (q_raw . z + eps).  z updated in place."""
    import oracle
    T = G * F
    wl = gin.GdnWorkload("norm_tc", B, H, T, d, d, group=G, seed=31)
    inp = gin.make_normalizer_inputs(wl)
    dev = torch.device("cuda:0")
    ex = inp.extras
    out = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
    S_out = torch.empty(B, H, d, d, device=dev)
    z = ex["z_in"].to(dev)
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, group=G, scale=0.5, flags=gdn.GDN_FLAG_NORMALIZER) as p:
        assert gdn.PATH_NAMES[p.info.path] == "tc_frame"
        for _ in range(2):                                        # the second call must not depend on leftovers of the first
            z.copy_(ex["z_in"])
            p.forward_norm(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev),
                           inp.alpha.to(dev), inp.beta.to(dev), inp.state.to(dev), z, out, S_out, z)
            torch.cuda.synchronize()
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, scale=0.5,
                                             q_raw=ex["q_raw"], k_raw=ex["k_raw"], z_in=ex["z_in"], normalizer=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16
    assert rel_err(S_out.cpu(), S_ref) <= TOL_BF16 and rel_err(z.cpu(), z_ref) <= TOL_BF16


def test_normalizer_tensor_core_frame_path_with_different_q_and_k_token_strides():
    """q / q_raw dense, k / k_raw / v with a packed token stride: k_raw is read with k's stride (include/gdn.h)."""
    import oracle
    B, H, G, F, d = 1, 4, 352, 2, 128
    T = G * F
    wl = gin.GdnWorkload("norm_strided", B, H, T, d, d, group=G, seed=34)
    inp = gin.make_normalizer_inputs(wl)
    ex = inp.extras
    dev = torch.device("cuda:0")
    kv = torch.stack([inp.k, inp.v], dim=2).contiguous().to(dev)                # [B,T,2,H,d]
    kr = torch.stack([ex["k_raw"], torch.zeros_like(ex["k_raw"])], dim=2).contiguous().to(dev)
    out = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
    S_out = torch.empty(B, H, d, d, device=dev)
    z = ex["z_in"].to(dev)
    ts = 2 * H * d
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_NORMALIZER,
                     k_token_stride=ts, v_token_stride=ts) as p:
        assert gdn.PATH_NAMES[p.info.path] == "tc_frame"
        p.forward_norm(inp.q.to(dev), kv[:, :, 0], kv[:, :, 1], ex["q_raw"].to(dev), kr[:, :, 0],
                       inp.alpha.to(dev), inp.beta.to(dev), inp.state.to(dev), z, out, S_out, z)
        torch.cuda.synchronize()
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G,
                                             q_raw=ex["q_raw"], k_raw=ex["k_raw"], z_in=ex["z_in"], normalizer=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16
    assert rel_err(S_out.cpu(), S_ref) <= TOL_BF16 and rel_err(z.cpu(), z_ref) <= TOL_BF16


# ---- bidirectional in-chunk scan (Alg. 1 l.8-22) on the frame path ------------------------------------
@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("B,H,G,F", [(1, 2, 256, 1), (1, 3, 352, 2), (2, 2, 880, 3), (1, 20, 200, 5)])
def test_bidirectional_frame_path(d, B, H, G, F):
    T = G * F
    wl = gin.GdnWorkload("bidir", B, H, T, d, d, group=G, seed=51)
    inp = gin.make_inputs(wl)
    out, S, info = run_cuda(inp, flags=gdn.GDN_FLAG_BIDIR, scale=0.8)
    assert gdn.PATH_NAMES[info[0]] == "tc_frame"
    import oracle
    o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, scale=0.8, bidir=True)
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S, S_ref) <= TOL_BF16
    if F > 1:                                                   # negative control: the forward-only result is far away
        o_fwd, _ = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, scale=0.8)
        assert rel_err(out, o_fwd) > 5 * TOL_BF16


def test_bidirectional_stream_with_normaliser_carries_forward_states():
    """Two chunks of the paper's shape (3 frames of 880 tokens, 20 heads, d = 128), bidirectional + normalised
    readout; the carried S and z are the FORWARD terminal states (L145: forward scan with the previous cache)."""
    import oracle
    B, H, G, F, d = 1, 20, 880, 3, 128
    T = G * F
    dev = torch.device("cuda:0")
    S_d = z_d = None
    S_o = z_o = None
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_NORMALIZER | gdn.GDN_FLAG_BIDIR) as p:
        for ci in range(2):
            wl = gin.GdnWorkload("bidir_norm", B, H, T, d, d, group=G, seed=60 + ci)
            inp = gin.make_normalizer_inputs(wl)
            ex = inp.extras
            if ci == 0:
                S_d, z_d = inp.state.to(dev), ex["z_in"].to(dev)
                S_o, z_o = inp.state, ex["z_in"]
            out = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
            p.forward_norm(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev),
                           inp.alpha.to(dev), inp.beta.to(dev), S_d, z_d, out, S_d, z_d)
            torch.cuda.synchronize()
            o_ref, S_o, z_o = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, S_o, group=G, q_raw=ex["q_raw"],
                                                 k_raw=ex["k_raw"], z_in=z_o, normalizer=True, bidir=True)
            assert rel_err(out.cpu(), o_ref) <= TOL_BF16
            assert rel_err(S_d.cpu(), S_o) <= TOL_BF16 and rel_err(z_d.cpu(), z_o) <= TOL_BF16


def test_bidirectional_log_alpha_zero_state_and_rerun_is_bit_identical():
    """log-alpha input, state_in = NULL, and determinism: two runs of the same call give the same bits (fixed reduction
    orders everywhere: DESIGN.md reading 17), also with a token split in Phase A (few heads -> NSPLIT > 1)."""
    import oracle
    B, H, G, F, d = 1, 2, 1000, 3, 128
    wl = gin.GdnWorkload("bidir_log", B, H, G * F, d, d, group=G, seed=52)
    inp = gin.make_inputs(wl)
    dev = torch.device("cuda:0")
    q, k, v, b = inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), inp.beta.to(dev)
    la = torch.log(inp.alpha).to(dev)
    outs = []
    with gdn.GdnPlan(B=B, H=H, T=G * F, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_BIDIR | gdn.GDN_FLAG_LOG_ALPHA) as p:
        for _ in range(2):
            out = torch.empty(B, G * F, H, d, device=dev, dtype=torch.bfloat16)
            S = torch.empty(B, H, d, d, device=dev)
            p.forward(q, k, v, la, b, None, out, S)
            torch.cuda.synchronize()
            outs.append((out.cpu(), S.cpu()))
    assert torch.equal(outs[0][0], outs[1][0]) and torch.equal(outs[0][1], outs[1][1])
    o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, None, group=G, bidir=True)
    assert rel_err(outs[0][0], o_ref) <= TOL_BF16 and rel_err(outs[0][1], S_ref) <= TOL_BF16


def test_normalizer_tensor_core_zero_z_and_separate_output_and_errors():
    import oracle
    B, H, G, F, d = 1, 3, 300, 2, 64
    wl = gin.GdnWorkload("norm_tc0", B, H, G * F, d, d, group=G, seed=33)
    inp = gin.make_normalizer_inputs(wl)
    ex = inp.extras
    dev = torch.device("cuda:0")
    out = torch.empty(B, G * F, H, d, device=dev, dtype=torch.bfloat16)
    S_out = torch.empty(B, H, d, d, device=dev)
    z_out = torch.full((B, H, d), float("nan"), device=dev)
    args = [inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev), inp.alpha.to(dev), inp.beta.to(dev)]
    with gdn.GdnPlan(B=B, H=H, T=G * F, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_NORMALIZER) as p:
        p.forward_norm(*args, None, None, out, S_out, z_out)               # S_in = z_in = NULL: zeros
        torch.cuda.synchronize()
        with pytest.raises(gdn.GdnError):                                  # q_raw missing
            p.forward_norm(args[0], args[1], args[2], None, args[4], args[5], args[6], None, None, out, S_out, z_out)
        with pytest.raises(gdn.GdnError):                                  # plain entry point on a normaliser plan
            p.forward(args[0], args[1], args[2], args[5], args[6], None, out, S_out)
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, None, group=G, q_raw=ex["q_raw"],
                                             k_raw=ex["k_raw"], z_in=None, normalizer=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16 and rel_err(S_out.cpu(), S_ref) <= TOL_BF16 and rel_err(z_out.cpu(), z_ref) <= TOL_BF16


# ---- head dim 112 (the paper's; "Pad head dimension to BLOCK_D = 128", Alg. 1 l.1, L316) -----------------
@pytest.mark.parametrize("G,F,H", [(1, 1000, 3), (880, 3, 20), (352, 2, 4)])
def test_head_dim_112_is_padded_inside_the_kernels(G, F, H):
    """d_k = d_v = 112 tensors go in and come out unpadded: the tensor maps zero-fill / clip features 112..127 and the
    state is [112][112]; token-wise (fused kernel) and frame-wise."""
    T = F if G == 1 else G * F
    wl = gin.GdnWorkload("d112", 1, H, T, 112, 112, group=G, seed=71)
    inp = gin.make_inputs(wl)
    out, S, info = run_cuda(inp)
    assert gdn.PATH_NAMES[info[0]] in ("tc_token", "tc_frame")
    o_ref, S_ref = run_oracle(inp)
    assert out.shape[-1] == 112 and S.shape[-2:] == (112, 112)
    assert rel_err(out, o_ref) <= TOL_BF16 and rel_err(S, S_ref) <= TOL_BF16


def test_head_dim_112_full_operator_at_the_papers_shape():
    import oracle
    B, H, G, F, d = 1, 20, 880, 3, 112
    wl = gin.GdnWorkload("d112_full", B, H, G * F, d, d, group=G, seed=72)
    inp = gin.make_normalizer_inputs(wl)
    ex = inp.extras
    dev = torch.device("cuda:0")
    out = torch.empty(B, G * F, H, d, device=dev, dtype=torch.bfloat16)
    S_out = torch.empty(B, H, d, d, device=dev)
    z = ex["z_in"].to(dev)
    with gdn.GdnPlan(B=B, H=H, T=G * F, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_NORMALIZER | gdn.GDN_FLAG_BIDIR) as p:
        p.forward_norm(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev),
                       inp.alpha.to(dev), inp.beta.to(dev), inp.state.to(dev), z, out, S_out, z)
        torch.cuda.synchronize()
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, q_raw=ex["q_raw"],
                                             k_raw=ex["k_raw"], z_in=ex["z_in"], normalizer=True, bidir=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16 and rel_err(S_out.cpu(), S_ref) <= TOL_BF16 and rel_err(z.cpu(), z_ref) <= TOL_BF16


def test_head_dim_112_is_refused_without_a_tensor_core_path():
    for kw in (dict(io_dtype=gdn.GDN_FP32), dict(chunk=64), dict(flags=gdn.GDN_FLAG_FORCE_SIMT), dict(d_v=128)):
        args = dict(B=1, H=2, T=256, d_k=112, d_v=112)
        args.update(kw)
        with pytest.raises(gdn.GdnError) as ei:
            gdn.GdnPlan(**args)
        assert ei.value.status == gdn.GDN_ERR_UNSUPPORTED


def test_bidirectional_flag_is_refused_where_it_has_no_path():
    for kw in (dict(group=1), dict(group=64, io_dtype=gdn.GDN_FP32), dict(group=64, d_k=32, d_v=32)):
        args = dict(B=1, H=2, T=256, d_k=64, d_v=64, flags=gdn.GDN_FLAG_BIDIR)
        args.update(kw)
        with pytest.raises(gdn.GdnError) as ei:
            gdn.GdnPlan(**args)
        assert ei.value.status == gdn.GDN_ERR_UNSUPPORTED


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


# =====================================================================================================
# Tensor-core (tcgen05) token-wise path: BASELINE.json's configs, literal (G = 1)
# =====================================================================================================
def _assert_tc(info):
    assert info[0] == 1, f"expected the tensor-core token path, plan resolved to {info}"


@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("C", [64, 128])
@pytest.mark.parametrize("T", [1, 64, 128, 129, 200, 704, 1000])
def test_tc_token_small(d, C, T):
    wl = gin.GdnWorkload("tc", 2, 3, T, d, d, seed=7 * d + C + T, chunk=C)
    eo, es, info = check(gin.make_inputs(wl))
    _assert_tc(info)
    assert info[1] == C


@pytest.mark.parametrize("C", [64, 128])
def test_tc_token_zero_state_and_scale(C):
    wl = gin.GdnWorkload("tc0", 1, 2, 512, 64, 64, seed=21, chunk=C)
    inp = gin.make_inputs(wl)
    check(inp, state_in=None, scale=0.125)


def test_tc_token_matches_simt_kernel():
    """Two independent CUDA implementations (tensor-core chunkwise vs fp32 token loop) agree."""
    wl = gin.GdnWorkload("x", 1, 4, 1024, 128, 128, seed=22)
    inp = gin.make_inputs(wl)
    o1, s1, i1 = run_cuda(inp)
    o2, s2, i2 = run_cuda(inp, flags=gdn.GDN_FLAG_FORCE_SIMT)
    assert i1[0] == 1 and i2[0] == 0
    assert rel_err(o1, o2.double().numpy()) <= TOL_BF16 and rel_err(s1, s2.double().numpy()) <= TOL_BF16


@pytest.mark.parametrize("cfg", [2, 5])
def test_fused_token_kernel_is_bit_repeatable_over_many_calls(cfg):
    """The fused kernel hands tiles from prepass workers to chain workers through release / acquire flags in L2 (the
    release is issued by a different thread than the one that waited for the TMA stores).  A hand-over that is not
    properly ordered shows up as a stale summary, i.e. as a run that differs from the others: 40 calls on the same
    inputs (rotating output buffers, state fed back) must reproduce the first pass bit for bit."""
    wl = gin.config(cfg)
    inp = gin.make_inputs(wl)
    dev = torch.device("cuda:0")
    q, k, v, a, b = (t.to(dev) for t in (inp.q, inp.k, inp.v, inp.alpha, inp.beta))
    outs = [torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=wl.dtype, device=dev) for _ in range(4)]
    ref = None
    with gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v) as p:
        assert p.info.launches_per_call == 1
        for rep in range(10):
            S = inp.state.to(dev).clone()
            res = []
            for i in range(4):                                   # a 4-call stream: state carried
                p.forward(q, k, v, a, b, S, outs[i], S)
                res.append(outs[i])
            torch.cuda.synchronize()
            cur = [o.clone() for o in res] + [S.clone()]
            if ref is None:
                ref = cur
            else:
                assert all(torch.equal(x, y) for x, y in zip(cur, ref)), f"pass {rep} differs from pass 0"


@pytest.mark.parametrize("C", [64, 128])
def test_config2(C):
    eo, es, info = check(gin.make_inputs(gin.config(2, chunk=C)))
    _assert_tc(info)


@pytest.mark.parametrize("C", [64, 128])
def test_config3(C):
    eo, es, info = check(gin.make_inputs(gin.config(3, chunk=C)))
    _assert_tc(info)


def test_config4_stream_of_20_chunks():
    """20-chunk stream: the CUDA path carries its own fp32 state, the oracle carries its own fp64 state;
    the error is tracked per chunk (it may accumulate -- that is the point of the config)."""
    import oracle
    dev = torch.device("cuda:0")
    wl = gin.config(4)
    plan = gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=1, chunk=wl.chunk)
    inp0 = gin.make_inputs(wl)
    S_gpu = inp0.state.to(dev)
    S_ref = inp0.state.double().numpy()
    out = torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=torch.bfloat16, device=dev)
    errs = []
    for i in range(20):
        inp = gin.make_inputs(gin.config(4, chunk_index=i), with_state=False)
        plan.forward(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), inp.alpha.to(dev), inp.beta.to(dev), S_gpu, out, S_gpu)
        torch.cuda.synchronize()
        o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, S_ref)
        errs.append((rel_err(out.cpu(), o_ref), rel_err(S_gpu.cpu(), S_ref)))
    plan.close()
    print("config 4 per-chunk (err_o, err_S):", [(f"{a:.2e}", f"{b:.2e}") for a, b in errs])
    assert max(e[0] for e in errs) <= TOL_BF16 and max(e[1] for e in errs) <= TOL_BF16


@pytest.mark.parametrize("T", [3520, 10560])
def test_config5_stress(T):
    """Strong decay tail (alpha down to ~2e-3): both compute tiles against the oracle and against each other."""
    res = {}
    inp = gin.make_inputs(gin.config(5, T=T))
    o_ref, S_ref = run_oracle(inp)
    for C in (64, 128):
        out, S, info = run_cuda(inp, chunk=C)
        _assert_tc(info)
        eo, es = rel_err(out, o_ref), rel_err(S, S_ref)
        assert eo <= TOL_BF16 and es <= TOL_BF16, f"C={C}: err_o={eo:.3e} err_S={es:.3e}"
        res[C] = (out, S)
    assert rel_err(res[64][0], res[128][0].double().numpy()) <= TOL_BF16
    assert rel_err(res[64][1], res[128][1].double().numpy()) <= TOL_BF16


def _oracle_all_streams(inp, group=1, heads_per_call=16):
    """The oracle on EVERY (b,h) stream of a large input, a few heads at a time (bounds host memory; OpenMP runs the
    streams of one call in parallel) -> yields (b, h0, h1, out [T,h1-h0,dv], S [h1-h0,dk,dv])."""
    import oracle
    wl = inp.wl
    for b in range(wl.B):
        for h0 in range(0, wl.H, heads_per_call):
            h1 = min(wl.H, h0 + heads_per_call)
            o, s = oracle.gdn_forward(inp.q[b:b + 1, :, h0:h1], inp.k[b:b + 1, :, h0:h1], inp.v[b:b + 1, :, h0:h1],
                                      inp.alpha[b:b + 1, h0:h1], inp.beta[b:b + 1, h0:h1],
                                      None if inp.state is None else inp.state[b:b + 1, h0:h1], group=group)
            yield b, h0, h1, o[0], s[0]


@pytest.mark.slow
def test_config5_T65536_all_streams():
    """Full size (B=2, H=32, T=65536, d=128): the oracle runs on ALL 64 (b,h) streams (first and last stream of each
    batch included: the largest workspace / activation offsets), both compute tiles, plus C=64 vs C=128 agreement."""
    inp = gin.make_inputs(gin.config(5, T=65536))
    outs = {}
    for C in (128, 64):
        out, S, info = run_cuda(inp, chunk=C)
        _assert_tc(info)
        assert torch.isfinite(out.float()).all() and torch.isfinite(S).all()
        outs[C] = (out, S)
    worst = {128: (0.0, 0.0, None), 64: (0.0, 0.0, None)}
    for b, h0, h1, o_ref, S_ref in _oracle_all_streams(inp):
        for C in (128, 64):
            out, S = outs[C]
            for h in range(h0, h1):
                eo, es = rel_err(out[b, :, h], o_ref[:, h - h0]), rel_err(S[b, h], S_ref[h - h0])
                assert eo <= TOL_BF16 and es <= TOL_BF16, f"C={C} stream {(b, h)}: err_o={eo:.3e} err_S={es:.3e}"
                if eo > worst[C][0]:
                    worst[C] = (eo, es, (b, h))
    print("config 5 T=65536 worst stream per tile size (err_o, err_S, (b,h)):", worst)
    assert rel_err(outs[64][0], outs[128][0].double().numpy()) <= TOL_BF16
    assert rel_err(outs[64][1], outs[128][1].double().numpy()) <= TOL_BF16


# =====================================================================================================
# Tensor-core (tcgen05) frame-wise path: the paper's variant (G = tokens per frame), same shapes
# =====================================================================================================
def _assert_tc_frame(info):
    assert info[0] == 2, f"expected the tensor-core frame path, plan resolved to {info}"


@pytest.mark.parametrize("d", [64, 128])
@pytest.mark.parametrize("G,F", [(1 * 128, 1), (100, 3), (128, 4), (352, 2), (880, 3), (1000, 2)])
def test_tc_frame_small(d, G, F):
    wl = gin.GdnWorkload("tcF", 2, 3, G * F, d, d, group=G, seed=3 * d + G + F)
    eo, es, info = check(gin.make_inputs(wl))
    _assert_tc_frame(info)


def test_tc_frame_zero_state_scale_and_log_alpha():
    wl = gin.GdnWorkload("tcF0", 1, 2, 3 * 352, 64, 64, group=352, seed=31)
    inp = gin.make_inputs(wl)
    check(inp, state_in=None, scale=0.5)
    o1, s1, _ = run_cuda(inp)
    inp2 = gin.make_inputs(wl)
    inp2.alpha = torch.log(inp.alpha)
    o2, s2, _ = run_cuda(inp2, flags=gdn.GDN_FLAG_LOG_ALPHA)
    assert rel_err(o2, o1.double().numpy()) < 1e-2 and rel_err(s2, s1.double().numpy()) < 1e-3


def test_tc_frame_matches_simt_kernel():
    wl = gin.GdnWorkload("xF", 1, 4, 2 * 880, 128, 128, group=880, seed=32)
    inp = gin.make_inputs(wl)
    o1, s1, i1 = run_cuda(inp)
    o2, s2, i2 = run_cuda(inp, flags=gdn.GDN_FLAG_FORCE_SIMT)
    assert i1[0] == 2 and i2[0] == 0
    assert rel_err(o1, o2.double().numpy()) <= TOL_BF16 and rel_err(s1, s2.double().numpy()) <= TOL_BF16


@pytest.mark.parametrize("cfg", [2, 3])
def test_config_frame_variants(cfg):
    eo, es, info = check(gin.make_inputs(gin.config(cfg, frame=True)))
    _assert_tc_frame(info)


@pytest.mark.parametrize("frames", [3, 5])
def test_paper_shape(frames):
    """The paper's production chunk: 880 tokens per frame (22x40), 20 heads, d = 128; 5-frame first chunk, 3 after."""
    eo, es, info = check(gin.make_inputs(gin.paper_shape(frames)))
    _assert_tc_frame(info)


def test_config4_frame_stream():
    """Frame-wise 20-chunk stream with carried state (config 4, G = 3520)."""
    import oracle
    dev = torch.device("cuda:0")
    wl = gin.config(4, frame=True)
    plan = gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=wl.group)
    inp0 = gin.make_inputs(wl)
    S_gpu = inp0.state.to(dev)
    S_ref = inp0.state.double().numpy()
    out = torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=torch.bfloat16, device=dev)
    errs = []
    for i in range(20):
        inp = gin.make_inputs(gin.config(4, frame=True, chunk_index=i), with_state=False)
        plan.forward(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), inp.alpha.to(dev), inp.beta.to(dev), S_gpu, out, S_gpu)
        torch.cuda.synchronize()
        o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, S_ref, group=wl.group)
        errs.append((rel_err(out.cpu(), o_ref), rel_err(S_gpu.cpu(), S_ref)))
    plan.close()
    print("config 4 (frame-wise) per-chunk (err_o, err_S):", [(f"{a:.2e}", f"{b:.2e}") for a, b in errs])
    assert max(e[0] for e in errs) <= TOL_BF16 and max(e[1] for e in errs) <= TOL_BF16


@pytest.mark.parametrize("T", [3520, 10560])
def test_config5_frame(T):
    eo, es, info = check(gin.make_inputs(gin.config(5, T=T, frame=True)))
    _assert_tc_frame(info)


@pytest.mark.slow
def test_config5_frame_T65536_all_streams():
    inp = gin.make_inputs(gin.config(5, T=65536, frame=True))
    out, S, info = run_cuda(inp)
    _assert_tc_frame(info)
    assert torch.isfinite(out.float()).all() and torch.isfinite(S).all()
    for b, h0, h1, o_ref, S_ref in _oracle_all_streams(inp, group=inp.wl.group):
        for h in range(h0, h1):
            eo, es = rel_err(out[b, :, h], o_ref[:, h - h0]), rel_err(S[b, h], S_ref[h - h0])
            assert eo <= TOL_BF16 and es <= TOL_BF16, f"stream {(b, h)}: err_o={eo:.3e} err_S={es:.3e}"


# =====================================================================================================
# d = 64, C = 64: light 64-token tile workers (gdn_tc_tile64.cuh) and the single persistent kernel with the
# two-level, segment-parallel scan (gdn_tc_fused64.cuh, Eq. 5)
# =====================================================================================================
@pytest.mark.parametrize("T", [64, 200, 704, 3520])
def test_tile64_three_kernel_path(T):
    """GDN_FLAG_UNFUSED + chunk 64 at d = 64: gdn_tok_tile64 feeds the chain and output kernels."""
    wl = gin.GdnWorkload("tile64u", 2, 3, T, 64, 64, seed=900 + T, chunk=64)
    eo, es, info = check(gin.make_inputs(wl), flags=gdn.GDN_FLAG_UNFUSED)
    assert info == (1, 64, 3)


@pytest.mark.parametrize("B,H,T", [(1, 16, 3520), (2, 32, 704), (1, 2, 8192), (1, 1, 130), (3, 5, 64)])
def test_fused64_two_level_scan(B, H, T):
    """One launch; the number of segments per stream follows the stream count (64 streams: plain scan, NS = 1;
    few streams: NS up to 4), so the shapes cover segment 0, the identity-started segments, level 2 and short tails."""
    wl = gin.GdnWorkload("fused64", B, H, T, 64, 64, seed=950 + T + H, chunk=64)
    eo, es, info = check(gin.make_inputs(wl))
    assert info == (1, 64, 1)
    print(f"fused64 B={B} H={H} T={T}: err_o={eo:.2e} err_S={es:.2e}")


def test_fused64_stream_with_carried_state_and_rerun_is_bit_identical():
    """Carried state over four calls on one plan (epoch-stamped flags are never reset), log-alpha input, and the same
    bits on a second pass over the same inputs (fixed reduction orders: DESIGN.md reading 17)."""
    B, H, T = 1, 4, 1000
    dev = torch.device("cuda:0")
    runs = []
    for rep in range(2):
        with gdn.GdnPlan(B=B, H=H, T=T, d_k=64, d_v=64, group=1, chunk=64, flags=gdn.GDN_FLAG_LOG_ALPHA) as p:
            S = torch.zeros(B, H, 64, 64, device=dev)
            S_ref = None
            outs = []
            for ci in range(4):
                inp = gin.make_inputs(gin.GdnWorkload("f64s", B, H, T, 64, 64, seed=970 + ci, chunk=64), with_state=False)
                out = torch.empty(B, T, H, 64, device=dev, dtype=torch.bfloat16)
                p.forward(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), torch.log(inp.alpha).to(dev), inp.beta.to(dev), S, out, S)
                torch.cuda.synchronize()
                outs.append(out.cpu())
                if rep == 0:
                    import oracle
                    o_ref, S_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, S_ref, group=1)
                    assert rel_err(out.cpu(), o_ref) <= TOL_BF16 and rel_err(S.cpu(), S_ref) <= TOL_BF16
            runs.append((outs, S.cpu()))
    assert all(torch.equal(a, b) for a, b in zip(runs[0][0], runs[1][0])) and torch.equal(runs[0][1], runs[1][1])


def test_host_entry_point_pipelined_across_calls():
    """Five unsegmented host calls issued back to back WITHOUT synchronising in between, each with its own inputs and
    output buffer, the state carried through ONE host buffer (state_out of call i is state_in of call i + 1): the
    double-buffered input staging and the stream-ordered state copies must give exactly what the device path gives."""
    B, H, T, d = 1, 4, 1024, 64
    dev = torch.device("cuda:0")
    pin = lambda t: t.contiguous().pin_memory()
    inps = [gin.make_inputs(gin.GdnWorkload("hostpipe", B, H, T, d, d, seed=80 + i), with_state=False) for i in range(5)]
    host = [tuple(map(pin, (x.q, x.k, x.v, x.alpha, x.beta))) for x in inps]
    outs = [torch.full((B, T, H, d), float("nan"), dtype=torch.bfloat16).pin_memory() for _ in inps]
    hs = pin(0.02 * torch.randn(B, H, d, d, generator=torch.Generator().manual_seed(5)))
    S0 = hs.clone()
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d) as p:
        for (q, k, v, a, b), o in zip(host, outs):
            p.forward_host(q, k, v, a, b, hs, o, hs)
        torch.cuda.synchronize()
        S = S0.to(dev)
        for x, o in zip(inps, outs):
            od = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
            p.forward(x.q.to(dev), x.k.to(dev), x.v.to(dev), x.alpha.to(dev), x.beta.to(dev), S, od, S)
            torch.cuda.synchronize()
            assert torch.equal(o, od.cpu())
        assert torch.equal(hs, S.cpu())


def test_host_entry_point_input_that_is_the_previous_calls_output_stays_in_stream_order():
    """The copy-in of an unsegmented host call does not wait for the caller's stream -- EXCEPT when an input overlaps a host
    buffer the previous call writes (gdn.h).  Call 2 takes call 1's out_host as its v_host, with no synchronisation in
    between: the result must be what two device calls chained through that tensor give."""
    B, H, T, d = 1, 4, 1024, 64
    dev = torch.device("cuda:0")
    pin = lambda t: t.contiguous().pin_memory()
    x1 = gin.make_inputs(gin.GdnWorkload("hostchain", B, H, T, d, d, seed=90), with_state=False)
    x2 = gin.make_inputs(gin.GdnWorkload("hostchain", B, H, T, d, d, seed=91), with_state=False)
    h1 = tuple(map(pin, (x1.q, x1.k, x1.v, x1.alpha, x1.beta)))
    h2 = tuple(map(pin, (x2.q, x2.k, x2.v, x2.alpha, x2.beta)))
    o1 = torch.full((B, T, H, d), float("nan"), dtype=torch.bfloat16).pin_memory()
    o2 = torch.full((B, T, H, d), float("nan"), dtype=torch.bfloat16).pin_memory()
    hs = pin(torch.zeros(B, H, d, d))
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d) as p:
        for _ in range(3):                                   # (the third round runs with both staging sets in use)
            hs.zero_()
            p.forward_host(h1[0], h1[1], h1[2], h1[3], h1[4], hs, o1, hs)
            p.forward_host(h2[0], h2[1], o1, h2[3], h2[4], hs, o2, hs)       # v = the previous call's output
            torch.cuda.synchronize()
        S = torch.zeros(B, H, d, d, device=dev)
        d1 = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
        d2 = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
        p.forward(x1.q.to(dev), x1.k.to(dev), x1.v.to(dev), x1.alpha.to(dev), x1.beta.to(dev), S, d1, S)
        p.forward(x2.q.to(dev), x2.k.to(dev), d1, x2.alpha.to(dev), x2.beta.to(dev), S, d2, S)
        torch.cuda.synchronize()
        assert torch.equal(o1, d1.cpu()) and torch.equal(o2, d2.cpu()) and torch.equal(hs, S.cpu())


@pytest.mark.parametrize("B,H,G,F,d", [
    (1, 20, 40, 6, 128),        # frames shorter than one 64-token tile of the dual Phase A
    (1, 40, 65, 7, 128),        # one token over a tile, seven frames, more (b, h, f, column) units than SMs
    (2, 10, 64, 3, 128),        # exactly one tile per frame
    (1, 20, 129, 3, 64),        # d = 64: the two-stream path (no dual Phase A), one token over a 128-token tile
])
def test_normalised_bidirectional_short_and_ragged_frames(B, H, G, F, d):
    """Alg. 1 with the normalised readout on frame lengths around the tile sizes of Phase A (64 tokens in the dual kernel,
    128 otherwise), called twice on the same plan (the bidirectional path adds both scans into snapshot slots that Phase A
    must have zeroed again)."""
    import oracle
    T = G * F
    dev = torch.device("cuda:0")
    wl = gin.GdnWorkload("ragged", B, H, T, d, d, group=G, seed=77)
    inp = gin.make_normalizer_inputs(wl)
    ex = inp.extras
    out = torch.empty(B, T, H, d, device=dev, dtype=torch.bfloat16)
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=d, d_v=d, group=G, flags=gdn.GDN_FLAG_NORMALIZER | gdn.GDN_FLAG_BIDIR) as p:
        for _ in range(2):
            S, z = inp.state.to(dev), ex["z_in"].to(dev)
            p.forward_norm(inp.q.to(dev), inp.k.to(dev), inp.v.to(dev), ex["q_raw"].to(dev), ex["k_raw"].to(dev),
                           inp.alpha.to(dev), inp.beta.to(dev), S, z, out, S, z)
            torch.cuda.synchronize()
    o_ref, S_ref, z_ref = oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, inp.state, group=G, q_raw=ex["q_raw"],
                                             k_raw=ex["k_raw"], z_in=ex["z_in"], normalizer=True, bidir=True)
    assert rel_err(out.cpu(), o_ref) <= TOL_BF16 and rel_err(S.cpu(), S_ref) <= TOL_BF16 and rel_err(z.cpu(), z_ref) <= TOL_BF16
