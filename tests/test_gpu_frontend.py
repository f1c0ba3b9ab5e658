"""GPU parity of the block's front end against oracle/frontend.py (Eq. 12-15, 23, L554; Alg. 1 boundary):
gdn_feature_map, gdn_compute_gates, gdn_forward_chunk_full.  All through the C ABI."""
import numpy as np
import pytest
import torch

import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import inputs as gin
from tests.gpu_util import rel_err

pytestmark = pytest.mark.gpu
TOL_BF16 = 2e-2
DEV = "cuda:0"


def _packed_views(fi):
    qkv = fi["qkv"]
    return qkv[:, :, 0], qkv[:, :, 1], qkv[:, :, 2]


def _plan(B, H, T, D, G, flags, packed=True):
    kw = {}
    if packed:
        kw = dict(q_token_stride=3 * H * D, k_token_stride=3 * H * D, v_token_stride=3 * H * D)
    return gdn.GdnPlan(B=B, H=H, T=T, d_k=D, d_v=D, group=G, flags=flags, **kw)


@pytest.mark.parametrize("D,G,F,H", [(112, 880, 3, 20), (128, 352, 2, 4), (64, 200, 3, 3)])
def test_feature_map_matches_oracle(D, G, F, H):
    from oracle import frontend as fe
    B, T = 2 if D != 112 else 1, G * F
    wl = gin.GdnWorkload("fm", B, H, T, D, D, group=G, seed=300 + D)
    fi = gin.make_frontend_inputs(wl)
    qkv = fi["qkv"].to(DEV)
    q_d, k_d = qkv[:, :, 0], qkv[:, :, 1]
    outs = [torch.empty(B, T, H, D, device=DEV, dtype=torch.bfloat16) for _ in range(4)]
    with _plan(B, H, T, D, G, gdn.GDN_FLAG_NORMALIZER) as p:
        fm = gdn.make_featmap_args(q_d, k_d, fi["w_q"].to(DEV), fi["w_k"].to(DEV), fi["cos"].to(DEV), fi["sin"].to(DEV), 1e-6)
        wq, wk, cs, sn = (fi[n].to(DEV) for n in ("w_q", "w_k", "cos", "sin"))
        fm = gdn.make_featmap_args(q_d, k_d, wq, wk, cs, sn, 1e-6)
        p.feature_map(fm, *outs)
        torch.cuda.synchronize()
    q, k, _ = _packed_views(fi)
    ref = fe.feature_map(q, k, fi["w_q"], fi["w_k"], fi["cos"], fi["sin"], group=G, eps_rms=1e-6)
    for name, got, want in zip(("q_rot", "k_rot", "q_raw", "k_raw"), outs, ref):
        err = np.abs(got.cpu().double().numpy() - want).max() / np.abs(want).max()
        assert err <= 2 ** -8, f"{name}: {err:.3e}"          # one bf16 rounding of an fp32 evaluation
    assert (outs[2].cpu().float() >= 0).all() and (outs[3].cpu().float() >= 0).all()


@pytest.mark.parametrize("log_alpha", [False, True])
@pytest.mark.parametrize("D,G,F,H,B", [(112, 880, 3, 20, 1), (64, 3520, 1, 2, 1), (128, 100, 4, 3, 2)])
def test_gates_match_oracle_and_are_deterministic(D, G, F, H, B, log_alpha):
    from oracle import frontend as fe
    T = G * F
    wl = gin.GdnWorkload("gates", B, H, T, D, D, group=G, seed=400 + D)
    fi = gin.make_frontend_inputs(wl)
    dev = {n: fi[n].to(DEV) for n in ("x", "w_alpha", "b_alpha", "a_log", "w_beta", "b_beta")}
    flags = gdn.GDN_FLAG_NORMALIZER | (gdn.GDN_FLAG_LOG_ALPHA if log_alpha else 0)
    res = []
    with _plan(B, H, T, D, G, flags, packed=False) as p:
        ga = gdn.make_gate_args(dev["x"], dev["w_alpha"], dev["b_alpha"], dev["a_log"], dev["w_beta"], dev["b_beta"])
        for _ in range(2):
            a = torch.full((B, H, F), float("nan"), device=DEV)
            b = torch.full((B, H, T), float("nan"), device=DEV)
            p.compute_gates(ga, a, b)
            torch.cuda.synchronize()
            res.append((a.cpu(), b.cpu()))
    assert torch.equal(res[0][0], res[1][0]) and torch.equal(res[0][1], res[1][1])      # fixed summation order
    alpha, la, beta = fe.gates(fi["x"], fi["w_alpha"], fi["b_alpha"], fi["a_log"], fi["w_beta"], fi["b_beta"], group=G)
    want_a = la if log_alpha else alpha
    np.testing.assert_allclose(res[0][0].double().numpy(), want_a, rtol=2e-5, atol=2e-6)
    np.testing.assert_allclose(res[0][1].double().numpy(), beta, rtol=2e-5, atol=2e-6)


def _full_reference(fi, wl, G, use_gates, alpha, beta, bidir, gate):
    import oracle
    from oracle import frontend as fe
    q, k, v = _packed_views(fi)
    q_rot, k_rot, q_raw, k_raw = fe.feature_map(q, k, fi["w_q"], fi["w_k"], fi["cos"], fi["sin"], group=G, eps_rms=1e-6)
    if use_gates:
        alpha, _, beta = fe.gates(fi["x"], fi["w_alpha"], fi["b_alpha"], fi["a_log"], fi["w_beta"], fi["b_beta"], group=G)
    o, S, z = oracle.gdn_forward(q_rot, k_rot, v, alpha, beta, fi["state"], group=G, q_raw=q_raw, k_raw=k_raw, z_in=fi["z_in"],
                                 normalizer=True, bidir=bidir)
    if gate:
        o = fe.output_gate(o, fi["gate"])
    return o, S, z


@pytest.mark.parametrize("D,G,F,H,bidir,use_gates,gate", [
    (112, 880, 3, 20, True, True, True),          # the paper's production chunk, its full operator (Alg. 1)
    (128, 352, 2, 4, False, False, True),
    (64, 200, 3, 3, True, True, False),
])
def test_forward_full_matches_oracle(D, G, F, H, bidir, use_gates, gate):
    B, T = 1, G * F
    wl = gin.GdnWorkload("full", B, H, T, D, D, group=G, seed=500 + D)
    fi = gin.make_frontend_inputs(wl)
    g = torch.Generator().manual_seed(7)
    alpha = torch.sigmoid(3 + torch.randn(B, H, F, generator=g))
    beta = torch.sigmoid(torch.randn(B, H, T, generator=g))
    qkv = fi["qkv"].to(DEV)
    dv = {n: fi[n].to(DEV) for n in ("x", "w_q", "w_k", "cos", "sin", "w_alpha", "b_alpha", "a_log", "w_beta", "b_beta", "gate")}
    S = fi["state"].to(DEV)
    z = fi["z_in"].to(DEV)
    out = torch.empty(B, T, H, D, device=DEV, dtype=torch.bfloat16)
    flags = gdn.GDN_FLAG_NORMALIZER | (gdn.GDN_FLAG_BIDIR if bidir else 0)
    with _plan(B, H, T, D, G, flags) as p:
        fm = gdn.make_featmap_args(qkv[:, :, 0], qkv[:, :, 1], dv["w_q"], dv["w_k"], dv["cos"], dv["sin"], 1e-6)
        ga = gdn.make_gate_args(dv["x"], dv["w_alpha"], dv["b_alpha"], dv["a_log"], dv["w_beta"], dv["b_beta"]) if use_gates else None
        p.forward_full(fm, qkv[:, :, 2], ga, None if use_gates else alpha.to(DEV), None if use_gates else beta.to(DEV),
                       dv["gate"] if gate else None, S, z, out, S, z)
        torch.cuda.synchronize()
    o_ref, S_ref, z_ref = _full_reference(fi, wl, G, use_gates, alpha, beta, bidir, gate)
    eo, es, ez = rel_err(out.cpu(), o_ref), rel_err(S.cpu(), S_ref), rel_err(z.cpu(), z_ref)
    print(f"full D={D} G={G} F={F} bidir={bidir} gates={use_gates} gate={gate}: err_o={eo:.2e} err_S={es:.2e} err_z={ez:.2e}")
    assert eo <= TOL_BF16 and es <= TOL_BF16 and ez <= TOL_BF16


def test_front_end_rejects_unsupported_plans():
    with gdn.GdnPlan(B=1, H=2, T=256, d_k=64, d_v=64, group=1) as p:         # token-wise: no full operator
        with pytest.raises(gdn.GdnError) as ei:
            p.forward_full(gdn.make_featmap_args(0, 0, 0, 0, 0, 0), 0, None, 0, 0, None, None, None, 0, 0, 0)
        assert ei.value.status == gdn.GDN_ERR_UNSUPPORTED


def test_graph_replay_on_a_user_stream_matches_direct_calls():
    """On a non-default stream the frame-wise calls are captured once per tuple of argument pointers and replayed as a
    CUDA graph (gdn_api.cu: run_graphed).  Two input sets alternate over six calls with a carried state; the outputs
    must be bit-identical to the same six calls on the default stream (issued directly), for the plain frame path, the
    normalised + bidirectional one and the full operator."""
    B, H, G, F, D = 1, 4, 352, 2, 128
    T = G * F
    wl = gin.GdnWorkload("graph", B, H, T, D, D, group=G, seed=600)
    sets = []
    for i in range(2):
        fi = gin.make_frontend_inputs(wl, seed=600 + i)
        d = {n: fi[n].to(DEV) for n in fi}
        d["out"] = torch.empty(B, T, H, D, device=DEV, dtype=torch.bfloat16)
        sets.append(d)
    g = torch.Generator().manual_seed(3)
    alpha = torch.sigmoid(3 + torch.randn(B, H, F, generator=g)).to(DEV)
    beta = torch.sigmoid(torch.randn(B, H, T, generator=g)).to(DEV)
    st3 = 3 * H * D
    results = {}
    for mode in ("direct", "graph"):
        stream = torch.cuda.current_stream() if mode == "direct" else torch.cuda.Stream()
        stream.wait_stream(torch.cuda.current_stream())
        outs = []
        with gdn.GdnPlan(B=B, H=H, T=T, d_k=D, d_v=D, group=G, flags=gdn.GDN_FLAG_NORMALIZER | gdn.GDN_FLAG_BIDIR,
                         q_token_stride=st3, k_token_stride=st3, v_token_stride=st3) as p, \
             gdn.GdnPlan(B=B, H=H, T=T, d_k=D, d_v=D, group=G, q_token_stride=st3, k_token_stride=st3, v_token_stride=st3) as pp:
            S = sets[0]["state"].clone()
            z = sets[0]["z_in"].clone()
            S2 = sets[0]["state"].clone()
            with torch.cuda.stream(stream):
                for i in range(6):
                    d = sets[i % 2]
                    fm = gdn.make_featmap_args(d["qkv"][:, :, 0], d["qkv"][:, :, 1], d["w_q"], d["w_k"], d["cos"], d["sin"], 1e-6)
                    ga = gdn.make_gate_args(d["x"], d["w_alpha"], d["b_alpha"], d["a_log"], d["w_beta"], d["b_beta"])
                    p.forward_full(fm, d["qkv"][:, :, 2], ga, None, None, d["gate"], S, z, d["out"], S, z, stream=stream)
                    stream.synchronize()
                    outs.append(d["out"].clone())
                    pp.forward(d["qkv"][:, :, 0], d["qkv"][:, :, 1], d["qkv"][:, :, 2], alpha, beta, S2, d["out"], S2, stream=stream)
                    stream.synchronize()
                    outs.append(d["out"].clone())
            outs += [S.clone(), z.clone(), S2.clone()]
        results[mode] = [o.cpu() for o in outs]
    assert all(torch.isfinite(o.float()).all() for o in results["graph"])
    for a, b in zip(results["direct"], results["graph"]):
        assert torch.equal(a, b)


def test_full_operator_is_bit_repeatable_over_many_calls():
    """The paper's production chunk through gdn_forward_chunk_full, 30 times from the same inputs and state: every
    output, state and z must be bit-identical to the first call's.  The readout CTAs run several tiles each (ring slots,
    staging buffers and the q_raw slot are reused), Phase A reduces in a fixed order, the scans hand their history sum to
    whichever CTA of a pair finishes last: any reuse-before-read or order dependence shows up as a differing bit."""
    B, H, G, F, D = 1, 20, 880, 3, 128
    T = G * F
    wl = gin.GdnWorkload("repeat", B, H, T, D, D, group=G, seed=700)
    fi = gin.make_frontend_inputs(wl)
    d = {n: fi[n].to(DEV) for n in fi}
    out = torch.empty(B, T, H, D, device=DEV, dtype=torch.bfloat16)
    st3 = 3 * H * D
    first = None
    with gdn.GdnPlan(B=B, H=H, T=T, d_k=D, d_v=D, group=G, flags=gdn.GDN_FLAG_NORMALIZER | gdn.GDN_FLAG_BIDIR,
                     q_token_stride=st3, k_token_stride=st3, v_token_stride=st3) as p:
        fm = gdn.make_featmap_args(d["qkv"][:, :, 0], d["qkv"][:, :, 1], d["w_q"], d["w_k"], d["cos"], d["sin"], 1e-6)
        ga = gdn.make_gate_args(d["x"], d["w_alpha"], d["b_alpha"], d["a_log"], d["w_beta"], d["b_beta"])
        for i in range(30):
            S = d["state"].clone()
            z = d["z_in"].clone()
            out.fill_(float("nan"))
            p.forward_full(fm, d["qkv"][:, :, 2], ga, None, None, d["gate"], S, z, out, S, z)
            torch.cuda.synchronize()
            got = (out.clone(), S, z)
            if first is None:
                first = got
                assert torch.isfinite(out.float()).all()
            else:
                for a, b in zip(first, got):
                    assert torch.equal(a, b), f"call {i} differs from call 0"
