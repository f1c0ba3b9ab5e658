"""Helpers for the -m gpu parity tests: run the CUDA path through the C ABI, run the oracle, compare."""
from __future__ import annotations

import numpy as np
import torch

import oracle
import paper_2605_30409_b200 as gdn
from paper_2605_30409_b200 import inputs as gin

TOL_BF16 = 2e-2     # north_star: max abs error <= 2e-2 * max|o| for bf16 inputs with fp32 state
TOL_FP32 = 1e-4     # north_star: <= 1e-4 in the fp32-input mode


def io_dtype(t: torch.dtype) -> int:
    return gdn.GDN_FP32 if t == torch.float32 else gdn.GDN_BF16


def run_cuda(inp: gin.GdnInputs, state_in="default", flags=0, chunk=None, scale=1.0, plan=None):
    """-> (out [B,T,H,dv] torch on cpu, S_out [B,H,dk,dv] fp32 cpu, plan info)."""
    wl = inp.wl
    dev = torch.device("cuda:0")
    q, k, v = inp.q.to(dev), inp.k.to(dev), inp.v.to(dev)
    alpha, beta = inp.alpha.to(dev), inp.beta.to(dev)
    st = inp.state if isinstance(state_in, str) else state_in
    st_d = st.to(dev).contiguous() if st is not None else None
    out = torch.empty(wl.B, wl.T, wl.H, wl.d_v, dtype=wl.dtype, device=dev)
    S_out = torch.full((wl.B, wl.H, wl.d_k, wl.d_v), float("nan"), dtype=torch.float32, device=dev)
    own = plan is None
    if own:
        plan = gdn.GdnPlan(B=wl.B, H=wl.H, T=wl.T, d_k=wl.d_k, d_v=wl.d_v, group=wl.group,
                           chunk=wl.chunk if chunk is None else chunk, io_dtype=io_dtype(wl.dtype),
                           scale=scale, flags=flags)
    info = plan.info
    plan.forward(q, k, v, alpha, beta, st_d, out, S_out)
    torch.cuda.synchronize()
    res = out.cpu(), S_out.cpu(), (info.path, info.chunk, info.launches_per_call)
    if own:
        plan.close()
    return res


def run_oracle(inp: gin.GdnInputs, state_in="default", scale=1.0, heads=None):
    """Oracle on the same seeded arrays (bf16 widened exactly). `heads`: optional list of (b,h)
    streams to sample -> dict {(b,h): (out [T,dv], S [dk,dv])} instead of full tensors."""
    wl = inp.wl
    st = inp.state if isinstance(state_in, str) else state_in
    if heads is None:
        return oracle.gdn_forward(inp.q, inp.k, inp.v, inp.alpha, inp.beta, st, group=wl.group, scale=scale)
    res = {}
    for (b, h) in heads:
        o, s = oracle.gdn_forward(inp.q[b:b + 1, :, h:h + 1], inp.k[b:b + 1, :, h:h + 1], inp.v[b:b + 1, :, h:h + 1],
                                  inp.alpha[b:b + 1, h:h + 1], inp.beta[b:b + 1, h:h + 1],
                                  None if st is None else st[b:b + 1, h:h + 1], group=wl.group, scale=scale)
        res[(b, h)] = (o[0, :, 0], s[0, 0])
    return res


def rel_err(x, ref) -> float:
    """max|x - ref| / max|ref| (the north_star error metric)."""
    x = np.asarray(x.double().numpy() if hasattr(x, "numpy") else x, dtype=np.float64)
    ref = np.asarray(ref, dtype=np.float64)
    if not np.isfinite(x).all():
        return float("inf")
    denom = np.abs(ref).max()
    return float(np.abs(x - ref).max() / (denom if denom > 0 else 1.0))


def tol_for(dtype) -> float:
    return TOL_FP32 if dtype == torch.float32 else TOL_BF16
