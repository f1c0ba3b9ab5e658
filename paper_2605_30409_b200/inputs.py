"""Seeded synthetic inputs for the GDN forward -- shared by the CUDA path's callers and by the oracle's.

This module holds NONE of the method's arithmetic (no recurrence, no decay products, no readout): it
only draws random tensors with the shapes and value distributions BASELINE.json's five configs name
and the layout the C ABI fixes (include/gdn.h).  The paper's real workload is latent video pushed
through trained projections (Eq. 11-15); neither weights nor videos exist here,
so these tensors STAND IN for it.

Recipe (fixed draw order q, k, v, a_raw, b_raw, state from one CPU ``torch.Generator``):
  q, k   randn -> L2-normalised per token and head in fp32 -> (mode F: k *= 1/sqrt(G)) -> cast
  v      randn -> cast
  alpha  sigmoid(mu_a + sd_a * a_raw), fp32, one per token (G=1) or one per frame (G>1)
  beta   sigmoid(mu_b + sd_b * b_raw), fp32, one per token
  state  state_std * randn, fp32, [B,H,d_k,d_v]  (None when state_std == 0)
The 1/sqrt(G) key scale of mode F is the stand-in for the paper's 1/sqrt(DN) rescale (L554) that keeps
the frame-wise update a contraction.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field
from typing import Optional

import torch


@dataclass
class GdnWorkload:
    """Shape + distribution of one call (one streaming chunk)."""
    name: str
    B: int
    H: int
    T: int
    d_k: int
    d_v: int
    dtype: torch.dtype = torch.bfloat16
    group: int = 1                 # G: 1 = token-wise, N_frame = frame-wise (paper)
    chunk: int = 0                 # mode-T compute tile (0 = library default)
    alpha_mu: float = 3.0
    alpha_sd: float = 1.0
    beta_mu: float = 0.0
    beta_sd: float = 1.0
    state_std: float = 0.02
    seed: int = 0

    def with_(self, **kw) -> "GdnWorkload":
        d = dict(self.__dict__)
        d.update(kw)
        return GdnWorkload(**d)


@dataclass
class GdnInputs:
    wl: GdnWorkload
    q: torch.Tensor
    k: torch.Tensor
    v: torch.Tensor
    alpha: torch.Tensor            # [B,H,T/G] fp32
    beta: torch.Tensor             # [B,H,T]   fp32
    state: Optional[torch.Tensor]  # [B,H,d_k,d_v] fp32 or None
    extras: dict = field(default_factory=dict)


def make_inputs(wl: GdnWorkload, seed: Optional[int] = None, with_state: bool = True) -> GdnInputs:
    g = torch.Generator(device="cpu")
    g.manual_seed(int(wl.seed if seed is None else seed))
    B, H, T, dk, dv, G = wl.B, wl.H, wl.T, wl.d_k, wl.d_v, wl.group
    assert T % G == 0
    q = torch.randn(B, T, H, dk, generator=g, dtype=torch.float32)
    k = torch.randn(B, T, H, dk, generator=g, dtype=torch.float32)
    v = torch.randn(B, T, H, dv, generator=g, dtype=torch.float32)
    a_raw = torch.randn(B, H, T // G, generator=g, dtype=torch.float32)
    b_raw = torch.randn(B, H, T, generator=g, dtype=torch.float32)
    st = torch.randn(B, H, dk, dv, generator=g, dtype=torch.float32)
    q = torch.nn.functional.normalize(q, dim=-1)
    k = torch.nn.functional.normalize(k, dim=-1)
    if G > 1:
        k = k * (1.0 / math.sqrt(G))
    alpha = torch.sigmoid(wl.alpha_mu + wl.alpha_sd * a_raw)
    beta = torch.sigmoid(wl.beta_mu + wl.beta_sd * b_raw)
    state = (wl.state_std * st) if (with_state and wl.state_std > 0) else None
    return GdnInputs(wl, q.to(wl.dtype).contiguous(), k.to(wl.dtype).contiguous(),
                     v.to(wl.dtype).contiguous(), alpha.contiguous(), beta.contiguous(), state)


def make_normalizer_inputs(wl: GdnWorkload, seed: Optional[int] = None) -> GdnInputs:
    """Inputs shaped like the paper's features for the normalised readout (Eq. 12, 20-22):
    q_raw,k_raw = ReLU(RMS-normalised randn) (non-negative), k_raw *= 1/sqrt(d*G), rotated copies by
    a seeded per-token pairwise rotation (a stand-in for the fixed 3D RoPE), z_in >= 0."""
    g = torch.Generator(device="cpu")
    g.manual_seed(int(wl.seed if seed is None else seed))
    B, H, T, dk, dv, G = wl.B, wl.H, wl.T, wl.d_k, wl.d_v, wl.group

    def feat():
        x = torch.randn(B, T, H, dk, generator=g, dtype=torch.float32)
        x = x * torch.rsqrt(x.pow(2).mean(-1, keepdim=True) + 1e-6)
        return torch.relu(x)

    q_raw = feat()
    k_raw = feat() * (1.0 / math.sqrt(dk * G))
    v = torch.randn(B, T, H, dv, generator=g, dtype=torch.float32)
    a_raw = torch.randn(B, H, T // G, generator=g, dtype=torch.float32)
    b_raw = torch.randn(B, H, T, generator=g, dtype=torch.float32)
    st = torch.randn(B, H, dk, dv, generator=g, dtype=torch.float32)
    zt = torch.rand(B, H, dk, generator=g, dtype=torch.float32)
    theta = torch.rand(B, T, 1, dk // 2, generator=g, dtype=torch.float32) * (2 * math.pi)

    def rot(x):
        x1, x2 = x[..., 0::2], x[..., 1::2]
        c, s = torch.cos(theta), torch.sin(theta)
        y = torch.empty_like(x)
        y[..., 0::2] = x1 * c - x2 * s
        y[..., 1::2] = x1 * s + x2 * c
        return y

    alpha = torch.sigmoid(wl.alpha_mu + wl.alpha_sd * a_raw)
    beta = torch.sigmoid(wl.beta_mu + wl.beta_sd * b_raw)
    dt = wl.dtype
    inp = GdnInputs(wl, rot(q_raw).to(dt).contiguous(), rot(k_raw).to(dt).contiguous(),
                    v.to(dt).contiguous(), alpha.contiguous(), beta.contiguous(), wl.state_std * st)
    inp.extras = {"q_raw": q_raw.to(dt).contiguous(), "k_raw": k_raw.to(dt).contiguous(),
                  "z_in": (wl.state_std * zt).contiguous()}
    return inp


def make_frontend_inputs(wl: GdnWorkload, seed: Optional[int] = None, grid_w: int = 40) -> dict:
    """Seeded operands of the block's front end (App. G.2-G.3, Alg. 1): a packed qkv tensor
    [B,T,3,H,D] of raw projections, the per-head latent features x [B,T,H,D], RMSNorm weights, rotation tables
    for a (frame, row, column) position with three frequency bands, gate parameters, an evaluated output gate.
    Only random draws and table look-ups: none of the method's arithmetic."""
    g = torch.Generator(device="cpu")
    g.manual_seed(int(wl.seed if seed is None else seed))
    B, H, T, D, G = wl.B, wl.H, wl.T, wl.d_k, wl.group
    dt = wl.dtype
    qkv = torch.randn(B, T, 3, H, D, generator=g, dtype=torch.float32).to(dt).contiguous()
    x = torch.randn(B, T, H, D, generator=g, dtype=torch.float32).to(dt).contiguous()
    w_q = 0.5 + torch.rand(H, D, generator=g, dtype=torch.float32)
    w_k = 0.5 + torch.rand(H, D, generator=g, dtype=torch.float32)
    # position of token t: frame t // G, row (t % G) // grid_w, column (t % G) % grid_w; pair i belongs to one of three bands
    t = torch.arange(T)
    pos = torch.stack([t // G, (t % G) // grid_w, (t % G) % grid_w], dim=1).to(torch.float32)        # [T, 3]
    npair = D // 2
    band = torch.arange(npair) % 3
    freq = 1.0 / (10000.0 ** (torch.arange(npair, dtype=torch.float32) / npair))
    ang = pos[:, band] * freq[None, :]
    out = {
        "qkv": qkv, "x": x, "w_q": w_q.contiguous(), "w_k": w_k.contiguous(),
        "cos": torch.cos(ang).contiguous(), "sin": torch.sin(ang).contiguous(),
        "w_alpha": (torch.randn(H, D, generator=g) / math.sqrt(D)).contiguous(),
        "b_alpha": torch.randn(H, generator=g).contiguous() - 2.0,
        "a_log": (0.5 * torch.randn(H, generator=g)).contiguous(),
        "w_beta": (torch.randn(H, D, generator=g) / math.sqrt(D)).contiguous(),
        "b_beta": torch.randn(H, generator=g).contiguous(),
        "gate": torch.nn.functional.silu(torch.randn(B, T, H, D, generator=g, dtype=torch.float32)).to(dt).contiguous(),
        "state": (wl.state_std * torch.randn(B, H, D, D, generator=g, dtype=torch.float32)).contiguous(),
        "z_in": (wl.state_std * torch.rand(B, H, D, generator=g, dtype=torch.float32)).contiguous(),
    }
    return out


# --- BASELINE.json's five configs (mode T = literal; *_F = the paper's frame-wise semantics) -------
def config(idx: int, *, T: Optional[int] = None, chunk: int = 0, frame: bool = False,
           chunk_index: int = 0) -> GdnWorkload:
    """Workload ``idx`` (1..5) of BASELINE.json. seed = 1000*idx + chunk_index (config 1: seed 0)."""
    if idx == 1:
        wl = GdnWorkload("cfg1", 1, 2, 256, 32, 32, dtype=torch.float32, state_std=0.0, seed=0,
                         chunk=chunk or 64)
        G = 64
    elif idx == 2:
        wl = GdnWorkload("cfg2", 1, 16, 3520, 64, 64, seed=2000, chunk=chunk)
        G = 3520
    elif idx in (3, 4):
        wl = GdnWorkload(f"cfg{idx}", 1, 20, 10560, 128, 128, seed=1000 * idx + chunk_index, chunk=chunk)
        G = 3520
    elif idx == 5:
        t = T or 3520
        wl = GdnWorkload(f"cfg5_T{t}", 2, 32, t, 128, 128, alpha_mu=1.0, alpha_sd=2.0, beta_mu=1.0,
                         beta_sd=1.0, seed=5000 + (t % 997), chunk=chunk)
        G = 4096 if t == 65536 else 3520
    else:
        raise ValueError(idx)
    if frame:
        wl = wl.with_(group=G, name=wl.name + "_F")
    return wl


def paper_shape(frames: int = 3, d: int = 128) -> GdnWorkload:
    """The paper's production chunk: 22x40 = 880 tokens per frame, 20 heads, d padded to 128
    (PAPER.md L270, L316, L385); first chunk has 5 frames, later ones 3 (L460)."""
    return GdnWorkload(f"paper_{frames}x880" + ("" if d == 128 else f"_d{d}"), 1, 20, frames * 880, d, d, group=880, seed=7000 + frames)
