"""Test-only fp64 numpy restatements of the GDN recurrence, each structurally DIFFERENT from
oracle/gdn_oracle.c (different loop structure / different algebraic form), used to pin the oracle.

All take one (b,h) stream: q,k [T,dk], v [T,dv], alpha [T/G], beta [T], S0 [dk,dv].
Orientation: S in R^{dk x dv}, o_t = q_t S (Alg. 1 / Eq. 5 of PAPER.md, L118, L369).
"""
import numpy as np


def brute_force_products(q, k, v, alpha, beta, S0, G=1, scale=1.0):
    """Pin 1. Explicit unrolled product formula, no running state:
         S_g = (prod_{r<=g} M_r) S_in + sum_{s<=g} (prod_{s<r<=g} M_r) W_s,
       M_g = alpha_g (I - K_g^T B_g K_g),  W_g = K_g^T B_g V_g   (compact form, Eq. 19).
       Every S_g is rebuilt from scratch from the transition matrices (O(F^2) products)."""
    T, dk = k.shape
    F = T // G
    Ms, Ws = [], []
    for g in range(F):
        Kg, Vg, Bg = k[g * G:(g + 1) * G], v[g * G:(g + 1) * G], np.diag(beta[g * G:(g + 1) * G])
        Ms.append(alpha[g] * (np.eye(dk) - Kg.T @ Bg @ Kg))
        Ws.append(Kg.T @ Bg @ Vg)
    out = np.zeros((T, v.shape[1]))
    S_last = S0.copy()
    for g in range(F):
        P = np.eye(dk)
        for r in range(g + 1):              # prod over r = g, g-1, ..., 0 applied to S_in
            P = P @ Ms[g - r]
        S = P @ S0
        for s in range(g + 1):
            P = np.eye(dk)
            for r in range(g, s, -1):       # prod_{s<r<=g} M_r, later factors on the left
                P = P @ Ms[r]
            S = S + P @ Ws[s]
        out[g * G:(g + 1) * G] = scale * (q[g * G:(g + 1) * G] @ S)
        S_last = S
    return out, S_last


def compact_form(q, k, v, alpha, beta, S0, G=1, scale=1.0):
    """Pin 2a. Eq. 19 (L599) as a running recurrence with dense matrices."""
    T, dk = k.shape
    S = S0.copy()
    out = np.zeros((T, v.shape[1]))
    for g in range(T // G):
        sl = slice(g * G, (g + 1) * G)
        Kg, Vg, Bg = k[sl], v[sl], np.diag(beta[sl])
        S = alpha[g] * (np.eye(dk) - Kg.T @ Bg @ Kg) @ S + Kg.T @ Bg @ Vg
        out[sl] = scale * (q[sl] @ S)
    return out, S


def summaries_scan_readout(q, k, v, alpha, beta, S0, G, scale=1.0):
    """Pin 2b. Eq. 4-5 (L114-L118) / Alg. 1 phases: Phase A summaries for all frames first, then the
    scan, then the readout."""
    T, dk = k.shape
    F = T // G
    P = [np.eye(dk) - k[f * G:(f + 1) * G].T @ (beta[f * G:(f + 1) * G, None] * k[f * G:(f + 1) * G]) for f in range(F)]
    A = [k[f * G:(f + 1) * G].T @ (beta[f * G:(f + 1) * G, None] * v[f * G:(f + 1) * G]) for f in range(F)]
    hist, S = [], S0.copy()
    for f in range(F):
        S = alpha[f] * (P[f] @ S) + A[f]
        hist.append(S)
    out = np.concatenate([scale * (q[f * G:(f + 1) * G] @ hist[f]) for f in range(F)], axis=0)
    return out, S


def chunkwise_wy(q, k, v, alpha, beta, S0, C, scale=1.0):
    """Pin 9. Token-wise (G=1) recurrence in the chunkwise WY/UT form (derived from
    Eq. 17-19 at N=1):  (I+L) U = diag(beta)(V - diag(gamma) K S0),
       L_ij = beta_i e^{Gam_i-Gam_j} k_i.k_j (j<i);  O = diag(gamma) Q S0 + (M o QK^T) U;
       S_C = gamma_C S0 + (diag(gamma_C/gamma) K)^T U.  Any tile size C, ragged tail allowed."""
    T, dk = k.shape
    S = S0.copy()
    out = np.zeros((T, v.shape[1]))
    for c0 in range(0, T, C):
        sl = slice(c0, min(c0 + C, T))
        Q, K, V, b = q[sl], k[sl], v[sl], beta[sl]
        Gam = np.cumsum(np.log(alpha[sl]))
        n = len(Gam)
        D = np.exp(np.minimum(Gam[:, None] - Gam[None, :], 0.0))     # only i>=j entries are used
        L = np.tril(b[:, None] * D * (K @ K.T), -1)
        U = np.linalg.solve(np.eye(n) + L, b[:, None] * (V - np.exp(Gam)[:, None] * (K @ S)))
        M = np.tril(D)                                               # diagonal included (=1)
        out[sl] = scale * (np.exp(Gam)[:, None] * (Q @ S) + (M * (Q @ K.T)) @ U)
        S = np.exp(Gam[-1]) * S + (np.exp(Gam[-1] - Gam)[:, None] * K).T @ U
    return out, S


def affine_chunk_summaries(k, v, alpha, beta, C):
    """State-independent per-chunk affine maps S_{c+1} = (gamma_C I - Kt^T W) S_c + Kt^T Ut
    (SURVEY 8c "affine summary"); returns lists (Mc, Nc). Used to pin the chain form."""
    T, dk = k.shape
    Ms, Ns = [], []
    for c0 in range(0, T, C):
        sl = slice(c0, min(c0 + C, T))
        K, V, b = k[sl], v[sl], beta[sl]
        Gam = np.cumsum(np.log(alpha[sl]))
        n = len(Gam)
        D = np.exp(np.minimum(Gam[:, None] - Gam[None, :], 0.0))
        L = np.tril(b[:, None] * D * (K @ K.T), -1)
        Tm = np.linalg.inv(np.eye(n) + L)
        W = Tm @ ((b * np.exp(Gam))[:, None] * K)
        Ut = Tm @ (b[:, None] * V)
        Kt = np.exp(Gam[-1] - Gam)[:, None] * K
        Ms.append(np.exp(Gam[-1]) * np.eye(dk) - Kt.T @ W)
        Ns.append(Kt.T @ Ut)
    return Ms, Ns


def segment_scan(q, k, v, alpha, beta, S0, C, NS, scale=1.0):
    """Two-level (segment-parallel) scan over the per-chunk affine maps (Eq. 5: S_f = alpha_f P_f S_{f-1}
    + A_f is affine in the state; the columns are independent, L419-L423), as gdn_tc_fused64.cuh runs it:
      per chunk c (state-independent):  G_c = Kt^T W, N_c = Kt^T Ut, gamma_c, Qt_c = diag(gamma) Q - P W, Ol_c = P Ut;
      the chunks are cut into NS segments; segment 0 is scanned from S0; every other segment k from the IDENTITY map:
          Gacc <- gamma_c Gacc + gacc G_c - G_c Gacc,   B <- gamma_c B - G_c B + N_c,   gacc <- gamma_c gacc
      (prefix map of chunk c: S_c = gacc_c S_k - Gacc_c S_k + B_c, recorded BEFORE chunk c is applied);
      level 2: S_{k+1} = gseg_k S_k - Gseg_k S_k + Bseg_k;  outputs: O_c = scale (Qt_c S_c + Ol_c).
    Returns (out, S_final).  Pins the associativity the kernel relies on against the token loop of the oracle."""
    T, dk = k.shape
    dv = v.shape[1]
    chunks = []
    for c0 in range(0, T, C):
        sl = slice(c0, min(c0 + C, T))
        Q, K, V, b = q[sl], k[sl], v[sl], beta[sl]
        Gam = np.cumsum(np.log(alpha[sl]))
        n = len(Gam)
        D = np.exp(np.minimum(Gam[:, None] - Gam[None, :], 0.0))
        L = np.tril(b[:, None] * D * (K @ K.T), -1)
        Tm = np.linalg.inv(np.eye(n) + L)
        W = Tm @ ((b * np.exp(Gam))[:, None] * K)
        Ut = Tm @ (b[:, None] * V)
        Kt = np.exp(Gam[-1] - Gam)[:, None] * K
        P = np.tril(D) * (Q @ K.T)
        chunks.append(dict(sl=sl, G=Kt.T @ W, N=Kt.T @ Ut, gamma=np.exp(Gam[-1]), Qt=np.exp(Gam)[:, None] * Q - P @ W, Ol=P @ Ut))
    NC = len(chunks)
    LSEG = -(-NC // NS)
    segs = [list(range(s, min(s + LSEG, NC))) for s in range(0, NC, LSEG)]
    # level 1: prefix maps of every chunk inside its segment (segment 0 directly on the state)
    pre = [None] * NC
    segmap = []
    S = S0.copy()
    for kseg, idx in enumerate(segs):
        if kseg == 0:
            for c in idx:
                pre[c] = ("state", S.copy())
                S = chunks[c]["gamma"] * S - chunks[c]["G"] @ S + chunks[c]["N"]
            S1 = S
            continue
        Gacc, B, gacc = np.zeros((dk, dk)), np.zeros((dk, dv)), 1.0
        for c in idx:
            pre[c] = ("map", gacc, Gacc.copy(), B.copy())
            g, G, N = chunks[c]["gamma"], chunks[c]["G"], chunks[c]["N"]
            Gacc, B, gacc = g * Gacc + gacc * G - G @ Gacc, g * B - G @ B + N, g * gacc
        segmap.append((gacc, Gacc, B))
    # level 2: the segment maps in order
    S_seg = [None, S1] if len(segs) > 1 else [None]
    Sk = S1 if len(segs) > 1 else S
    for gacc, Gacc, B in segmap:
        Sk = gacc * Sk - Gacc @ Sk + B
        S_seg.append(Sk)
    # parallel fix-up and outputs
    out = np.zeros((T, dv))
    for kseg, idx in enumerate(segs):
        for c in idx:
            if pre[c][0] == "state":
                Sc = pre[c][1]
            else:
                _, gacc, Gacc, B = pre[c]
                Sc = gacc * S_seg[kseg] - Gacc @ S_seg[kseg] + B
            out[chunks[c]["sl"]] = scale * (chunks[c]["Qt"] @ Sc + chunks[c]["Ol"])
    return out, (S_seg[-1] if len(segs) > 1 else S)
