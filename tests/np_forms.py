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
