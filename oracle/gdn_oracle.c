/*
 * gdn_oracle.c -- CPU ORACLE for the (frame-wise / token-wise) Gated DeltaNet forward.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and the
 * cpu_baseline / --impl reference legs of bench.py may build, load or call it.  It shares no code,
 * header, table or helper with paper_2605_30409_b200/csrc (the CUDA path) and neither imports the
 * other.  It is plain, slow and meant to be checked against the paper by eye.
 *
 * What it computes (App. G.4-G.5, "Frame-wise delta-rule update" / "Normalized readout",
 * Eq. 17, 18, 20, 22, L587-L624; the streaming cache of App. G.6; Alg. 1 line 9 L338 for
 * "cached state or zero"), in fp64, one (b,h) stream at a time, in the paper's
 * predict-then-correct order:
 *
 *   for each group g of G consecutive tokens (a "frame" of N = G tokens; G = 1 is the token-wise
 *   Gated DeltaNet the paper cites as [35] and that BASELINE.json's configs parametrise):
 *       S~ = alpha_g * S_{g-1}          z~ = alpha_g * z_{g-1}                      (Eq. 17)
 *       r_n = v_n - khat_n S~           e_n = 1 - k_n . z~       for every n in g   (Eq. 18, 20)
 *       S_g = S~ + sum_n khat_n^T (beta_n r_n)                                      (Eq. 18)
 *       z_g = z~ + sum_n k_n (beta_n e_n)                                           (Eq. 20)
 *       num_n = scale * qhat_n S_g      den_n = q_n . z_g                           (Eq. 22)
 *       out_n = num_n                   (default)   or   num_n / (den_n + eps)      (NORMALIZER)
 *
 * Orientation (reading 4): row-token convention of Alg. 1 / Eq. 5 (L118, L369):
 * q,k in R^{T x d_k}, v,out in R^{T x d_v}, state S in R^{d_k x d_v} (the transpose of App. G's
 * S^kv), o_t = q_t S.  All residuals r_n of a group are taken against the SAME decayed state S~
 * (Eq. 18 is one joint rank-N update, Eq. 19: K B K^T is a SUM of N rank-1 terms).
 *
 * Inputs are fp32 arrays (bf16 test inputs are widened to fp32 exactly by the caller) addressed by
 * explicit element strides so that a single (b,h) stream of a big tensor can be run without copies;
 * every arithmetic step is done in double.  The decay is applied by plain multiplication, step by
 * step (no logs, no chunking, no re-association).
 *
 * Parity pins: see tests/test_oracle_pins.py (brute-force product formula, closed forms,
 * hand-worked example in tests/golden/, invariants; for the bidirectional scan at the end of this file:
 * the dense Alg. 1 recursion on explicit P_f, A_f, the F = 1 and F = 2 closed forms, time-reversal symmetry).
 * Nothing in this file is "parity unpinned".
 */
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct {
    int64_t batch, token, head;   /* element strides of a [B,T,H,d] tensor (last dim contiguous) */
} gdn_oracle_strides_t;

/* one (b,h) stream; all pointers already offset to the stream's first token */
static int run_stream(int T, int dk, int dv, int G,
                      const float* q, int64_t q_ts, const float* k, int64_t k_ts,
                      const float* v, int64_t v_ts,
                      const float* q_raw, int64_t qr_ts, const float* k_raw, int64_t kr_ts,
                      const float* alpha /* [T/G] */, const float* beta /* [T] */,
                      const double* S_in /* [dk,dv] or NULL */, const double* z_in /* [dk] or NULL */,
                      double scale, double eps, int normalizer,
                      double* out, int64_t o_ts, double* S_out, double* z_out)
{
    double* S = (double*)calloc((size_t)dk * dv, sizeof(double));
    double* z = (double*)calloc((size_t)dk, sizeof(double));
    double* r = (double*)malloc((size_t)G * dv * sizeof(double));   /* beta_n * r_n, per token of the group */
    double* e = (double*)malloc((size_t)G * sizeof(double));        /* beta_n * e_n */
    if (!S || !z || !r || !e) { free(S); free(z); free(r); free(e); return 1; }
    if (S_in) memcpy(S, S_in, (size_t)dk * dv * sizeof(double));    /* "cached state or zero", L338 */
    if (z_in) memcpy(z, z_in, (size_t)dk * sizeof(double));

    const int n_groups = T / G;
    for (int g = 0; g < n_groups; ++g) {
        const double a = (double)alpha[g];
        /* Eq. 17: decay first */
        for (int i = 0; i < dk * dv; ++i) S[i] *= a;
        if (normalizer) for (int i = 0; i < dk; ++i) z[i] *= a;
        /* Eq. 18 / 20: residuals of every token of the group against the same decayed state */
        for (int n = 0; n < G; ++n) {
            const int t = g * G + n;
            const float* kt = k + (int64_t)t * k_ts;
            const float* vt = v + (int64_t)t * v_ts;
            const double b = (double)beta[t];
            for (int j = 0; j < dv; ++j) {
                double pred = 0.0;                                   /* (khat_n S~)_j */
                for (int i = 0; i < dk; ++i) pred += (double)kt[i] * S[(size_t)i * dv + j];
                r[(size_t)n * dv + j] = b * ((double)vt[j] - pred);
            }
            if (normalizer) {
                const float* krt = k_raw + (int64_t)t * kr_ts;
                double pred = 0.0;                                   /* k_n . z~ */
                for (int i = 0; i < dk; ++i) pred += (double)krt[i] * z[i];
                e[n] = b * (1.0 - pred);
            }
        }
        /* write the corrections: S_g = S~ + sum_n khat_n^T (beta_n r_n) */
        for (int n = 0; n < G; ++n) {
            const int t = g * G + n;
            const float* kt = k + (int64_t)t * k_ts;
            for (int i = 0; i < dk; ++i) {
                const double ki = (double)kt[i];
                for (int j = 0; j < dv; ++j) S[(size_t)i * dv + j] += ki * r[(size_t)n * dv + j];
            }
            if (normalizer) {
                const float* krt = k_raw + (int64_t)t * kr_ts;
                for (int i = 0; i < dk; ++i) z[i] += (double)krt[i] * e[n];
            }
        }
        /* Eq. 22: every token of the group reads the post-update state */
        for (int n = 0; n < G; ++n) {
            const int t = g * G + n;
            const float* qt = q + (int64_t)t * q_ts;
            double* ot = out + (int64_t)t * o_ts;
            double den = 1.0;
            if (normalizer) {
                const float* qrt = q_raw + (int64_t)t * qr_ts;
                double d = 0.0;
                for (int i = 0; i < dk; ++i) d += (double)qrt[i] * z[i];
                den = d + eps;
            }
            for (int j = 0; j < dv; ++j) {
                double num = 0.0;
                for (int i = 0; i < dk; ++i) num += (double)qt[i] * S[(size_t)i * dv + j];
                num *= scale;
                ot[j] = normalizer ? num / den : num;
            }
        }
    }
    if (S_out) memcpy(S_out, S, (size_t)dk * dv * sizeof(double));
    if (z_out && normalizer) memcpy(z_out, z, (size_t)dk * sizeof(double));
    free(S); free(z); free(r); free(e);
    return 0;
}

/*
 * gdn_oracle_forward: all B*H streams.
 *   q,k,v      fp32, [B,T,H,d] addressed by the given strides (last dim contiguous)
 *   q_raw,k_raw  un-rotated copies for the normaliser path (Eq. 20-22); ignored unless normalizer
 *   alpha      fp32 [B,H,T/G]  (the decay itself, in (0,1])
 *   beta       fp32 [B,H,T]
 *   S_in/z_in  fp64 [B,H,dk,dv] / [B,H,dk] or NULL (= zeros)
 *   out        fp64 [B,T,H,dv] contiguous;  S_out fp64 [B,H,dk,dv];  z_out fp64 [B,H,dk]
 * returns 0 on success, 1 on allocation failure, 2 on bad arguments.
 */
int gdn_oracle_forward(int B, int H, int T, int dk, int dv, int G,
                       const float* q, const gdn_oracle_strides_t* qs,
                       const float* k, const gdn_oracle_strides_t* ks,
                       const float* v, const gdn_oracle_strides_t* vs,
                       const float* q_raw, const gdn_oracle_strides_t* qrs,
                       const float* k_raw, const gdn_oracle_strides_t* krs,
                       const float* alpha, const float* beta,
                       const double* S_in, const double* z_in,
                       double scale, double eps, int normalizer,
                       double* out, double* S_out, double* z_out, int nthreads)
{
    if (B < 0 || H < 0 || T < 0 || dk <= 0 || dv <= 0 || G <= 0 || (T % G) != 0) return 2;
    if (normalizer && (!q_raw || !k_raw || !qrs || !krs)) return 2;
    int fail = 0;
    const int n_streams = B * H;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < n_streams; ++s) {
        const int b = s / H, h = s % H;
        const int64_t nG = T / G;
        int rc = run_stream(T, dk, dv, G,
                            q + b * qs->batch + h * qs->head, qs->token,
                            k + b * ks->batch + h * ks->head, ks->token,
                            v + b * vs->batch + h * vs->head, vs->token,
                            normalizer ? q_raw + b * qrs->batch + h * qrs->head : NULL, normalizer ? qrs->token : 0,
                            normalizer ? k_raw + b * krs->batch + h * krs->head : NULL, normalizer ? krs->token : 0,
                            alpha + (int64_t)s * nG, beta + (int64_t)s * T,
                            S_in ? S_in + (int64_t)s * dk * dv : NULL,
                            z_in ? z_in + (int64_t)s * dk : NULL,
                            scale, eps, normalizer,
                            out + ((int64_t)b * T * H + h) * dv, (int64_t)H * dv,
                            S_out ? S_out + (int64_t)s * dk * dv : NULL,
                            z_out ? z_out + (int64_t)s * dk : NULL);
        if (rc) {
#pragma omp atomic write
            fail = 1;
        }
    }
    return fail;
}

/* ------------------------------------------------------------------------------------------------
 * Bidirectional in-chunk scan: PAPER.md Alg. 1 lines 8-22 (L337-L359), "forward scan with previous
 * cache and backward scan within the chunk" (L145), one output pass on the summed histories (L122).
 *
 *   forward : S>_{-1} = cached state or zero;  S>_f = alpha_f P_f S>_{f-1} + A_f,  f = 0..F-1      (l. 9-12)
 *   reverse : S<_{F-1} = 0;  for f = F-1 down to 1:  S<_{f-1} = alpha_f P_f S<_f + A_f             (l. 14-17)
 *   S^hist_f = S>_f + S<_f  (same for z);  N = Q_rot S^hist_f,  d = Q z^hist_f,  O = N / (d + eps) (l. 19-29)
 *
 * "alpha_f P_f X + A_f" is applied here in the predict-then-correct form of Eq. 17-18 (decay, residuals of
 * every token of frame f against the same decayed state, joint write), i.e. the very update of run_stream,
 * so that nothing is re-associated.  S_out / z_out are the FORWARD terminal states S>_{F-1}, z>_{F-1} (the cache
 * handed to the next chunk, L72 / App. G.6).  Without the normaliser O = scale * N.
 * ------------------------------------------------------------------------------------------------ */
/* X <- alpha_f P_f X + A_f  and  y <- alpha_f P^z_f y + b_f  with the tokens of frame f (Eq. 17, 18, 20) */
static void frame_update(int f, int G, int dk, int dv,
                         const float* k, int64_t k_ts, const float* v, int64_t v_ts, const float* k_raw, int64_t kr_ts,
                         const float* alpha, const float* beta, int normalizer,
                         double* X, double* y, double* r, double* e)
{
    const double a = (double)alpha[f];
    for (int i = 0; i < dk * dv; ++i) X[i] *= a;
    if (normalizer) for (int i = 0; i < dk; ++i) y[i] *= a;
    for (int n = 0; n < G; ++n) {
        const int t = f * G + n;
        const float* kt = k + (int64_t)t * k_ts;
        const float* vt = v + (int64_t)t * v_ts;
        const double b = (double)beta[t];
        for (int j = 0; j < dv; ++j) {
            double pred = 0.0;
            for (int i = 0; i < dk; ++i) pred += (double)kt[i] * X[(size_t)i * dv + j];
            r[(size_t)n * dv + j] = b * ((double)vt[j] - pred);
        }
        if (normalizer) {
            const float* krt = k_raw + (int64_t)t * kr_ts;
            double pred = 0.0;
            for (int i = 0; i < dk; ++i) pred += (double)krt[i] * y[i];
            e[n] = b * (1.0 - pred);
        }
    }
    for (int n = 0; n < G; ++n) {
        const int t = f * G + n;
        const float* kt = k + (int64_t)t * k_ts;
        for (int i = 0; i < dk; ++i) {
            const double ki = (double)kt[i];
            for (int j = 0; j < dv; ++j) X[(size_t)i * dv + j] += ki * r[(size_t)n * dv + j];
        }
        if (normalizer) {
            const float* krt = k_raw + (int64_t)t * kr_ts;
            for (int i = 0; i < dk; ++i) y[i] += (double)krt[i] * e[n];
        }
    }
}

static int run_stream_bidir(int T, int dk, int dv, int G,
                            const float* q, int64_t q_ts, const float* k, int64_t k_ts, const float* v, int64_t v_ts,
                            const float* q_raw, int64_t qr_ts, const float* k_raw, int64_t kr_ts,
                            const float* alpha, const float* beta, const double* S_in, const double* z_in,
                            double scale, double eps, int normalizer,
                            double* out, int64_t o_ts, double* S_out, double* z_out)
{
    const int F = T / G;
    const size_t ns = (size_t)dk * dv;
    double* Sf = (double*)calloc((size_t)(F + 1) * ns, sizeof(double));      /* Sf[f] = S>_f (slot F: work copy) */
    double* Sr = (double*)calloc((size_t)(F + 1) * ns, sizeof(double));      /* Sr[f] = S<_f */
    double* zf = (double*)calloc((size_t)(F + 1) * dk, sizeof(double));
    double* zr = (double*)calloc((size_t)(F + 1) * dk, sizeof(double));
    double* r = (double*)malloc((size_t)G * dv * sizeof(double));
    double* e = (double*)malloc((size_t)G * sizeof(double));
    if (!Sf || !Sr || !zf || !zr || !r || !e) { free(Sf); free(Sr); free(zf); free(zr); free(r); free(e); return 1; }
    double* X = Sf + (size_t)F * ns;
    double* y = zf + (size_t)F * dk;
    /* forward scan, lines 9-12 */
    if (S_in) memcpy(X, S_in, ns * sizeof(double));
    if (z_in) memcpy(y, z_in, (size_t)dk * sizeof(double));
    for (int f = 0; f < F; ++f) {
        frame_update(f, G, dk, dv, k, k_ts, v, v_ts, k_raw, kr_ts, alpha, beta, normalizer, X, y, r, e);
        memcpy(Sf + (size_t)f * ns, X, ns * sizeof(double));
        memcpy(zf + (size_t)f * dk, y, (size_t)dk * sizeof(double));
    }
    if (S_out && F > 0) memcpy(S_out, Sf + (size_t)(F - 1) * ns, ns * sizeof(double));
    if (S_out && F == 0) { if (S_in) memcpy(S_out, S_in, ns * sizeof(double)); else memset(S_out, 0, ns * sizeof(double)); }
    if (z_out && normalizer && F > 0) memcpy(z_out, zf + (size_t)(F - 1) * dk, (size_t)dk * sizeof(double));
    /* reverse scan, lines 14-17: S<_{F-1} = 0 (calloc), then f = F-1 down to 1 */
    X = Sr + (size_t)F * ns;
    y = zr + (size_t)F * dk;
    memset(X, 0, ns * sizeof(double));
    memset(y, 0, (size_t)dk * sizeof(double));
    for (int f = F - 1; f >= 1; --f) {
        frame_update(f, G, dk, dv, k, k_ts, v, v_ts, k_raw, kr_ts, alpha, beta, normalizer, X, y, r, e);
        memcpy(Sr + (size_t)(f - 1) * ns, X, ns * sizeof(double));
        memcpy(zr + (size_t)(f - 1) * dk, y, (size_t)dk * sizeof(double));
    }
    /* lines 19-29: one output pass on S^hist_f = S>_f + S<_f */
    for (int f = 0; f < F; ++f) {
        const double* A = Sf + (size_t)f * ns; const double* Bv = Sr + (size_t)f * ns;
        const double* za = zf + (size_t)f * dk; const double* zb = zr + (size_t)f * dk;
        for (int n = 0; n < G; ++n) {
            const int t = f * G + n;
            const float* qt = q + (int64_t)t * q_ts;
            double* ot = out + (int64_t)t * o_ts;
            double den = 1.0;
            if (normalizer) {
                const float* qrt = q_raw + (int64_t)t * qr_ts;
                double d = 0.0;
                for (int i = 0; i < dk; ++i) d += (double)qrt[i] * (za[i] + zb[i]);
                den = d + eps;
            }
            for (int j = 0; j < dv; ++j) {
                double num = 0.0;
                for (int i = 0; i < dk; ++i) num += (double)qt[i] * (A[(size_t)i * dv + j] + Bv[(size_t)i * dv + j]);
                num *= scale;
                ot[j] = normalizer ? num / den : num;
            }
        }
    }
    free(Sf); free(Sr); free(zf); free(zr); free(r); free(e);
    return 0;
}

/* gdn_oracle_forward_bidir: arguments as gdn_oracle_forward; G = tokens per frame, F = T / G frames per call. */
int gdn_oracle_forward_bidir(int B, int H, int T, int dk, int dv, int G,
                             const float* q, const gdn_oracle_strides_t* qs,
                             const float* k, const gdn_oracle_strides_t* ks,
                             const float* v, const gdn_oracle_strides_t* vs,
                             const float* q_raw, const gdn_oracle_strides_t* qrs,
                             const float* k_raw, const gdn_oracle_strides_t* krs,
                             const float* alpha, const float* beta,
                             const double* S_in, const double* z_in,
                             double scale, double eps, int normalizer,
                             double* out, double* S_out, double* z_out, int nthreads)
{
    if (B < 0 || H < 0 || T < 0 || dk <= 0 || dv <= 0 || G <= 0 || (T % G) != 0) return 2;
    if (normalizer && (!q_raw || !k_raw || !qrs || !krs)) return 2;
    int fail = 0;
    const int n_streams = B * H;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#else
    (void)nthreads;
#endif
#pragma omp parallel for schedule(dynamic, 1)
    for (int s = 0; s < n_streams; ++s) {
        const int b = s / H, h = s % H;
        const int64_t nG = T / G;
        int rc = run_stream_bidir(T, dk, dv, G,
                                  q + b * qs->batch + h * qs->head, qs->token,
                                  k + b * ks->batch + h * ks->head, ks->token,
                                  v + b * vs->batch + h * vs->head, vs->token,
                                  normalizer ? q_raw + b * qrs->batch + h * qrs->head : NULL, normalizer ? qrs->token : 0,
                                  normalizer ? k_raw + b * krs->batch + h * krs->head : NULL, normalizer ? krs->token : 0,
                                  alpha + (int64_t)s * nG, beta + (int64_t)s * T,
                                  S_in ? S_in + (int64_t)s * dk * dv : NULL,
                                  z_in ? z_in + (int64_t)s * dk : NULL,
                                  scale, eps, normalizer,
                                  out + ((int64_t)b * T * H + h) * dv, (int64_t)H * dv,
                                  S_out ? S_out + (int64_t)s * dk * dv : NULL,
                                  z_out ? z_out + (int64_t)s * dk : NULL);
        if (rc) {
#pragma omp atomic write
            fail = 1;
        }
    }
    return fail;
}

int gdn_oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
