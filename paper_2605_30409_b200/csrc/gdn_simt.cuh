// gdn_simt.cuh -- fp32 CUDA-core GDN forward for any update granularity G (both modes).
//
// This is the library's "fp32-input mode" (north_star: <= 1e-4 vs the oracle; single-pass TF32 MMAs
// miss that bound, reading 19) and the generic path for shapes the tensor-core kernels do
// not take.  It evaluates PAPER.md Eq. 17-18, 20, 22 (L587-L624) in the paper's own order:
//   S~ = alpha_g S;  u_n = beta_n (v_n - k_n S~) for all n of the group against the same S~;
//   S = S~ + sum_n k_n^T u_n;  o_n = scale q_n S.
//
// Mapping: ONE WARP per (b, h, 8-column tile of d_v).  The 32 lanes split d_k (lane l owns rows
// l, l+32, ...), so the state tile S[d_k x 8] lives in DK/32*8 registers per lane, k/q rows are read
// with one coalesced 128-byte request per 32 features, and the two dot products per token are warp
// shuffles -- no shared memory, no block barrier on the serial chain.  The (independent, PAPER.md
// L419-L423) d_v column tiles of one head sit in the same block so their k/q reads hit L1.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gdn {

struct SimtParams {
    const void* q; const void* k; const void* v;         // [B,T,H,d]
    const void* q_raw; const void* k_raw;                // normaliser path (un-rotated), or nullptr
    const float* alpha; const float* beta;               // [B,H,T/G], [B,H,T]
    const float* S_in; const float* z_in;                // [B,H,dk,dv], [B,H,dk] or nullptr
    void* out; float* S_out; float* z_out;
    int B, H, T, G, dv;
    long long q_ts, k_ts, v_ts, o_ts;                    // token strides (elements)
    float scale, eps;
    int log_alpha, normalizer;
};

__device__ __forceinline__ float ld_in(const float* p) { return __ldg(p); }
__device__ __forceinline__ float ld_in(const __nv_bfloat16* p) { return __bfloat162float(*p); }
__device__ __forceinline__ void st_out(float* p, float x) { *p = x; }
__device__ __forceinline__ void st_out(__nv_bfloat16* p, float x) { *p = __float2bfloat16_rn(x); }

__device__ __forceinline__ float warp_sum(float x) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) x += __shfl_xor_sync(0xffffffffu, x, o);
    return x;
}

constexpr int kSimtCols = 8;        // d_v columns per warp
constexpr int kSimtWarps = 4;       // warps (= column tiles) per block

template <int DK, typename TIn>
__global__ void __launch_bounds__(kSimtWarps * 32)
gdn_simt_kernel(const SimtParams p) {
    constexpr int R = DK / 32;
    const int lane = threadIdx.x & 31;
    const int tiles = p.dv / kSimtCols;
    const int wglobal = blockIdx.x * kSimtWarps + (threadIdx.x >> 5);
    if (wglobal >= p.B * p.H * tiles) return;
    const int tile = wglobal % tiles;
    const int bh = wglobal / tiles;
    const int b = bh / p.H, h = bh % p.H;
    const int c0 = tile * kSimtCols;
    const int dv = p.dv;

    const TIn* q = reinterpret_cast<const TIn*>(p.q) + (long long)b * p.T * p.q_ts + (long long)h * DK;
    const TIn* k = reinterpret_cast<const TIn*>(p.k) + (long long)b * p.T * p.k_ts + (long long)h * DK;
    const TIn* v = reinterpret_cast<const TIn*>(p.v) + (long long)b * p.T * p.v_ts + (long long)h * dv + c0;
    TIn* out = reinterpret_cast<TIn*>(p.out) + (long long)b * p.T * p.o_ts + (long long)h * dv + c0;
    const TIn* qr = p.normalizer ? reinterpret_cast<const TIn*>(p.q_raw) + (long long)b * p.T * p.q_ts + (long long)h * DK : nullptr;
    const TIn* kr = p.normalizer ? reinterpret_cast<const TIn*>(p.k_raw) + (long long)b * p.T * p.k_ts + (long long)h * DK : nullptr;
    const int nG = p.T / p.G;
    const float* alpha = p.alpha + (long long)bh * nG;
    const float* beta = p.beta + (long long)bh * p.T;

    float S[R][kSimtCols], dS[R][kSimtCols], z[R], dz[R];
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int row = lane + 32 * r;
#pragma unroll
        for (int c = 0; c < kSimtCols; ++c)
            S[r][c] = p.S_in ? p.S_in[((long long)bh * DK + row) * dv + c0 + c] : 0.f;
        z[r] = (p.normalizer && p.z_in) ? p.z_in[(long long)bh * DK + row] : 0.f;
    }

    if (p.G == 1) {
        // token-wise (G = 1): decay, correct, write and read per token; 4 tokens of loads in flight
        for (int t0 = 0; t0 < p.T; t0 += 4) {
            float kk[4][R], qq[4][R], vv[4][kSimtCols], bb[4], aa[4], kkr[4][R], qqr[4][R];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int t = t0 + i;
                const bool ok = t < p.T;
                bb[i] = ok ? beta[t] : 0.f;
                aa[i] = ok ? alpha[t] : 1.f;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    kk[i][r] = ok ? ld_in(k + (long long)t * p.k_ts + lane + 32 * r) : 0.f;
                    qq[i][r] = ok ? ld_in(q + (long long)t * p.q_ts + lane + 32 * r) : 0.f;
                    kkr[i][r] = (ok && p.normalizer) ? ld_in(kr + (long long)t * p.k_ts + lane + 32 * r) : 0.f;
                    qqr[i][r] = (ok && p.normalizer) ? ld_in(qr + (long long)t * p.q_ts + lane + 32 * r) : 0.f;
                }
#pragma unroll
                for (int c = 0; c < kSimtCols; ++c) vv[i][c] = ok ? ld_in(v + (long long)t * p.v_ts + c) : 0.f;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int t = t0 + i;
                if (t >= p.T) break;
                const float a = p.log_alpha ? expf(aa[i]) : aa[i];
                float mine = 0.f;
#pragma unroll
                for (int c = 0; c < kSimtCols; ++c) {
                    float pred = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) { S[r][c] *= a; pred = fmaf(kk[i][r], S[r][c], pred); }
                    pred = warp_sum(pred);
                    const float u = bb[i] * (vv[i][c] - pred);
                    float o = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) { S[r][c] = fmaf(kk[i][r], u, S[r][c]); o = fmaf(qq[i][r], S[r][c], o); }
                    o = warp_sum(o);
                    if (lane == c) mine = o;
                }
                float inv_den = 1.f;
                if (p.normalizer) {
                    float pred = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) { z[r] *= a; pred = fmaf(kkr[i][r], z[r], pred); }
                    pred = warp_sum(pred);
                    const float e = bb[i] * (1.f - pred);
                    float d = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) { z[r] = fmaf(kkr[i][r], e, z[r]); d = fmaf(qqr[i][r], z[r], d); }
                    d = warp_sum(d);
                    inv_den = 1.f / (d + p.eps);
                }
                if (lane < kSimtCols) st_out(out + (long long)t * p.o_ts + lane, p.scale * mine * inv_den);
            }
        }
    } else
    for (int g = 0; g < nG; ++g) {
        float a = alpha[g];
        if (p.log_alpha) a = expf(a);
        // Eq. 17: decay first
#pragma unroll
        for (int r = 0; r < R; ++r) {
#pragma unroll
            for (int c = 0; c < kSimtCols; ++c) { S[r][c] *= a; dS[r][c] = 0.f; }
            z[r] *= a; dz[r] = 0.f;
        }
        // Eq. 18 / 20: corrections of every token of the group against the same decayed state
        const int t0 = g * p.G;
        for (int n0 = 0; n0 < p.G; n0 += 4) {
            float kk[4][R], vv[4][kSimtCols], bb[4], kkr[4][R];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int t = t0 + n0 + i;
                const bool ok = (n0 + i) < p.G;
                bb[i] = ok ? beta[t] : 0.f;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    kk[i][r] = ok ? ld_in(k + (long long)t * p.k_ts + lane + 32 * r) : 0.f;
                    kkr[i][r] = (ok && p.normalizer) ? ld_in(kr + (long long)t * p.k_ts + lane + 32 * r) : 0.f;
                }
#pragma unroll
                for (int c = 0; c < kSimtCols; ++c) vv[i][c] = ok ? ld_in(v + (long long)t * p.v_ts + c) : 0.f;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (n0 + i >= p.G) break;
                float u[kSimtCols];
#pragma unroll
                for (int c = 0; c < kSimtCols; ++c) {
                    float pred = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) pred = fmaf(kk[i][r], S[r][c], pred);
                    pred = warp_sum(pred);
                    u[c] = bb[i] * (vv[i][c] - pred);
                }
#pragma unroll
                for (int r = 0; r < R; ++r)
#pragma unroll
                    for (int c = 0; c < kSimtCols; ++c) dS[r][c] = fmaf(kk[i][r], u[c], dS[r][c]);
                if (p.normalizer) {
                    float pred = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) pred = fmaf(kkr[i][r], z[r], pred);
                    pred = warp_sum(pred);
                    const float e = bb[i] * (1.f - pred);
#pragma unroll
                    for (int r = 0; r < R; ++r) dz[r] = fmaf(kkr[i][r], e, dz[r]);
                }
            }
        }
#pragma unroll
        for (int r = 0; r < R; ++r) {
#pragma unroll
            for (int c = 0; c < kSimtCols; ++c) S[r][c] += dS[r][c];
            z[r] += dz[r];
        }
        // Eq. 22: every token of the group reads the post-update state
        for (int n0 = 0; n0 < p.G; n0 += 4) {
            float qq[4][R], qqr[4][R];
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                const int t = t0 + n0 + i;
                const bool ok = (n0 + i) < p.G;
#pragma unroll
                for (int r = 0; r < R; ++r) {
                    qq[i][r] = ok ? ld_in(q + (long long)t * p.q_ts + lane + 32 * r) : 0.f;
                    qqr[i][r] = (ok && p.normalizer) ? ld_in(qr + (long long)t * p.q_ts + lane + 32 * r) : 0.f;
                }
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                if (n0 + i >= p.G) break;
                const int t = t0 + n0 + i;
                float inv_den = 1.f;
                if (p.normalizer) {
                    float d = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) d = fmaf(qqr[i][r], z[r], d);
                    d = warp_sum(d);
                    inv_den = 1.f / (d + p.eps);
                }
                float mine = 0.f;
#pragma unroll
                for (int c = 0; c < kSimtCols; ++c) {
                    float o = 0.f;
#pragma unroll
                    for (int r = 0; r < R; ++r) o = fmaf(qq[i][r], S[r][c], o);
                    o = warp_sum(o);
                    if (lane == c) mine = o;
                }
                if (lane < kSimtCols) st_out(out + (long long)t * p.o_ts + lane, p.scale * mine * inv_den);
            }
        }
    }
#pragma unroll
    for (int r = 0; r < R; ++r) {
        const int row = lane + 32 * r;
#pragma unroll
        for (int c = 0; c < kSimtCols; ++c) p.S_out[((long long)bh * DK + row) * dv + c0 + c] = S[r][c];
        if (p.normalizer && tile == 0 && p.z_out) p.z_out[(long long)bh * DK + row] = z[r];
    }
}

}  // namespace gdn
