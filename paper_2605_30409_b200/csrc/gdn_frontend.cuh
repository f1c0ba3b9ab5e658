// gdn_frontend.cuh -- the front end of the GDN block around the recurrence (App. G.2, G.3; Alg. 1 "Require:
// qkv, beta, decay alpha, normalization weights, RoPE tables", L325): both are HBM-bound element-wise / reduction passes
// (no contraction worth a tensor core), written for coalesced 16-byte accesses.
//
//   featmap_body         Eq. 12 (L552) + key rescale (L554): per (token, head) row of D channels
//                            y = ReLU(RMSNorm(x) * w),  raw = y,  rot = rho(y) on adjacent channel pairs,
//                            keys additionally * 1/sqrt(D N).  q and k are read ONCE and all four feature tensors the
//                            recurrence needs (q_rot, k_rot for the KV memory; q_raw, k_raw for the normaliser) leave.
//   gates_body           Eq. 13-15 (L562-L572): beta_n = sigmoid(W_beta . x_n + b_beta) per token,
//                            alpha_f = exp(-e^{A_log} softplus(W_alpha . mean_n x_n + b_alpha)) per frame.  The mean
//                            commutes with the projection, so the frame sum of the per-token dots is accumulated in a
//                            FIXED order (per 16-lane group, then over groups, then over the splits of a frame by the
//                            last CTA to arrive): reruns are bit-identical.
#pragma once
#include <cuda_bf16.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace gdn {

struct FeatmapParams {
    const __nv_bfloat16 *q, *k;            // [B][T][H][D], token strides q_ts / k_ts (elements)
    const float *wq, *wk;                  // [H][D] RMSNorm weights
    const float *cosT, *sinT;              // [T][D/2] rotation tables
    __nv_bfloat16 *q_rot, *k_rot, *q_raw, *k_raw;   // dense [B][T][H][D]
    long long q_ts, k_ts;
    int B, T, H, D;
    float rms_eps, kscale;                 // kscale = 1 / sqrt(D N)
};

struct GateParams {
    const __nv_bfloat16* x;                // [B][T][H][D], token stride x_ts
    const float *w_alpha, *b_alpha, *a_log, *w_beta, *b_beta;   // [H][D], [H], [H], [H][D], [H]
    float *alpha_out, *beta_out;           // [B][H][F], [B][H][T]
    float* part;                           // [B*H*F][NSPL] partial frame sums of W_alpha . x_n
    unsigned int* counters;                // [B*H*F], zero between calls (self-resetting)
    long long x_ts;
    int B, T, H, D, G, F, NSPL;
    int log_alpha;                         // write log(alpha) instead of alpha (plans with GDN_FLAG_LOG_ALPHA)
};

namespace fe {

// a 16-byte read of data that is used once (q, k, x): non-coherent path, and an L2 evict-first policy so that the stream does
// not push the previous kernel's dirty lines (or the feature tensors this kernel writes for the next one) out of L2
__device__ __forceinline__ uint4 ldg_stream(const uint4* p, uint64_t pol) {
    uint4 v;
    asm volatile("ld.global.nc.L2::cache_hint.v4.u32 {%0, %1, %2, %3}, [%4], %5;" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p), "l"(pol));
    return v;
}
__device__ __forceinline__ uint64_t stream_policy() {
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}


__device__ __forceinline__ void unpack8f(const uint4& u, float (&f)[8]) {
    const __nv_bfloat162* h = reinterpret_cast<const __nv_bfloat162*>(&u);
#pragma unroll
    for (int i = 0; i < 4; ++i) { const float2 t = __bfloat1622float2(h[i]); f[2 * i] = t.x; f[2 * i + 1] = t.y; }
}
__device__ __forceinline__ uint4 pack8f(const float (&f)[8]) {
    uint4 u;
    __nv_bfloat162* h = reinterpret_cast<__nv_bfloat162*>(&u);
#pragma unroll
    for (int i = 0; i < 4; ++i) h[i] = __floats2bfloat162_rn(f[2 * i], f[2 * i + 1]);
    return u;
}
// sum over the 16 lanes of a half-warp (xor butterflies stay inside the half)
__device__ __forceinline__ float group16_sum(float v) {
#pragma unroll
    for (int o = 8; o >= 1; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    return v;
}

constexpr int kFeThreads = 256;            // 16 rows of 16 lanes; a lane owns 8 consecutive channels (D <= 128)

constexpr int kFeRows = 2;                 // rows / tokens a 16-lane group has in flight per iteration (independent loads)

// Feature map of rows r0 + g + 16 j (j < kFeRows) of [B*T*H] (row = one token of one head), grid-stride over row groups.
__device__ __forceinline__ void featmap_body(const FeatmapParams& p, int block, int nblocks) {
    const int g = threadIdx.x >> 4, l = threadIdx.x & 15;
    const int rows = p.B * p.T * p.H;           // < 2^31 (checked by the host): 32-bit index arithmetic, the 64-bit
    const int c0 = l * 8;                       // divisions by H and T were a third of this kernel's instructions
    const bool on = c0 < p.D;
    const float inv_d = 1.f / (float)p.D;
    constexpr int R = kFeRows;
    for (int r0 = block * 16 * R; r0 < rows; r0 += nblocks * 16 * R) {   // uniform trip count: the shuffles need the whole warp
        float xq[R][8], xk[R][8];
        int rr[R], hh[R], tt[R];
        bool valid[R];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            valid[j] = r0 + g + 16 * j < rows;
            rr[j] = valid[j] ? r0 + g + 16 * j : rows - 1;
            const unsigned int btu = (unsigned int)rr[j] / (unsigned int)p.H;
            const int h = rr[j] - (int)btu * p.H;
            const long long bt = btu;
            hh[j] = h;
            tt[j] = (int)(btu % (unsigned int)p.T);
#pragma unroll
            for (int i = 0; i < 8; ++i) { xq[j][i] = 0.f; xk[j][i] = 0.f; }
            if (on) {
                unpack8f(ldg_stream(reinterpret_cast<const uint4*>(p.q + bt * p.q_ts + (long long)h * p.D + c0), stream_policy()), xq[j]);
                unpack8f(ldg_stream(reinterpret_cast<const uint4*>(p.k + bt * p.k_ts + (long long)h * p.D + c0), stream_policy()), xk[j]);
            }
        }
#pragma unroll
        for (int j = 0; j < R; ++j) {
            float sq = 0.f, sk = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) { sq = fmaf(xq[j][i], xq[j][i], sq); sk = fmaf(xk[j][i], xk[j][i], sk); }
            sq = group16_sum(sq);
            sk = group16_sum(sk);
            if (!on || !valid[j]) continue;
            const int h = hh[j], t = tt[j];
            const float rq = rsqrtf(sq * inv_d + p.rms_eps), rk = rsqrtf(sk * inv_d + p.rms_eps);
            const float4 wq0 = __ldg(reinterpret_cast<const float4*>(p.wq + (long long)h * p.D + c0));
            const float4 wq1 = __ldg(reinterpret_cast<const float4*>(p.wq + (long long)h * p.D + c0 + 4));
            const float4 wk0 = __ldg(reinterpret_cast<const float4*>(p.wk + (long long)h * p.D + c0));
            const float4 wk1 = __ldg(reinterpret_cast<const float4*>(p.wk + (long long)h * p.D + c0 + 4));
            const float wqv[8] = {wq0.x, wq0.y, wq0.z, wq0.w, wq1.x, wq1.y, wq1.z, wq1.w};
            const float wkv[8] = {wk0.x, wk0.y, wk0.z, wk0.w, wk1.x, wk1.y, wk1.z, wk1.w};
            const float4 cs = __ldg(reinterpret_cast<const float4*>(p.cosT + (long long)t * (p.D / 2) + c0 / 2));
            const float4 sn = __ldg(reinterpret_cast<const float4*>(p.sinT + (long long)t * (p.D / 2) + c0 / 2));
            const float cv[4] = {cs.x, cs.y, cs.z, cs.w}, sv[4] = {sn.x, sn.y, sn.z, sn.w};
            float qr[8], kr[8], qo[8], ko[8];
#pragma unroll
            for (int i = 0; i < 8; ++i) {
                qr[i] = fmaxf(xq[j][i] * rq * wqv[i], 0.f);
                kr[i] = fmaxf(xk[j][i] * rk * wkv[i], 0.f) * p.kscale;
            }
#pragma unroll
            for (int i = 0; i < 4; ++i) {
                qo[2 * i] = qr[2 * i] * cv[i] - qr[2 * i + 1] * sv[i];
                qo[2 * i + 1] = qr[2 * i] * sv[i] + qr[2 * i + 1] * cv[i];
                ko[2 * i] = kr[2 * i] * cv[i] - kr[2 * i + 1] * sv[i];
                ko[2 * i + 1] = kr[2 * i] * sv[i] + kr[2 * i + 1] * cv[i];
            }
            const long long o = (long long)rr[j] * p.D + c0;
            *reinterpret_cast<uint4*>(p.q_raw + o) = pack8f(qr);
            *reinterpret_cast<uint4*>(p.k_raw + o) = pack8f(kr);
            *reinterpret_cast<uint4*>(p.q_rot + o) = pack8f(qo);
            *reinterpret_cast<uint4*>(p.k_rot + o) = pack8f(ko);
        }
    }
}

// Split s of frame (b, h, f) owns the tokens [s*per, (s+1)*per): group g of the CTA takes tokens base + g, base + g + 16, ...
// in order, so every partial sum has a fixed association.
__device__ __forceinline__ void gates_body(const GateParams& p, int bhf, int s, float* s_sum, unsigned int* s_last) {
    const int g = threadIdx.x >> 4, l = threadIdx.x & 15;
    const int f = bhf % p.F, bh = bhf / p.F, b = bh / p.H, h = bh % p.H;
    const int per = (p.G + p.NSPL - 1) / p.NSPL;               // tokens per split
    const int n_lo = s * per, n_hi = min(n_lo + per, p.G);
    const int c0 = l * 8;
    const bool on = c0 < p.D;
    constexpr int R = kFeRows;
    float wa[8], wb[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) { wa[i] = 0.f; wb[i] = 0.f; }
    if (on) {
#pragma unroll
        for (int i = 0; i < 8; ++i) { wa[i] = __ldg(p.w_alpha + (long long)h * p.D + c0 + i); wb[i] = __ldg(p.w_beta + (long long)h * p.D + c0 + i); }
    }
    const float bb = __ldg(p.b_beta + h);
    float acc = 0.f;                                           // sum of W_alpha . x_n over this group's tokens, in token order
    for (int n0 = n_lo; n0 < n_hi; n0 += 16 * R) {             // uniform trip count: the shuffles need the whole warp
        float x[R][8];
        bool valid[R];
#pragma unroll
        for (int j = 0; j < R; ++j) {
            const int n = n0 + g + 16 * j;
            valid[j] = n < n_hi;
#pragma unroll
            for (int i = 0; i < 8; ++i) x[j][i] = 0.f;
            if (on && valid[j])
                unpack8f(ldg_stream(reinterpret_cast<const uint4*>(p.x + ((long long)b * p.T + (long long)f * p.G + n) * p.x_ts + (long long)h * p.D + c0), stream_policy()), x[j]);
        }
#pragma unroll
        for (int j = 0; j < R; ++j) {
            float da = 0.f, db = 0.f;
#pragma unroll
            for (int i = 0; i < 8; ++i) { da = fmaf(wa[i], x[j][i], da); db = fmaf(wb[i], x[j][i], db); }
            da = group16_sum(da);
            db = group16_sum(db);
            acc += da;                                         // da = 0 for a tail slot (x = 0)
            if (l == 0 && valid[j]) p.beta_out[(long long)bh * p.T + (long long)f * p.G + n0 + g + 16 * j] = 1.f / (1.f + __expf(-(db + bb)));      // Eq. 15
        }
    }
    if (l == 0) s_sum[g] = acc;
    __syncthreads();
    if (threadIdx.x == 0) {
        float tot = 0.f;
#pragma unroll
        for (int i = 0; i < 16; ++i) tot += s_sum[i];
        p.part[(long long)bhf * p.NSPL + s] = tot;
        __threadfence();
        *s_last = atomicAdd(p.counters + bhf, 1u) == (unsigned int)(p.NSPL - 1) ? 1u : 0u;
        if (*s_last) {
            __threadfence();
            float sum = 0.f;
            for (int i = 0; i < p.NSPL; ++i) sum += __ldcg(p.part + (long long)bhf * p.NSPL + i);
            const float pre = sum / (float)p.G + __ldg(p.b_alpha + h);                           // W_alpha . x_bar + b_alpha (Eq. 13-14)
            const float delta = fmaxf(pre, 0.f) + log1pf(__expf(-fabsf(pre)));                   // softplus
            const float la = -__expf(__ldg(p.a_log + h)) * delta;
            p.alpha_out[(long long)bh * p.F + f] = p.log_alpha ? la : __expf(la);
            p.counters[bhf] = 0u;
        }
    }
}

// ONE launch for the front end: blocks [0, n_g) run the gates, the remaining n_fm the feature map (either part may be empty).
// The gate blocks come first: their two-step reduction is a chain of latencies (13 us alone for 13.5 MB), which then runs
// beside the bandwidth-bound feature map instead of after it.  The recurrence's first kernel is launched as a programmatic
// dependent of this one.
__global__ void __launch_bounds__(kFeThreads, 4)
gdn_frontend_kernel(const FeatmapParams fm, const GateParams gp, const int n_g) {
    __shared__ float s_sum[16];
    __shared__ unsigned int s_last;
    if ((int)blockIdx.x >= n_g) {
        featmap_body(fm, (int)blockIdx.x - n_g, (int)gridDim.x - n_g);
    } else {
        const int idx = (int)blockIdx.x;
        gates_body(gp, idx / gp.NSPL, idx % gp.NSPL, s_sum, &s_last);
    }
    // only now: dependents launched earlier would sit on the SMs (Phase A's CTAs take most of an SM's shared memory)
    // while blocks of this grid are still waiting to be scheduled
    asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
}

}  // namespace fe
}  // namespace gdn
