// gdn_tc_token.cuh -- token-wise (G = 1) Gated DeltaNet forward on tcgen05 tensor cores.
//
// Chunkwise-parallel (WY/UT) form of PAPER.md Eq. 17-19 at N = 1, per
// compute tile of C tokens with tile-initial state S0, Gam_i = sum_{j<=i} log alpha_j, gamma = e^Gam:
//     L_ij = beta_i e^{Gam_i-Gam_j} k_i.k_j (j<i),   Tm = (I+L)^-1,
//     W = Tm diag(beta gamma) K,   Ut = Tm diag(beta) V,   Kt = diag(gamma_C/gamma) K,
//     P_ij = e^{Gam_i-Gam_j} q_i.k_j (j<=i)
//   state-independent per-chunk summaries (all chunks in parallel, kernel 1 "prepass"):
//     G_c = Kt^T W,  N_c = Kt^T Ut,  Qt = diag(gamma) Q - P W,  Ol = P Ut,  gamma_C
//   serial chain over chunks, ONE MMA per chunk (kernel 2 "chain"):
//     S_{c+1} = gamma_C S_c - G_c S_c + N_c          (fp32 master state in registers)
//   output, all chunks in parallel (kernel 3 "output"):
//     O_c = scale (Qt_c S_c + Ol_c)
// Every exponent is a difference Gam_i - Gam_j with i >= j (<= 0): nothing overflows.
//
// All kernels: 128 threads, thread i <-> token row i <-> TMEM lane i; one elected thread issues TMA and
// tcgen05.mma; operands are 128-byte-swizzled bf16 tiles (tc_common.cuh); accumulators live in TMEM.
// The prepass always works on 128-token tiles; for C = 64 the two chunks of a tile are handled as a
// block-diagonal pair so every MMA keeps M = 128.
#pragma once
#include <cuda.h>

#include "tc_common.cuh"

namespace gdn {

struct TokParams {
    const float* alpha;          // [BH][T]
    const float* beta;           // [BH][T]
    const float* S_in;           // [BH][D][D] or nullptr
    float* S_out;                // [BH][D][D]
    void* out;                   // [B][T][H][D] bf16
    __nv_bfloat16* Gw;           // [BH][NC][D][D]     G_c
    float* Nw;                   // [BH][NC][D][D]     N_c
    float* gam;                  // [BH][NC]           gamma_C
    __nv_bfloat16* Qt;           // [BH][NT*128][D]    Qt rows
    __nv_bfloat16* Ol;           // [BH][NT*128][D]    Ol rows
    __nv_bfloat16* Sc;           // [BH][NC][D][D]     state at chunk start (bf16 MMA operand)
    int B, H, T, NT, NC;
    long long o_ts;              // out token stride (elements)
    float scale;
    int log_alpha;
};

namespace tok {

using namespace tc;

constexpr uint32_t kBlk = 16384;      // one [128][64] bf16 block

__device__ __forceinline__ void st_global_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.global.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Kernel 1: prepass.  grid = BH * NT, block = 128.
// ---------------------------------------------------------------------------------------------------
template <int D, int C>
__global__ void __launch_bounds__(128, 1)
gdn_tok_prepass(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const TokParams p) {
    constexpr int NB = D / 64;
    constexpr uint32_t TILE = NB * kBlk;
    constexpr int KS = 8;                         // K = 16 steps over the 128 tokens of a tile
    constexpr int DS = D / 16;                    // K = 16 steps over the head dim
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sK = smem;
    uint8_t* sQ = smem + TILE;
    uint8_t* sV = smem + 2 * TILE;
    uint8_t* sA = smem + 3 * TILE;                // L_off -> Tm diag(beta gamma) -> Ut
    uint8_t* sB = sA + 2 * kBlk;                  // D (block-diagonal inverse) -> W
    uint8_t* sC = sB + 2 * kBlk;                  // X -> Tm diag(beta) -> P
    float* sGam = reinterpret_cast<float*>(sC + 2 * kBlk);     // [128] Gam_i (segmented for C = 64)
    float* sBeta = sGam + 128;                                 // [128] beta_j
    float* sBG = sBeta + 128;                                  // [128] beta_j e^{Gam_j}
    float* sWarp = sBG + 128;                                  // [4] per-warp sums of log alpha
    uint64_t* bars = reinterpret_cast<uint64_t*>(sWarp + 4);   // [3]
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int tile = blockIdx.x % p.NT, bh = blockIdx.x / p.NT;
    const int b = bh / p.H, h = bh % p.H;
    uint64_t* bar_kq = &bars[0];
    uint64_t* bar_v = &bars[1];
    uint64_t* bar_mma = &bars[2];

    if (tid == 0) {
        mbar_init(bar_kq, 1); mbar_init(bar_v, 1); mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t c0 = tmem, c1 = tmem + 128, c2 = tmem + 256, c3 = tmem + 384;

    if (tid == 0) {
        mbar_expect_tx(bar_kq, 2 * TILE);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            tma_load_5d(sK + nb * kBlk, &tmK, bar_kq, nb * 64, h, tile * 128, 0, b);
            tma_load_5d(sQ + nb * kBlk, &tmQ, bar_kq, nb * 64, h, tile * 128, 0, b);
        }
        mbar_expect_tx(bar_v, TILE);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_5d(sV + nb * kBlk, &tmV, bar_v, nb * 64, h, tile * 128, 0, b);
    }

    // ---- T0: gates, in-tile inclusive scan of log alpha ------------------------------------------
    const int t = tile * 128 + tid;
    const bool valid = t < p.T;
    float g = 0.f, beta_i = 0.f;
    if (valid) {
        const float a = p.alpha[(long long)bh * p.T + t];
        g = p.log_alpha ? a : logf(a);
        beta_i = p.beta[(long long)bh * p.T + t];
    }
    float x = g;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const float y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (lane == 31) sWarp[warp] = x;
    __syncthreads();
    float gam_i, gam_end;            // Gam_i and Gam at the end of this row's chunk
    {
        const float w0 = sWarp[0], w1 = sWarp[1], w2 = sWarp[2], w3 = sWarp[3];
        if (C == 128) {
            gam_i = x + (warp > 0 ? w0 : 0.f) + (warp > 1 ? w1 : 0.f) + (warp > 2 ? w2 : 0.f);
            gam_end = w0 + w1 + w2 + w3;
        } else {
            gam_i = x + ((warp & 1) ? (warp == 1 ? w0 : w2) : 0.f);
            gam_end = warp < 2 ? (w0 + w1) : (w2 + w3);
        }
    }
    sGam[tid] = gam_i;
    sBeta[tid] = beta_i;
    sBG[tid] = beta_i * __expf(gam_i);
    __syncthreads();
    const int half_lo = (C == 128) ? 0 : (warp >> 1) * 2;      // first 32-column chunk of this row's chunk

    uint32_t ph = 0;
    // ---- T1: K K^T -> c0, Q K^T -> c1 ------------------------------------------------------------
    mbar_wait(bar_kq, 0);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, 128, false, false);
        const uint32_t aK = smem_u32(sK), aQ = smem_u32(sQ);
#pragma unroll
        for (int s = 0; s < DS; ++s) {
            const uint32_t off = (s >> 2) * kBlk + (s & 3) * 32;
            umma_bf16(c0, desc_kmajor(aK + off), desc_kmajor(aK + off), id, s > 0);
        }
#pragma unroll
        for (int s = 0; s < DS; ++s) {
            const uint32_t off = (s >> 2) * kBlk + (s & 3) * 32;
            umma_bf16(c1, desc_kmajor(aQ + off), desc_kmajor(aK + off), id, s > 0);
        }
        umma_commit(bar_mma);
    }
    mbar_wait(bar_mma, ph); ph ^= 1;
    tc_fence_after();

    // ---- T2: L (strictly lower, decay-masked), 32x32 diagonal-block inverse in registers ---------
    float Ld[32];
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        float v[32];
        if (cc > warp || cc < half_lo) {
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = 0.f;
        } else {
            tmem_ld32(tmem_addr(c0, warp * 32, cc * 32), v);
#pragma unroll
            for (int jj = 0; jj < 32; ++jj) {
                const int j = cc * 32 + jj;
                v[jj] = (j < tid) ? beta_i * __expf(gam_i - sGam[j]) * v[jj] : 0.f;
            }
            if (cc == warp) {
#pragma unroll
                for (int jj = 0; jj < 32; ++jj) { Ld[jj] = v[jj]; v[jj] = 0.f; }
            }
        }
        store_row32_bf16(smem_u32(sA), kBlk, tid, cc * 32, v);
    }
    float X[32];                                   // row `lane` of (I + Ld)^-1
#pragma unroll
    for (int c = 0; c < 32; ++c) X[c] = (c == lane) ? 1.f : 0.f;
#pragma unroll
    for (int j = 0; j < 31; ++j) {
#pragma unroll
        for (int c = 0; c <= j; ++c) {
            const float xjc = __shfl_sync(0xffffffffu, X[c], j);
            if (lane > j) X[c] = fmaf(-Ld[j], xjc, X[c]);
        }
    }
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        float v[32];
#pragma unroll
        for (int j = 0; j < 32; ++j) v[j] = (cc == warp) ? X[j] : 0.f;
        store_row32_bf16(smem_u32(sB), kBlk, tid, cc * 32, v);
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    // one doubling level: Y = D (L_off D); returns with Y in c0
    auto doubling_mmas = [&]() {
        if (tid == 0) {           // X = L_off * D  (A = sA K-major, B = sB MN-major)
            tc_fence_after();
            const uint32_t id = umma_idesc(128, 128, false, true);
            const uint32_t aA = smem_u32(sA), aB = smem_u32(sB);
#pragma unroll
            for (int s = 0; s < KS; ++s)
                umma_bf16(c0, desc_kmajor(aA + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aB + s * 2048, kBlk), id, s > 0);
            umma_commit(bar_mma);
        }
        mbar_wait(bar_mma, ph); ph ^= 1;
        tc_fence_after();
#pragma unroll
        for (int cc = 0; cc < 4; ++cc) {
            float v[32];
            tmem_ld32(tmem_addr(c0, warp * 32, cc * 32), v);
            store_row32_bf16(smem_u32(sC), kBlk, tid, cc * 32, v);
        }
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
        if (tid == 0) {           // Y = D * X  (A = sB K-major, B = sC MN-major)
            tc_fence_after();
            const uint32_t id = umma_idesc(128, 128, false, true);
            const uint32_t aB = smem_u32(sB), aC = smem_u32(sC);
#pragma unroll
            for (int s = 0; s < KS; ++s)
                umma_bf16(c0, desc_kmajor(aB + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aC + s * 2048, kBlk), id, s > 0);
            umma_commit(bar_mma);
        }
        mbar_wait(bar_mma, ph); ph ^= 1;
        tc_fence_after();
    };

    // ---- T3/T4: 32 -> 64 blocks: D' = D - mask(D L_off D) ------------------------------------------
    doubling_mmas();
    float Dlow[32];                                // block (warp, warp-1) of the 64x64 inverse, odd warps
#pragma unroll
    for (int j = 0; j < 32; ++j) Dlow[j] = 0.f;
    if (warp & 1) {
        float v[32];
        tmem_ld32(tmem_addr(c0, warp * 32, (warp - 1) * 32), v);
#pragma unroll
        for (int j = 0; j < 32; ++j) Dlow[j] = -v[j];
        store_row32_bf16(smem_u32(sB), kBlk, tid, (warp - 1) * 32, Dlow);
    }
    float Tlow[64];                                // rows >= 64, columns 0..63 of the 128x128 inverse
#pragma unroll
    for (int j = 0; j < 64; ++j) Tlow[j] = 0.f;
    if (C == 128) {
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
        doubling_mmas();
        if (warp >= 2) {
            float v[32];
            tmem_ld32(tmem_addr(c0, warp * 32, 0), v);
#pragma unroll
            for (int j = 0; j < 32; ++j) Tlow[j] = -v[j];
            tmem_ld32(tmem_addr(c0, warp * 32, 32), v);
#pragma unroll
            for (int j = 0; j < 32; ++j) Tlow[32 + j] = -v[j];
        }
    }
    // ---- scaled copies of Tm: sA = Tm diag(beta gamma), sC = Tm diag(beta) -------------------------
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        float va[32], vc[32];
#pragma unroll
        for (int jj = 0; jj < 32; ++jj) {
            float tm;
            if (cc == warp) tm = X[jj];
            else if ((warp & 1) && cc == warp - 1) tm = Dlow[jj];
            else if (C == 128 && warp >= 2 && cc < 2) tm = Tlow[cc * 32 + jj];
            else tm = 0.f;
            va[jj] = tm * sBG[cc * 32 + jj];
            vc[jj] = tm * sBeta[cc * 32 + jj];
        }
        store_row32_bf16(smem_u32(sA), kBlk, tid, cc * 32, va);
        store_row32_bf16(smem_u32(sC), kBlk, tid, cc * 32, vc);
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    // ---- T7: W = Tm diag(beta gamma) K -> c2,  Ut = Tm diag(beta) V -> c3 ---------------------------
    mbar_wait(bar_v, 0);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, D, false, true);
        const uint32_t aA = smem_u32(sA), aC = smem_u32(sC), aK = smem_u32(sK), aV = smem_u32(sV);
#pragma unroll
        for (int s = 0; s < KS; ++s)
            umma_bf16(c2, desc_kmajor(aA + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aK + s * 2048, kBlk), id, s > 0);
#pragma unroll
        for (int s = 0; s < KS; ++s)
            umma_bf16(c3, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aV + s * 2048, kBlk), id, s > 0);
        umma_commit(bar_mma);
    }
    mbar_wait(bar_mma, ph); ph ^= 1;
    tc_fence_after();

    // ---- round trip 6: W -> sB, Ut -> sA, P -> sC, Kt in place -------------------------------------
#pragma unroll
    for (int cc = 0; cc < D / 32; ++cc) {
        float v[32];
        tmem_ld32(tmem_addr(c2, warp * 32, cc * 32), v);
        store_row32_bf16(smem_u32(sB), kBlk, tid, cc * 32, v);
        tmem_ld32(tmem_addr(c3, warp * 32, cc * 32), v);
        store_row32_bf16(smem_u32(sA), kBlk, tid, cc * 32, v);
    }
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        float v[32];
        if (cc > warp || cc < half_lo) {
#pragma unroll
            for (int j = 0; j < 32; ++j) v[j] = 0.f;
        } else {
            tmem_ld32(tmem_addr(c1, warp * 32, cc * 32), v);
#pragma unroll
            for (int jj = 0; jj < 32; ++jj) {
                const int j = cc * 32 + jj;
                v[jj] = (j <= tid) ? __expf(gam_i - sGam[j]) * v[jj] : 0.f;
            }
        }
        store_row32_bf16(smem_u32(sC), kBlk, tid, cc * 32, v);
    }
    {
        const float ks = __expf(gam_end - gam_i);
#pragma unroll
        for (int ch = 0; ch < D / 8; ++ch) {
            const uint32_t addr = smem_u32(sK) + swz_chunk_off(tid, ch, kBlk);
            float f[8];
            unpack8(ld_shared_v4(addr), f);
            st_shared_v4(addr, pack_bf16(f[0] * ks, f[1] * ks), pack_bf16(f[2] * ks, f[3] * ks),
                         pack_bf16(f[4] * ks, f[5] * ks), pack_bf16(f[6] * ks, f[7] * ks));
        }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    // ---- T8: G = Kt^T W -> c0, N = Kt^T Ut -> c1, P W -> c2, P Ut -> c3 -----------------------------
    const float gamma_i = __expf(gam_i);
    constexpr int NHALF = (C == 128) ? 1 : 2;
#pragma unroll
    for (int hf = 0; hf < NHALF; ++hf) {
        if (tid == 0) {
            tc_fence_after();
            const uint32_t aA = smem_u32(sA), aB = smem_u32(sB), aC = smem_u32(sC), aK = smem_u32(sK);
            const uint32_t idg = umma_idesc(D, D, true, true);
            const int s_lo = (C == 128) ? 0 : hf * 4, s_hi = (C == 128) ? KS : hf * 4 + 4;
            for (int s = s_lo; s < s_hi; ++s)
                umma_bf16(c0, desc_mnmajor(aK + s * 2048, kBlk), desc_mnmajor(aB + s * 2048, kBlk), idg, s > s_lo);
            for (int s = s_lo; s < s_hi; ++s)
                umma_bf16(c1, desc_mnmajor(aK + s * 2048, kBlk), desc_mnmajor(aA + s * 2048, kBlk), idg, s > s_lo);
            if (hf == 0) {
                const uint32_t idp = umma_idesc(128, D, false, true);
#pragma unroll
                for (int s = 0; s < KS; ++s)
                    umma_bf16(c2, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aB + s * 2048, kBlk), idp, s > 0);
#pragma unroll
                for (int s = 0; s < KS; ++s)
                    umma_bf16(c3, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aA + s * 2048, kBlk), idp, s > 0);
            }
            umma_commit(bar_mma);
        }
        mbar_wait(bar_mma, ph); ph ^= 1;
        tc_fence_after();

        // ---- round trip 7: write the summaries to the workspace ----------------------------------
        const int chunk = (C == 128) ? tile : 2 * tile + hf;
        const long long cidx = (long long)bh * p.NC + chunk;
        const int m = (D == 128) ? tid : (16 * warp + lane);       // summary row held by this thread
        const bool m_ok = (D == 128) || (lane < 16);
#pragma unroll
        for (int cc = 0; cc < D / 32; ++cc) {
            float v[32];
            tmem_ld32(tmem_addr(c0, warp * 32, cc * 32), v);
            if (m_ok) {
                __nv_bfloat16* dst = p.Gw + (cidx * D + m) * D + cc * 32;
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4)
                    st_global_v4(dst + q4 * 8, pack_bf16(v[8 * q4], v[8 * q4 + 1]), pack_bf16(v[8 * q4 + 2], v[8 * q4 + 3]),
                                 pack_bf16(v[8 * q4 + 4], v[8 * q4 + 5]), pack_bf16(v[8 * q4 + 6], v[8 * q4 + 7]));
            }
            tmem_ld32(tmem_addr(c1, warp * 32, cc * 32), v);
            if (m_ok) {
                float* dst = p.Nw + (cidx * D + m) * D + cc * 32;
#pragma unroll
                for (int q4 = 0; q4 < 8; ++q4)
                    st_global_v4(dst + q4 * 4, __float_as_uint(v[4 * q4]), __float_as_uint(v[4 * q4 + 1]),
                                 __float_as_uint(v[4 * q4 + 2]), __float_as_uint(v[4 * q4 + 3]));
            }
        }
        if (C == 128) { if (tid == 0) p.gam[cidx] = __expf(gam_end); }
        else { if (tid == 64 * hf) p.gam[cidx] = __expf(gam_end); }
        if (hf == 0) {
            const long long row = ((long long)bh * p.NT + tile) * 128 + tid;
#pragma unroll
            for (int cc = 0; cc < D / 32; ++cc) {
                float v[32];
                tmem_ld32(tmem_addr(c2, warp * 32, cc * 32), v);        // (P W)_i
                __nv_bfloat16* dq = p.Qt + row * D + cc * 32;
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    float f[8];
                    unpack8(ld_shared_v4(smem_u32(sQ) + swz_chunk_off(tid, cc * 4 + q4, kBlk)), f);
#pragma unroll
                    for (int e = 0; e < 8; ++e) f[e] = gamma_i * f[e] - v[8 * q4 + e];
                    st_global_v4(dq + q4 * 8, pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
                }
                tmem_ld32(tmem_addr(c3, warp * 32, cc * 32), v);        // (P Ut)_i
                __nv_bfloat16* dl = p.Ol + row * D + cc * 32;
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4)
                    st_global_v4(dl + q4 * 8, pack_bf16(v[8 * q4], v[8 * q4 + 1]), pack_bf16(v[8 * q4 + 2], v[8 * q4 + 3]),
                                 pack_bf16(v[8 * q4 + 4], v[8 * q4 + 5]), pack_bf16(v[8 * q4 + 6], v[8 * q4 + 7]));
            }
        }
        if (hf + 1 < NHALF) { tc_fence_before(); __syncthreads(); }
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 512);
}

// ---------------------------------------------------------------------------------------------------
// Kernel 2: chain.  grid = BH * (D/64) column tiles, block = 128.  One MMA per chunk on the chain.
//   tmG: bf16 (D cols, D rows, BH*NC) box {64, D, 1} swizzle 128B  -> A operand (K-major)
//   tmN: fp32 (D cols, D rows, BH*NC) box {32, D, 1} swizzle 128B  -> read by threads
// ---------------------------------------------------------------------------------------------------
template <int D>
struct ChainSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t G_BYTES = (uint32_t)D * D * 2;           // NB blocks of [D][64] bf16
    static constexpr uint32_t N_BYTES = (uint32_t)D * 64 * 4;          // 2 blocks of [D][32] fp32
    static constexpr uint32_t STAGE = G_BYTES + N_BYTES;
    static constexpr int STAGES = (D == 128) ? 3 : 4;
    static constexpr uint32_t S_BYTES = (uint32_t)D * 128;             // [D][64] bf16
    static constexpr uint32_t TOTAL = STAGES * STAGE + 2 * S_BYTES + 256 + 1024;
};

template <int D>
__global__ void __launch_bounds__(128, 1)
gdn_tok_chain(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmN, const TokParams p) {
    using L = ChainSmem<D>;
    constexpr int NB = L::NB;
    constexpr int STAGES = L::STAGES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sStage = smem;
    uint8_t* sS = smem + STAGES * L::STAGE;                            // 2 x [D][64] bf16 (MN-major B operand)
    uint64_t* bars = reinterpret_cast<uint64_t*>(sS + 2 * L::S_BYTES); // full[STAGES], mma
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + STAGES + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    constexpr int NT_COL = D / 64;
    const int ct = blockIdx.x % NT_COL, bh = blockIdx.x / NT_COL;
    const int n0 = ct * 64;
    const int m = (D == 128) ? tid : (16 * warp + lane);
    const bool m_ok = (D == 128) || (lane < 16);
    uint64_t* bar_mma = &bars[STAGES];

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&bars[s], 1);
        mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(tmem_slot, 64);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    auto issue_loads = [&](int c) {
        const int st = c % STAGES;
        uint8_t* base = sStage + st * L::STAGE;
        mbar_expect_tx(&bars[st], L::STAGE);
        const int z = bh * p.NC + c;
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_3d(base + nb * (D * 128), &tmG, &bars[st], nb * 64, 0, z);
        tma_load_3d(base + L::G_BYTES, &tmN, &bars[st], n0, 0, z);
        tma_load_3d(base + L::G_BYTES + D * 128, &tmN, &bars[st], n0 + 32, 0, z);
    };
    if (tid == 0)
        for (int c = 0; c < STAGES && c < p.NC; ++c) issue_loads(c);

    // state row m, columns n0..n0+63, fp32 master copy in registers
    float S[64];
    if (m_ok && p.S_in) {
        const float4* src = reinterpret_cast<const float4*>(p.S_in + ((long long)bh * D + m) * D + n0);
#pragma unroll
        for (int i = 0; i < 16; ++i) { const float4 f = src[i]; S[4 * i] = f.x; S[4 * i + 1] = f.y; S[4 * i + 2] = f.z; S[4 * i + 3] = f.w; }
    } else {
#pragma unroll
        for (int i = 0; i < 64; ++i) S[i] = 0.f;
    }
    // publish S (bf16): shared operand buffer `buf` + global snapshot for chunk `c` (read by kernel 3)
    auto publish = [&](int buf, int c) {
        if (m_ok) {
            const uint32_t sbase = smem_u32(sS + buf * L::S_BYTES);
            __nv_bfloat16* g = p.Sc + (((long long)bh * p.NC + c) * D + m) * D + n0;
#pragma unroll
            for (int ch = 0; ch < 8; ++ch) {
                const uint32_t a = pack_bf16(S[8 * ch], S[8 * ch + 1]), b2 = pack_bf16(S[8 * ch + 2], S[8 * ch + 3]);
                const uint32_t c2 = pack_bf16(S[8 * ch + 4], S[8 * ch + 5]), d2 = pack_bf16(S[8 * ch + 6], S[8 * ch + 7]);
                st_shared_v4(sbase + swz_chunk_off(m, ch, 0), a, b2, c2, d2);
                if (c < p.NC) st_global_v4(g + ch * 8, a, b2, c2, d2);
            }
        }
    };
    publish(0, 0);
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    uint32_t ph_mma = 0;
    for (int c = 0; c < p.NC; ++c) {
        const int st = c % STAGES;
        const uint32_t ph_full = (uint32_t)(c / STAGES) & 1u;
        const float gamma_c = p.gam[(long long)bh * p.NC + c];
        uint8_t* base = sStage + st * L::STAGE;
        mbar_wait(&bars[st], ph_full);
        if (tid == 0) {
            tc_fence_after();
            const uint32_t id = umma_idesc(D, 64, false, true);
            const uint32_t aG = smem_u32(base), aS = smem_u32(sS + (c & 1) * L::S_BYTES);
#pragma unroll
            for (int s = 0; s < D / 16; ++s)
                umma_bf16(tmem, desc_kmajor(aG + (s >> 2) * (D * 128) + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), id, s > 0);
            umma_commit(bar_mma);
        }
        mbar_wait(bar_mma, ph_mma); ph_mma ^= 1;
        tc_fence_after();
        // S <- gamma_c S - G_c S + N_c
#pragma unroll
        for (int cc = 0; cc < 2; ++cc) {
            float v[32];
            tmem_ld32(tmem_addr(tmem, warp * 32, cc * 32), v);
            if (m_ok) {
                const uint32_t nbase = smem_u32(base + L::G_BYTES + cc * (D * 128));
#pragma unroll
                for (int ch = 0; ch < 8; ++ch) {
                    const uint4 u = ld_shared_v4(nbase + swz_chunk_off(m, ch, 0));
                    const int i0 = cc * 32 + ch * 4;
                    S[i0 + 0] = fmaf(gamma_c, S[i0 + 0], __uint_as_float(u.x) - v[ch * 4 + 0]);
                    S[i0 + 1] = fmaf(gamma_c, S[i0 + 1], __uint_as_float(u.y) - v[ch * 4 + 1]);
                    S[i0 + 2] = fmaf(gamma_c, S[i0 + 2], __uint_as_float(u.z) - v[ch * 4 + 2]);
                    S[i0 + 3] = fmaf(gamma_c, S[i0 + 3], __uint_as_float(u.w) - v[ch * 4 + 3]);
                }
            }
        }
        publish((c + 1) & 1, c + 1);
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
        if (tid == 0 && c + STAGES < p.NC) issue_loads(c + STAGES);
    }
    if (m_ok) {
        float4* dst = reinterpret_cast<float4*>(p.S_out + ((long long)bh * D + m) * D + n0);
#pragma unroll
        for (int i = 0; i < 16; ++i) dst[i] = make_float4(S[4 * i], S[4 * i + 1], S[4 * i + 2], S[4 * i + 3]);
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 64);
}

// ---------------------------------------------------------------------------------------------------
// Kernel 3: output.  grid = BH * NT, block = 128.   O = scale (Qt S_c + Ol)
//   tmQt: bf16 (D cols, BH*NT*128 rows) box {64, 128}       -> A operand (K-major)
//   tmSc: bf16 (D cols, D rows, BH*NC)  box {64, D, 1}      -> B operand (MN-major)
// ---------------------------------------------------------------------------------------------------
template <int D, int C>
__global__ void __launch_bounds__(128)
gdn_tok_output(const __grid_constant__ CUtensorMap tmQt, const __grid_constant__ CUtensorMap tmSc, const TokParams p) {
    constexpr int NB = D / 64;
    constexpr int NS = (C == 128) ? 1 : 2;                     // states per 128-token tile
    constexpr uint32_t QT_BYTES = NB * kBlk;
    constexpr uint32_t S_BYTES = (uint32_t)D * D * 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQt = smem;
    uint8_t* sS = smem + QT_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sS + NS * S_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int tile = blockIdx.x % p.NT, bh = blockIdx.x / p.NT;
    const int b = bh / p.H, h = bh % p.H;
    if (tid == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_fence_init(); }
    if (warp == 0) tmem_alloc(tmem_slot, NS * D);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const long long row = ((long long)bh * p.NT + tile) * 128 + tid;
    if (tid == 0) {
        mbar_expect_tx(&bars[0], QT_BYTES + NS * S_BYTES);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_2d(sQt + nb * kBlk, &tmQt, &bars[0], nb * 64, (int)(((long long)bh * p.NT + tile) * 128));
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int nb = 0; nb < NB; ++nb)
                tma_load_3d(sS + s * S_BYTES + nb * (D * 128), &tmSc, &bars[0], nb * 64, 0, bh * p.NC + tile * NS + s);
    }
    // prefetch this row's Ol
    uint4 ol[D / 8];
    {
        const uint4* src = reinterpret_cast<const uint4*>(p.Ol + row * D);
#pragma unroll
        for (int i = 0; i < D / 8; ++i) ol[i] = __ldg(src + i);
    }
    mbar_wait(&bars[0], 0);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, D, false, true);
        const uint32_t aQ = smem_u32(sQt);
#pragma unroll
        for (int s2 = 0; s2 < NS; ++s2) {
            const uint32_t aS = smem_u32(sS + s2 * S_BYTES);
#pragma unroll
            for (int s = 0; s < D / 16; ++s)
                umma_bf16(tmem + s2 * D, desc_kmajor(aQ + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aS + s * 2048, D * 128), id, s > 0);
        }
        umma_commit(&bars[1]);
    }
    mbar_wait(&bars[1], 0);
    tc_fence_after();
    const int t = tile * 128 + tid;
    const uint32_t acc = tmem + ((NS == 2 && tid >= 64) ? D : 0);
    __nv_bfloat16* dst = reinterpret_cast<__nv_bfloat16*>(p.out) + ((long long)b * p.T + t) * p.o_ts + (long long)h * D;
#pragma unroll
    for (int cc = 0; cc < D / 32; ++cc) {
        float v[32];
        tmem_ld32(tmem_addr(acc, warp * 32, cc * 32), v);
        if (t < p.T) {
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4) {
                float f[8];
                unpack8(ol[cc * 4 + q4], f);
#pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = p.scale * (v[8 * q4 + e] + f[e]);
                st_global_v4(dst + cc * 32 + q4 * 8, pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, NS * D);
}

}  // namespace tok
}  // namespace gdn
