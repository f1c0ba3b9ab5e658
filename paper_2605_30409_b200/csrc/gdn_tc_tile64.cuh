// gdn_tc_tile64.cuh -- token-wise (G = 1) path, d = 64: the state-independent chunk summaries computed by LIGHT CTAs.
//
// Same mathematics as gdn_tc_token.cuh (chunkwise WY/UT form of PAPER.md Eq. 17-19 at N = 1, DESIGN.md "Chunkwise
// form"), per chunk of C = 64 tokens:
//     L_ij = beta_i e^{Gam_i-Gam_j} k_i.k_j (j<i),  Tm = (I+L)^-1,  W = Tm diag(beta gamma) K,  Ut = Tm diag(beta) V,
//     Kt = diag(gamma_C/gamma) K,  P_ij = e^{Gam_i-Gam_j} q_i.k_j (j<=i),
//     G_c = Kt^T W,  N_c = Kt^T Ut,  Qt = diag(gamma) Q - P W,  Ol = P Ut,  gamma_C.
// What changes is the shape of the worker.  A 128-token tile of gdn_tc_token.cuh fills an SM (166 KB of shared memory,
// 512 TMEM columns, 16 warps in lock-step) and is a dependent sequence of seven MMA round trips, so one tile is in
// flight per SM and the SM idles through every round trip.  Here one CTA of 128 threads owns one 64-token chunk with
// 51 KB of shared memory and 128 TMEM columns, FOUR such CTAs are resident per SM and hide each other's latencies, and
// the sequence is three MMA round trips:
//     S1  [K ; Q] K^T                      (M = 128: lanes 0-63 = K K^T rows, lanes 64-127 = Q K^T rows; N = 64)
//         warps 0-1: decay-masked L -> fp32 scratch; warps 2-3: decay-masked P -> P^T (bf16)
//         (I + L)^-1 of the 64x64 block in fp32 on CUDA cores: 16-blocks by forward substitution, 16 -> 32 -> 64 by
//         X21 = -X22 L21 X11 (no tensor-core doubling round trips, no bf16 rounding inside the inverse)
//     S3  [Tm diag(beta gamma) ; Tm diag(beta)] [K | V]   (M = 128, N = 128: lanes 0-63 keep columns 0-63 = W,
//         lanes 64-127 keep columns 64-127 = Ut; the other two quadrants are computed and ignored)
//     S4  [Kt | P^T]^T [W | Ut]            (M = 128 as an MN-major A operand of two blocks: lanes 0-63 = [G | N] rows,
//         lanes 64-127 = [P W | P Ut] rows)
// so every TMEM lane and every thread has a row to work on in every epilogue.
#pragma once
#include <cuda.h>

#include "gdn_tc_token.cuh"

namespace gdn {
namespace t64 {

using namespace tc;

constexpr int kThreads = 128;
constexpr int kLS = 68;                               // floats per row of the fp32 inversion scratch (16-byte aligned rows)
constexpr uint32_t kTile = 8192;                      // one [64][64] bf16 tile (128-byte rows, 128-byte swizzle)
constexpr uint32_t OFF_K = 0;                         // K tile  } the stacked K-major A operand of S1; K alone is its B operand
constexpr uint32_t OFF_Q = 8192;                      // Q tile  }   later: Kt in place / Qt in place
constexpr uint32_t OFF_V = 16384;                     // V tile; later Ol
constexpr uint32_t OFF_PT = 24576;                    // P^T [j][i] bf16; later the staging of G
constexpr uint32_t OFF_X = 32768;                     // fp32 scratch [64][kLS] -> [Tm diag(beta gamma) ; Tm diag(beta)] bf16 [128][64]
                                                      //   -> [W | Ut] bf16 2 x [64][64] -> staging of N
constexpr uint32_t X_BYTES = 64u * kLS * 4u;          // 17408
constexpr uint32_t OFF_VEC = OFF_X + X_BYTES;         // Gam[64], Beta[64], BG[64], KS[64], CF[32]
constexpr uint32_t OFF_BAR = OFF_VEC + 1280;
constexpr uint32_t SMEM_BYTES = OFF_BAR + 64 + 1024;  // + slack for the 1024-byte alignment of the dynamic base

struct Tile64Maps {
    const CUtensorMap *tmQ, *tmK, *tmV;               // activations, box [64 tokens][64 features]
    const CUtensorMap *tmG, *tmN;                     // G bf16 box {64, 64, 1}; N fp32 box {32, 64, 1}
    const CUtensorMap *tmQt, *tmOl;                   // workspace rows, box {64, 64}
};

__device__ __forceinline__ void sts_b16(uint32_t a, unsigned short v) { asm volatile("st.shared.b16 [%0], %1;" ::"r"(a), "h"(v) : "memory"); }

// One 64-token chunk `chunk` of stream `bh`.  smem: 1024-byte aligned base; tmem: 128 columns; bars: 4 mbarriers
// (K+Q landed, V landed, MMA complete, spare) initialised to count 1; `use` = how many chunks this CTA has run before.
__device__ __forceinline__ void tile64(uint8_t* smem, uint32_t tmem, uint64_t* bars, const Tile64Maps& mp, const TokParams& p,
                                       int bh, int chunk, uint32_t use) {
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = bh / p.H, h = bh % p.H;
    const uint32_t aK = smem_u32(smem + OFF_K), aQ = smem_u32(smem + OFF_Q), aV = smem_u32(smem + OFF_V);
    const uint32_t aPT = smem_u32(smem + OFF_PT), aX = smem_u32(smem + OFF_X), aVec = smem_u32(smem + OFF_VEC);
    const uint32_t aGam = aVec, aBeta = aVec + 256, aBG = aVec + 512, aKS = aVec + 768, aCF = aVec + 1024;
    uint64_t *bar_kq = &bars[0], *bar_v = &bars[1], *bar_mma = &bars[2];
    const uint32_t par = use & 1u;
    uint32_t ph = (3u * use) & 1u;                    // bar_mma completes three phases per chunk
    const int row = tid;                              // TMEM lane
    const int i = tid & 63;                           // token row inside the chunk (both halves of the CTA)
    const uint32_t lane_base = (uint32_t)(warp * 32);

    if (tid == 0) {
        mbar_expect_tx(bar_kq, 2 * kTile);
        tma_load_5d(smem + OFF_K, mp.tmK, bar_kq, 0, h, chunk * 64, 0, b);
        tma_load_5d(smem + OFF_Q, mp.tmQ, bar_kq, 0, h, chunk * 64, 0, b);
        mbar_expect_tx(bar_v, kTile);
        tma_load_5d(smem + OFF_V, mp.tmV, bar_v, 0, h, chunk * 64, 0, b);
    }
    // ---- gates: every warp scans the 64 log alpha of the chunk (two per lane), no cross-warp exchange ----
    float gam_i, beta_i, gam_C, gam_31;
    {
        const int t0 = chunk * 64 + lane, t1 = t0 + 32;
        float a0 = p.log_alpha ? 0.f : 1.f, a1 = a0, b0 = 0.f, b1 = 0.f;       // padding rows: alpha = 1, beta = 0
        if (t0 < p.T) { a0 = p.alpha[(long long)bh * p.T + t0]; b0 = p.beta[(long long)bh * p.T + t0]; }
        if (t1 < p.T) { a1 = p.alpha[(long long)bh * p.T + t1]; b1 = p.beta[(long long)bh * p.T + t1]; }
        float x0 = p.log_alpha ? a0 : logf(a0), x1 = p.log_alpha ? a1 : logf(a1);
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const float y0 = __shfl_up_sync(0xffffffffu, x0, o), y1 = __shfl_up_sync(0xffffffffu, x1, o);
            if (lane >= o) { x0 += y0; x1 += y1; }
        }
        gam_31 = __shfl_sync(0xffffffffu, x0, 31);
        x1 += gam_31;
        gam_C = __shfl_sync(0xffffffffu, x1, 31);
        gam_i = (warp & 1) ? x1 : x0;
        beta_i = (warp & 1) ? b1 : b0;
        if (warp == 0) {
            sts_f32(aGam + lane * 4, x0); sts_f32(aGam + (32 + lane) * 4, x1);
            sts_f32(aBeta + lane * 4, b0); sts_f32(aBeta + (32 + lane) * 4, b1);
            sts_f32(aBG + lane * 4, b0 * fast_exp(x0)); sts_f32(aBG + (32 + lane) * 4, b1 * fast_exp(x1));
            sts_f32(aKS + lane * 4, fast_exp(gam_C - x0)); sts_f32(aKS + (32 + lane) * 4, fast_exp(gam_C - x1));
            sts_f32(aCF + lane * 4, fast_exp(gam_31 - x0));
        }
    }
    __syncthreads();
    auto sync_then_issue = [&]() { fence_proxy_async(); tc_fence_before(); __syncthreads(); };
    auto wait_mma = [&]() { mbar_wait(bar_mma, ph); ph ^= 1; tc_fence_after(); };

    // ---- S1: [K ; Q] K^T -> TMEM columns 0..63 ----
    mbar_wait(bar_kq, par);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, 64, false, false);
#pragma unroll
        for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aK + s * 32), desc_kmajor(aK + s * 32), id, s > 0);
        umma_commit(bar_mma);
    }
    wait_mma();

    // ---- S1 epilogue.  warps 0-1 (row i of K K^T): L_ij = beta_i e^{Gam_i-Gam_j} k_i.k_j (j < i), stored TRANSPOSED in
    //      the fp32 scratch M (M[j][i] = L[i][j]: "column j of L" is then a row of 16-byte loads); warps 2-3 (row i of
    //      Q K^T): P_ij = e^{Gam_i-Gam_j} q_i.k_j (j <= i) -> bf16 P^T[j][i].  Inside a 32-column block the exponent is
    //      taken directly; across blocks e^{Gam_i-Gam_j} = e^{Gam_i-Gam_31} e^{Gam_31-Gam_j} (both factors <= 1).
    {
        const int ci = warp & 1;                      // 32-block of this row
        const bool is_l = warp < 2;
        const float rowf = is_l ? beta_i : 1.f;
        const float rf = rowf * fast_exp(fminf(gam_i - gam_31, 0.f));
#pragma unroll
        for (int hc = 0; hc < 2; ++hc) {
            float v[32];
            if (hc <= ci) {
                tmem_ld32(tmem_addr(tmem, lane_base, hc * 32), v);
                if (hc == ci) {
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const float4 g = lds_f4(aGam + (hc * 32 + 4 * q) * 4);
                        const float gj[4] = {g.x, g.y, g.z, g.w};
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            const int j = 4 * q + e;
                            const bool keep = is_l ? (j < lane) : (j <= lane);
                            v[j] *= keep ? rowf * fast_exp(fminf(gam_i - gj[e], 0.f)) : 0.f;
                        }
                    }
                } else {
#pragma unroll
                    for (int q = 0; q < 8; ++q) {
                        const float4 c = lds_f4(aCF + 16 * q);
                        v[4 * q] *= rf * c.x; v[4 * q + 1] *= rf * c.y; v[4 * q + 2] *= rf * c.z; v[4 * q + 3] *= rf * c.w;
                    }
                }
            } else {
                if (is_l) continue;                   // M[j >= 32][i < 32] is the lower-left block: written by the inversion
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = 0.f;
            }
            if (is_l) {
#pragma unroll
                for (int j = 0; j < 32; ++j) sts_f32(aX + ((hc * 32 + j) * kLS + i) * 4, v[j]);
            } else {
                const uint32_t colb = aPT + (uint32_t)((i & 7) * 2);
#pragma unroll
                for (int j = 0; j < 32; ++j) {
                    const int jj = hc * 32 + j;
                    sts_b16(colb + jj * 128 + ((((uint32_t)i >> 3) ^ (jj & 7)) << 4), __bfloat16_as_ushort(__float2bfloat16_rn(v[j])));
                }
            }
        }
    }

    // ---- (I + L)^-1 in fp32, in place in M.  After each stage the finished diagonal blocks hold X row-major (zeros
    //      above the diagonal) and the blocks above them still hold L^T.
    constexpr uint32_t S = kLS * 4;
    if (warp < 2) {
        // 16-blocks: the two halves of warp w invert the two diagonal 16-blocks of 32-block w, one column per lane
        // (right-looking forward substitution, tok::inv16_columns); then X21 = -X22 (L21 X11) of the 32-block.
        __syncwarp();
        const uint32_t aL = aX + (uint32_t)(32 * warp * kLS + 32 * warp) * 4;
        const int o = lane & 16, col = lane & 15;
        float xc[16];
        tok::inv16_columns<kLS>(aL + o * S + o * 4, col, xc);
        __syncwarp();
#pragma unroll
        for (int r = 0; r < 16; ++r) sts_f32(aL + (o + r) * S + (o + col) * 4, xc[r]);
        __syncwarp();
        const int r2 = lane >> 1, cc0 = (lane & 1) * 8;
        float acc[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = 0.f;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float a = lds_f32(aL + k * S + (16 + r2) * 4);                  // L21[r2][k]
            const float4 b0 = lds_f4(aL + k * S + cc0 * 4);                       // X11[k][cc0 ..]
            const float4 b1 = lds_f4(aL + k * S + (cc0 + 4) * 4);
            acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
            acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
        }
        sts_f4(aL + (16 + r2) * S + cc0 * 4, make_float4(acc[0], acc[1], acc[2], acc[3]));          // M1 into the free lower-left block
        sts_f4(aL + (16 + r2) * S + (cc0 + 4) * 4, make_float4(acc[4], acc[5], acc[6], acc[7]));
        __syncwarp();
        float xr[16];                                                             // X22[r2][0..15]
#pragma unroll
        for (int k4 = 0; k4 < 4; ++k4) {
            const float4 f = lds_f4(aL + (16 + r2) * S + (16 + 4 * k4) * 4);
            xr[4 * k4] = f.x; xr[4 * k4 + 1] = f.y; xr[4 * k4 + 2] = f.z; xr[4 * k4 + 3] = f.w;
        }
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = 0.f;
#pragma unroll
        for (int k = 0; k < 16; ++k) {
            const float4 b0 = lds_f4(aL + (16 + k) * S + cc0 * 4);                // M1[k][cc0 ..]
            const float4 b1 = lds_f4(aL + (16 + k) * S + (cc0 + 4) * 4);
            const float a = xr[k];
            acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
            acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
        }
        __syncwarp();                                                             // every M1 has been read
        sts_f4(aL + (16 + r2) * S + cc0 * 4, make_float4(-acc[0], -acc[1], -acc[2], -acc[3]));
        sts_f4(aL + (16 + r2) * S + (cc0 + 4) * 4, make_float4(-acc[4], -acc[5], -acc[6], -acc[7]));
        sts_f4(aL + r2 * S + (16 + cc0) * 4, make_float4(0.f, 0.f, 0.f, 0.f));    // zeros over L21^T
        sts_f4(aL + r2 * S + (16 + cc0 + 4) * 4, make_float4(0.f, 0.f, 0.f, 0.f));
    }
    __syncthreads();
    {
        // 32 -> 64, all four warps: Y21 = -Y22 (L21 Y11), Y11 = M[0:32][0:32], Y22 = M[32:64][32:64] (both clean
        // lower-triangular), L21^T = M[0:32][32:64].  Thread (r, c8): row r of the block, eight columns.
        const int r = tid >> 2, c8 = (tid & 3) * 8;
        float acc[8];
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = 0.f;
#pragma unroll 8
        for (int k = 0; k < 32; ++k) {
            const float a = lds_f32(aX + (k * kLS + 32 + r) * 4);                 // L[32 + r][k]
            const float4 b0 = lds_f4(aX + (k * kLS + c8) * 4);                    // Y11[k][c8 ..] (zero for k < column)
            const float4 b1 = lds_f4(aX + (k * kLS + c8 + 4) * 4);
            acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
            acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
        }
        sts_f4(aX + ((32 + r) * kLS + c8) * 4, make_float4(acc[0], acc[1], acc[2], acc[3]));        // M1 -> lower-left block
        sts_f4(aX + ((32 + r) * kLS + c8 + 4) * 4, make_float4(acc[4], acc[5], acc[6], acc[7]));
        float yr[32];                                                             // Y22[r][0..31] (zero beyond the diagonal)
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            const float4 f = lds_f4(aX + ((32 + r) * kLS + 32 + 4 * k4) * 4);
            yr[4 * k4] = f.x; yr[4 * k4 + 1] = f.y; yr[4 * k4 + 2] = f.z; yr[4 * k4 + 3] = f.w;
        }
        __syncthreads();
#pragma unroll
        for (int e = 0; e < 8; ++e) acc[e] = 0.f;
#pragma unroll
        for (int k = 0; k < 32; ++k) {
            const float4 b0 = lds_f4(aX + ((32 + k) * kLS + c8) * 4);             // M1[k][c8 ..]
            const float4 b1 = lds_f4(aX + ((32 + k) * kLS + c8 + 4) * 4);
            const float a = yr[k];
            acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
            acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
        }
        __syncthreads();                                                          // every M1 has been read
        sts_f4(aX + ((32 + r) * kLS + c8) * 4, make_float4(-acc[0], -acc[1], -acc[2], -acc[3]));
        sts_f4(aX + ((32 + r) * kLS + c8 + 4) * 4, make_float4(-acc[4], -acc[5], -acc[6], -acc[7]));
    }
    __syncthreads();
    // ---- the two scaled copies of Tm, stacked as ONE K-major A operand [128][64] written over the scratch:
    //      rows 0-63 = Tm diag(beta gamma) (thread half 0), rows 64-127 = Tm diag(beta) (half 1) ----
    {
        const uint32_t vec = (tid < 64) ? aBG : aBeta;
        uint32_t pk[32];
#pragma unroll
        for (int q = 0; q < 16; ++q) {
            const float4 f = lds_f4(aX + (i * kLS + 4 * q) * 4);                  // Tm[i][4q ..]; above the diagonal: L^T leftovers
            const float4 s = lds_f4(vec + 16 * q);
            const float v0 = (4 * q + 0 <= i) ? f.x * s.x : 0.f, v1 = (4 * q + 1 <= i) ? f.y * s.y : 0.f;
            const float v2 = (4 * q + 2 <= i) ? f.z * s.z : 0.f, v3 = (4 * q + 3 <= i) ? f.w * s.w : 0.f;
            pk[2 * q] = pack_bf16(v0, v1); pk[2 * q + 1] = pack_bf16(v2, v3);
        }
        __syncthreads();                                                          // the scratch has been read by everyone
#pragma unroll
        for (int c = 0; c < 8; ++c) st_shared_v4(aX + swz_chunk_off(row, c, 0), pk[4 * c], pk[4 * c + 1], pk[4 * c + 2], pk[4 * c + 3]);
    }
    sync_then_issue();

    // ---- S3: [Tm diag(beta gamma) ; Tm diag(beta)] [K | V] -> TMEM columns 0..127 ----
    if (tid == 0) {
        mbar_wait(bar_v, par);
        tc_fence_after();
        const uint32_t id = umma_idesc(128, 128, false, true);
#pragma unroll
        for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aX + s * 32), desc_mnmajor(aK + s * 2048, OFF_V - OFF_K), id, s > 0);
        umma_commit(bar_mma);
    }
    wait_mma();
    {
        // lanes 0-63: W = columns 0..63 -> block 0 of [W | Ut]; lanes 64-127: Ut = columns 64..127 -> block 1
        float v[64];
        tmem_ld64(tmem_addr(tmem, lane_base, tid < 64 ? 0 : 64), v);
        const uint32_t dst = aX + (tid < 64 ? 0u : kTile);
#pragma unroll
        for (int c = 0; c < 8; ++c)
            st_shared_v4(dst + swz_chunk_off(i, c, 0), pack_bf16(v[8 * c], v[8 * c + 1]), pack_bf16(v[8 * c + 2], v[8 * c + 3]),
                         pack_bf16(v[8 * c + 4], v[8 * c + 5]), pack_bf16(v[8 * c + 6], v[8 * c + 7]));
        // Kt = diag(gamma_C / gamma) K in place (S3 was the last reader of K as it is)
        const int j = tid >> 1, c0 = (tid & 1) * 4;
        const float ks = lds_f32(aKS + j * 4);
#pragma unroll
        for (int c = c0; c < c0 + 4; ++c) {
            const uint32_t addr = aK + swz_chunk_off(j, c, 0);
            float f[8];
            unpack8(ld_shared_v4(addr), f);
            st_shared_v4(addr, pack_bf16(f[0] * ks, f[1] * ks), pack_bf16(f[2] * ks, f[3] * ks), pack_bf16(f[4] * ks, f[5] * ks), pack_bf16(f[6] * ks, f[7] * ks));
        }
    }
    sync_then_issue();

    // ---- S4: [Kt | P^T]^T [W | Ut] -> lanes 0-63: [G | N] rows, lanes 64-127: [P W | P Ut] rows ----
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, 128, true, true);
#pragma unroll
        for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_mnmajor(aK + s * 2048, OFF_PT - OFF_K), desc_mnmajor(aX + s * 2048, kTile), id, s > 0);
        umma_commit(bar_mma);
    }
    wait_mma();
    if (tid < 64) {
        // summary row m = tid: G bf16 -> the P^T buffer, N fp32 as two [64][32] blocks -> the scratch (both operands are dead)
        const int m = tid;
        float v[64];
        tmem_ld64(tmem_addr(tmem, lane_base, 0), v);
#pragma unroll
        for (int c = 0; c < 8; ++c)
            st_shared_v4(aPT + swz_chunk_off(m, c, 0), pack_bf16(v[8 * c], v[8 * c + 1]), pack_bf16(v[8 * c + 2], v[8 * c + 3]),
                         pack_bf16(v[8 * c + 4], v[8 * c + 5]), pack_bf16(v[8 * c + 6], v[8 * c + 7]));
        tmem_ld64(tmem_addr(tmem, lane_base, 64), v);
#pragma unroll
        for (int cc = 0; cc < 2; ++cc)
#pragma unroll
            for (int q = 0; q < 8; ++q)
                st_shared_v4(aX + cc * kTile + (uint32_t)m * 128u + (uint32_t)((q ^ (m & 7)) << 4), __float_as_uint(v[cc * 32 + 4 * q]),
                             __float_as_uint(v[cc * 32 + 4 * q + 1]), __float_as_uint(v[cc * 32 + 4 * q + 2]), __float_as_uint(v[cc * 32 + 4 * q + 3]));
    } else {
        // token row i: Qt = gamma_i Q - P W in place, Ol = P Ut over V
        const float gamma_i = fast_exp(gam_i);
#pragma unroll
        for (int hc = 0; hc < 2; ++hc) {
            float pw[32], pu[32];
            tmem_ld32(tmem_addr(tmem, lane_base, hc * 32), pw);
            tmem_ld32(tmem_addr(tmem, lane_base, 64 + hc * 32), pu);
#pragma unroll
            for (int c = 0; c < 4; ++c) {
                const uint32_t off = swz_chunk_off(i, hc * 4 + c, 0);
                float f[8];
                unpack8(ld_shared_v4(aQ + off), f);
#pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = gamma_i * f[e] - pw[8 * c + e];
                st_shared_v4(aQ + off, pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
                st_shared_v4(aV + off, pack_bf16(pu[8 * c], pu[8 * c + 1]), pack_bf16(pu[8 * c + 2], pu[8 * c + 3]),
                             pack_bf16(pu[8 * c + 4], pu[8 * c + 5]), pack_bf16(pu[8 * c + 6], pu[8 * c + 7]));
            }
        }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
        const int r0 = (int)((long long)bh * p.NT * 128 + (long long)chunk * 64);
        const int z = bh * p.NC + chunk;
        tma_store_2d(mp.tmQt, smem + OFF_Q, 0, r0);
        tma_store_2d(mp.tmOl, smem + OFF_V, 0, r0);
        tma_store_3d(mp.tmG, smem + OFF_PT, 0, 0, z);
        tma_store_3d(mp.tmN, smem + OFF_X, 0, 0, z);
        tma_store_3d(mp.tmN, smem + OFF_X + kTile, 32, 0, z);
        tma_store_commit();
        p.gam[(long long)bh * p.NC + chunk] = fast_exp(gam_C);
    }
}

// One CTA per 64-token chunk; four CTAs are resident per SM.
__global__ void __launch_bounds__(kThreads, 4)
gdn_tok_tile64(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
               const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmQt,
               const __grid_constant__ CUtensorMap tmOl, const TokParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + OFF_BAR);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 4);
    if (threadIdx.x == 0) {
        for (int s = 0; s < 4; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    if (threadIdx.x < 32) tmem_alloc(tmem_slot, 128);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_launch_dependents();
    Tile64Maps mp{&tmQ, &tmK, &tmV, &tmG, &tmN, &tmQt, &tmOl};
    tile64(smem, tmem, bars, mp, p, (int)blockIdx.x / p.NC, (int)blockIdx.x % p.NC, 0u);
    if (threadIdx.x == 0) tma_store_wait_all();
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(tmem, 128);
}

}  // namespace t64
}  // namespace gdn
