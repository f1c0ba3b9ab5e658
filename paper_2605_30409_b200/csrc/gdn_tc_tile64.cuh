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
//         warps 0-1: decay-masked L -> bf16 rows + fp32 diagonal 16-blocks; warps 2-3: decay-masked P -> P^T (bf16)
//         (I + L)^-1 of the 64x64 block: diagonal 16-blocks by fp32 forward substitution on CUDA cores, 16 -> 32 -> 64 by
//         X21 = -X22 (L21 X11) with warp-level mma.sync on the bf16 blocks (no asynchronous TMEM round trips)
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
constexpr uint32_t kTile = 8192;                      // one [64][64] bf16 tile (128-byte rows, 128-byte swizzle)
constexpr uint32_t OFF_K = 0;                         // K tile  } the stacked K-major A operand of S1; K alone is its B operand
constexpr uint32_t OFF_Q = 8192;                      // Q tile  }   later: Kt in place / Qt in place
constexpr uint32_t OFF_V = 16384;                     // V tile; later Ol
constexpr uint32_t OFF_PT = 24576;                    // P^T [j][i] bf16; later the staging of G
constexpr uint32_t OFF_X = 32768;                     // L_bf | D_bf (bf16 [64][64] each) | fp32 diagonal 16-blocks (4 KB)
                                                      //   -> [Tm diag(beta gamma) ; Tm diag(beta)] bf16 [128][64]
                                                      //   -> [W | Ut] bf16 2 x [64][64] -> staging of N
constexpr uint32_t X_BYTES = 2 * kTile + 4096;
constexpr uint32_t OFF_VEC = OFF_X + X_BYTES;         // Gam[64], Beta[64], BG[64], KS[64], CF[32]
constexpr uint32_t OFF_RAW = OFF_VEC + 1280;              // 2 x {alpha[64], beta[64]} of the next chunk, copied ahead (persistent workers)
constexpr uint32_t OFF_BAR = OFF_RAW + 1024;
constexpr uint32_t SMEM_BYTES = OFF_BAR + 64 + 1024;  // + slack for the 1024-byte alignment of the dynamic base

struct Tile64Maps {
    const CUtensorMap *tmQ, *tmK, *tmV;               // activations, box [64 tokens][64 features]
    const CUtensorMap *tmG, *tmN;                     // G bf16 box {64, 64, 1}; N fp32 box {32, 64, 1} (NBF16: bf16 like G)
    const CUtensorMap *tmQt, *tmOl;                   // workspace rows, box {64, 64}
    int zG, zN;                                       // first summary slot of G / N in their maps
    long long rows_per_bh;                            // Qt / Ol rows per stream
    long long rQt, rOl;                               // first row of Qt / Ol in their maps
};


// One 64-token chunk `chunk` of stream `bh`.  smem: 1024-byte aligned base; tmem: 128 columns; bars: 4 mbarriers
// (K+Q landed, V landed, MMA complete, spare) initialised to count 1; `pl` / `ph` = running parities of the two load
// barriers (both complete one phase per chunk) and of the MMA barrier, kept by the caller across tasks.
template <bool NBF16>
__device__ __forceinline__ void tile64(uint8_t* smem, uint32_t tmem, uint64_t* bars, const Tile64Maps& mp, const TokParams& p,
                                       int bh, int chunk, uint32_t& pl, uint32_t& ph, uint32_t pre_gates = 0u,
                                       unsigned long long* pend_flag = nullptr, unsigned long long pend_val = 0ull, float* gamma_out = nullptr) {
    // pre_gates: shared-space address of {alpha[64], beta[64]} of the chunk, copied ahead by the caller (0: read them
    // here).  pend_flag / pend_val: a flag word of the caller's previous task, released by thread 0 once that task's bulk stores have completed (behind this chunk's first MMA issue, where the wait costs nothing).  gamma_out:
    // receives gamma_C (thread 0) instead of p.gam.
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int b = bh / p.H, h = bh % p.H;
    const uint32_t aK = smem_u32(smem + OFF_K), aQ = smem_u32(smem + OFF_Q), aV = smem_u32(smem + OFF_V);
    const uint32_t aPT = smem_u32(smem + OFF_PT), aX = smem_u32(smem + OFF_X), aVec = smem_u32(smem + OFF_VEC);
    const uint32_t aGam = aVec, aBeta = aVec + 256, aBG = aVec + 512, aKS = aVec + 768, aCF = aVec + 1024;
    uint64_t *bar_kq = &bars[0], *bar_v = &bars[1], *bar_mma = &bars[2];
    const uint32_t par = pl;
    pl ^= 1u;
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
        if (pre_gates) { a0 = lds_f32(pre_gates + lane * 4); a1 = lds_f32(pre_gates + (32 + lane) * 4); b0 = lds_f32(pre_gates + (64 + lane) * 4); b1 = lds_f32(pre_gates + (96 + lane) * 4); }
        else {
            if (t0 < p.T) { a0 = p.alpha[(long long)bh * p.T + t0]; b0 = p.beta[(long long)bh * p.T + t0]; }
            if (t1 < p.T) { a1 = p.alpha[(long long)bh * p.T + t1]; b1 = p.beta[(long long)bh * p.T + t1]; }
        }
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
        if (pend_flag) {
            tma_store_wait_all();
            asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(pend_flag), "l"(pend_val) : "memory");
        }
    }
    wait_mma();

    // ---- S1 epilogue.  warps 0-1 (row i of K K^T): L_ij = beta_i e^{Gam_i-Gam_j} k_i.k_j (j < i) -> bf16 row of L_bf, and
    //      its diagonal 16-block TRANSPOSED in fp32 -> scratch (for the forward substitution); warps 2-3 (row i of Q K^T):
    //      P_ij = e^{Gam_i-Gam_j} q_i.k_j (j <= i) -> bf16 P^T[j][i].  Inside a 32-column block the exponent is taken
    //      directly; across blocks e^{Gam_i-Gam_j} = e^{Gam_i-Gam_31} e^{Gam_31-Gam_j} (both factors <= 1).
    const uint32_t aLB = aX, aDB = aX + kTile, aSC = aX + 2 * kTile;
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
                if (is_l) continue;                   // L above the diagonal blocks is never read
#pragma unroll
                for (int j = 0; j < 32; ++j) v[j] = 0.f;
            }
            if (is_l) {
                store_row32_bf16(aLB, 0, i, 32 * hc, v);
                if (hc == ci) {
                    // diagonal 16-block (i >> 4): Lt[jl][i & 15] = L[i][16 (i >> 4) + jl]
                    const uint32_t dst = aSC + (uint32_t)(i >> 4) * 1024u + (uint32_t)(i & 15) * 4u;
                    const bool hi = (lane & 16) != 0;
#pragma unroll
                    for (int jl = 0; jl < 16; ++jl) sts_f32(dst + jl * 64, hi ? v[16 + jl] : v[jl]);
                }
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

    // ---- Tm = (I + L)^-1 -> D_bf (bf16, swizzled rows).  Diagonal 16-blocks: fp32 forward substitution on CUDA cores
    //      (tok::inv16_columns, one column per lane).  16 -> 32 -> 64: X21 = -X22 (L21 X11) with warp-level mma.sync on
    //      the bf16 blocks: these products are 16^3 / 32^3, far below the M >= 64 tile of tcgen05.mma and not worth an
    //      asynchronous TMEM round trip each; the transposed first product (L21 X11)^T = X11^T L21^T leaves its fp32
    //      accumulator fragments in exactly the layout of the second product's B fragments, so nothing goes through memory.
    const int qm = lane >> 3, rr = lane & 7;          // ldmatrix: this lane addresses row rr of matrix qm
    const int g8 = lane >> 2, c2 = (lane & 3) * 2;    // mma fragments: row g8, column pair c2
    auto tile_addr = [](uint32_t base, int r, int chunk) { return base + (uint32_t)r * 128u + (uint32_t)((chunk ^ (r & 7)) << 4); };
    if (warp < 2) {
        __syncwarp();
        {
            const int bi = 2 * warp + (lane >> 4), col = lane & 15;
            float xc[16];
            tok::inv16_columns<16>(aSC + (uint32_t)bi * 1024u, col, xc);
            const int cg = 16 * bi + col;             // column of D_bf
#pragma unroll
            for (int r = 0; r < 16; ++r) {
                const int R = 16 * bi + r;
                sts_b16(tile_addr(aDB, R, cg >> 3) + (uint32_t)(cg & 7) * 2u, __bfloat16_as_ushort(__float2bfloat16_rn(xc[r])));
            }
            // zeros above the 16-blocks inside this warp's 32-block: rows 32w .. 32w+15, columns 32w+16 .. 32w+31
            st_shared_v4(tile_addr(aDB, 32 * warp + (lane >> 1), 4 * warp + 2 + (lane & 1)), 0u, 0u, 0u, 0u);
        }
        __syncwarp();
        const int b0 = 32 * warp;
        uint32_t a[4], bb[4], a2[4];
        ldsm_x4_trans(a, tile_addr(aDB, b0 + (qm >> 1) * 8 + rr, 4 * warp + (qm & 1)));              // X00^T
        ldsm_x4(bb, tile_addr(aLB, b0 + 16 + (qm >> 1) * 8 + rr, 4 * warp + (qm & 1)));              // L10^T as [n][k]
        ldsm_x4(a2, tile_addr(aDB, b0 + 16 + (qm & 1) * 8 + rr, 4 * warp + 2 + (qm >> 1)));          // X11
        float t0[4] = {0.f, 0.f, 0.f, 0.f}, t1[4] = {0.f, 0.f, 0.f, 0.f};
        mma_bf16_16816(t0, a, bb[0], bb[1]);
        mma_bf16_16816(t1, a, bb[2], bb[3]);
        float y0[4] = {0.f, 0.f, 0.f, 0.f}, y1[4] = {0.f, 0.f, 0.f, 0.f};
        mma_bf16_16816(y0, a2, pack_bf16(t0[0], t0[1]), pack_bf16(t1[0], t1[1]));
        mma_bf16_16816(y1, a2, pack_bf16(t0[2], t0[3]), pack_bf16(t1[2], t1[3]));
        // X10 = -Y: rows b0+16+g8 (+8), columns b0 + 8 j2 + c2
#pragma unroll
        for (int j2 = 0; j2 < 2; ++j2) {
            const float* y = j2 ? y1 : y0;
            const int C = b0 + 8 * j2 + c2;
            const int R0 = b0 + 16 + g8, R1 = R0 + 8;
            sts_b32(tile_addr(aDB, R0, C >> 3) + (uint32_t)(C & 7) * 2u, pack_bf16(-y[0], -y[1]));
            sts_b32(tile_addr(aDB, R1, C >> 3) + (uint32_t)(C & 7) * 2u, pack_bf16(-y[2], -y[3]));
        }
    }
    __syncthreads();
    {
        // 32 -> 64, all four warps: warp (mt, m2) = (warp & 1, warp >> 1) produces Y21[16 m2 .. +15][16 mt .. +15],
        // Y21 = -Y22 (L21 Y11), Y11 = D_bf[0:32][0:32], Y22 = D_bf[32:64][32:64], L21 = L_bf[32:64][0:32].
        const int mt = warp & 1, m2 = warp >> 1;
        float t[4][4];
#pragma unroll
        for (int n = 0; n < 4; ++n)
#pragma unroll
            for (int e = 0; e < 4; ++e) t[n][e] = 0.f;
#pragma unroll
        for (int ks = 0; ks < 2; ++ks) {
            uint32_t a[4];
            ldsm_x4_trans(a, tile_addr(aDB, 16 * ks + (qm >> 1) * 8 + rr, 2 * mt + (qm & 1)));       // Y11^T, rows c of tile mt
#pragma unroll
            for (int np = 0; np < 2; ++np) {
                uint32_t bb[4];
                ldsm_x4(bb, tile_addr(aLB, 32 + 16 * np + (qm >> 1) * 8 + rr, 2 * ks + (qm & 1)));   // L21^T as [n = r][k]
                mma_bf16_16816(t[2 * np], a, bb[0], bb[1]);
                mma_bf16_16816(t[2 * np + 1], a, bb[2], bb[3]);
            }
        }
        float y[2][4];
#pragma unroll
        for (int j2 = 0; j2 < 2; ++j2)
#pragma unroll
            for (int e = 0; e < 4; ++e) y[j2][e] = 0.f;
#pragma unroll
        for (int ks2 = 0; ks2 < 2; ++ks2) {
            uint32_t a2[4];
            ldsm_x4(a2, tile_addr(aDB, 32 + 16 * m2 + (qm & 1) * 8 + rr, 4 + 2 * ks2 + (qm >> 1)));  // Y22 rows of tile m2
            mma_bf16_16816(y[0], a2, pack_bf16(t[2 * ks2][0], t[2 * ks2][1]), pack_bf16(t[2 * ks2 + 1][0], t[2 * ks2 + 1][1]));
            mma_bf16_16816(y[1], a2, pack_bf16(t[2 * ks2][2], t[2 * ks2][3]), pack_bf16(t[2 * ks2 + 1][2], t[2 * ks2 + 1][3]));
        }
#pragma unroll
        for (int j2 = 0; j2 < 2; ++j2) {
            const int C = 16 * mt + 8 * j2 + c2;
            const int R0 = 32 + 16 * m2 + g8, R1 = R0 + 8;
            sts_b32(tile_addr(aDB, R0, C >> 3) + (uint32_t)(C & 7) * 2u, pack_bf16(-y[j2][0], -y[j2][1]));
            sts_b32(tile_addr(aDB, R1, C >> 3) + (uint32_t)(C & 7) * 2u, pack_bf16(-y[j2][2], -y[j2][3]));
        }
    }
    __syncthreads();
    // ---- the two scaled copies of Tm, stacked as ONE K-major A operand [128][64] written over L_bf / D_bf:
    //      rows 0-63 = Tm diag(beta gamma) (thread half 0), rows 64-127 = Tm diag(beta) (half 1).  Columns 32..63 of
    //      the rows below 32 were never written: zero.
    {
        const uint32_t vec = (tid < 64) ? aBG : aBeta;
        const int nch = (i < 32) ? 4 : 8;             // warp-uniform
        uint32_t pk[32];
#pragma unroll
        for (int c = 0; c < 8; ++c) {
            if (c < nch) {
                float f[8];
                unpack8(ld_shared_v4(tile_addr(aDB, i, c)), f);
                const float4 s0 = lds_f4(vec + 32 * c), s1 = lds_f4(vec + 32 * c + 16);
                pk[4 * c] = pack_bf16(f[0] * s0.x, f[1] * s0.y); pk[4 * c + 1] = pack_bf16(f[2] * s0.z, f[3] * s0.w);
                pk[4 * c + 2] = pack_bf16(f[4] * s1.x, f[5] * s1.y); pk[4 * c + 3] = pack_bf16(f[6] * s1.z, f[7] * s1.w);
            } else {
                pk[4 * c] = pk[4 * c + 1] = pk[4 * c + 2] = pk[4 * c + 3] = 0u;
            }
        }
        __syncthreads();                                                          // D_bf has been read by everyone
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
        if (NBF16) {
#pragma unroll
            for (int c = 0; c < 8; ++c)
                st_shared_v4(aX + swz_chunk_off(m, c, 0), pack_bf16(v[8 * c], v[8 * c + 1]), pack_bf16(v[8 * c + 2], v[8 * c + 3]),
                             pack_bf16(v[8 * c + 4], v[8 * c + 5]), pack_bf16(v[8 * c + 6], v[8 * c + 7]));
        } else {
#pragma unroll
            for (int cc = 0; cc < 2; ++cc)
#pragma unroll
                for (int q = 0; q < 8; ++q)
                    st_shared_v4(aX + cc * kTile + (uint32_t)m * 128u + (uint32_t)((q ^ (m & 7)) << 4), __float_as_uint(v[cc * 32 + 4 * q]),
                                 __float_as_uint(v[cc * 32 + 4 * q + 1]), __float_as_uint(v[cc * 32 + 4 * q + 2]), __float_as_uint(v[cc * 32 + 4 * q + 3]));
        }
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
        const long long r0 = (long long)bh * mp.rows_per_bh + (long long)chunk * 64;
        const int z = bh * p.NC + chunk;
        tma_store_2d(mp.tmQt, smem + OFF_Q, 0, (int)(mp.rQt + r0));
        tma_store_2d(mp.tmOl, smem + OFF_V, 0, (int)(mp.rOl + r0));
        tma_store_3d(mp.tmG, smem + OFF_PT, 0, 0, mp.zG + z);
        tma_store_3d(mp.tmN, smem + OFF_X, 0, 0, mp.zN + z);
        if (!NBF16) tma_store_3d(mp.tmN, smem + OFF_X + kTile, 32, 0, mp.zN + z);
        tma_store_commit();
        if (gamma_out) *gamma_out = fast_exp(gam_C);
        else p.gam[(long long)bh * p.NC + chunk] = fast_exp(gam_C);
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
    Tile64Maps mp{&tmQ, &tmK, &tmV, &tmG, &tmN, &tmQt, &tmOl, 0, 0, (long long)p.NT * 128, 0, 0};
    uint32_t pl = 0, ph = 0;
    tile64<false>(smem, tmem, bars, mp, p, (int)blockIdx.x / p.NC, (int)blockIdx.x % p.NC, pl, ph);
    if (threadIdx.x == 0) tma_store_wait_all();
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(tmem, 128);
}

}  // namespace t64
}  // namespace gdn
