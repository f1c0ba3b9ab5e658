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
    int NSc;                     // snapshot slots per (b,h) in Sc: NC (token-wise) or NC + 1 (frame-wise: also the final state)
    // chain kernel only.  NCa = entries per (b,h) in Gw / Nw / gam (= NC except for the reverse scan of the bidirectional
    // frame path, Alg. 1 l.14-17: rev = 1 runs NC = NCa - 1 steps over the entries NCa-1, NCa-2, ..., 1 from a zero
    // state and stores the state BEFORE entry e is applied (= S<_e) in snapshot slot e; S_out may be NULL).
    int NCa, rev;
    int dr;                      // real state dimension: D, or 112 when the head dim is zero-padded to D = 128 (Alg. 1 l.1); the
                                 // user's state / z tensors are [dr][dr] / [dr], everything inside the library is [D][D]
    // chain kernel, normaliser z pass: the state is a vector living in column 0 of the matrix state.  z_vec_in [BH][D] (or
    // NULL = zeros) initialises it instead of S_in, z_vec_out [BH][D] receives it instead of S_out (either may be NULL).
    int zvec;
    const float* z_vec_in;
    float* z_vec_out;
    int col_tiles;               // chain kernel: 64-column tiles of the state that are run (0 = all D / 64; the z pass runs tile 0 only)
    long long o_ts;              // out token stride (elements)
    float scale;
    int log_alpha;
    // chain kernel, bidirectional frame path (Alg. 1 l.19-21): S^hist_f = S>_f + S<_f.  snap_add = 1: both scans ADD their
    // snapshots (slots > 0) into the forward snapshot array by TMA reduction; Phase A has zeroed the slots, 0 + a is exact, so the
    // sum takes one bf16 rounding whichever scan lands first (deterministic), and nothing has to wait for anything.  The reverse
    // scan's S<_e joins slot e + 1 (snap_off = 1) of an array with snap_stride slots per (b,h) (0 = NSc).
    int snap_add, snap_off, snap_stride;
};


namespace tok {

using namespace tc;

constexpr uint32_t kBlk = 16384;      // one [128][64] bf16 block

__device__ __forceinline__ void st_global_v4(void* p, uint32_t a, uint32_t b, uint32_t c, uint32_t d) {
    asm volatile("st.global.v4.b32 [%0], {%1, %2, %3, %4};" ::"l"(p), "r"(a), "r"(b), "r"(c), "r"(d) : "memory");
}

// ---------------------------------------------------------------------------------------------------
// Kernel 1: prepass.  grid = BH * NT, block = 128 * NH threads (NH warps per TMEM lane quadrant).
//   Thread (row, hh): row = 32*(warp&3) + lane is the token row / TMEM lane; hh = warp>>2 picks which
//   CW = 32/NH columns of every 32-column chunk the thread handles, so each scheduler has NH warps to
//   interleave across the many short dependent phases.  Thread 0 issues TMA and tcgen05.mma.
// ---------------------------------------------------------------------------------------------------
constexpr int kPrepassNH = 4;
constexpr int kPrepassThreads = 128 * kPrepassNH;
constexpr int kPrepassFlagTid = 128;   // lane 0 of a warp that idles during the diagonal-block inversion (FUSED: releases the ready flags)

// The diagonal 32x32 blocks of I + L are inverted on CUDA cores, one warp per block, no shuffles.  Lt holds L TRANSPOSED
// (Lt[j*kLsStride + r] = L[r][j]) so that "column j of L" is a row of 16-byte loads.  Blocked in 16s:
// L = [[L11, 0], [L21, L22]]  ->  X = [[X11, 0], [-X22 L21 X11, X22]]; X11, X22 by right-looking forward substitution
// (once x_j is final every later row takes x_r -= L[r][j] x_j: the serial depth is 15 FMAs), the off-diagonal block by
// two register-tiled 16x16x16 products.
constexpr int kLsStride = 36;                     // floats per row: 16-byte aligned, conflict-free
// 16x16 unit-lower-triangular inverse: Lt[j*kLsStride + r] = L[r][j] (r, j < 16), the calling lane owns column `col` of
// X = (I + L)^-1.  Two of these (the two diagonal 16-blocks of a 32-block) run in the two halves of one warp with
// different base pointers.
template <int J, int LS>
__device__ __forceinline__ void inv16_load_row(uint32_t Lt, float4 (&l)[4]) {
#pragma unroll
    for (int r4 = (J + 1) / 4; r4 < 4; ++r4) l[r4] = lds_f4(Lt + (J * LS + 4 * r4) * 4);
}
template <int J>
__device__ __forceinline__ void inv16_apply_row(const float4 (&l)[4], float (&x)[16]) {
    const float xj = x[J];
#pragma unroll
    for (int r4 = (J + 1) / 4; r4 < 4; ++r4) {
        if (4 * r4 + 0 > J) x[4 * r4 + 0] = fmaf(-l[r4].x, xj, x[4 * r4 + 0]);
        if (4 * r4 + 1 > J) x[4 * r4 + 1] = fmaf(-l[r4].y, xj, x[4 * r4 + 1]);
        if (4 * r4 + 2 > J) x[4 * r4 + 2] = fmaf(-l[r4].z, xj, x[4 * r4 + 2]);
        if (4 * r4 + 3 > J) x[4 * r4 + 3] = fmaf(-l[r4].w, xj, x[4 * r4 + 3]);
    }
}
template <int J, int LS>
__device__ __forceinline__ void inv16_steps(uint32_t Lt, float4 (&cur)[4], float4 (&nxt)[4], float (&x)[16]) {
    if constexpr (J < 15) {
        if constexpr (J + 1 < 15) inv16_load_row<J + 1, LS>(Lt, nxt);
        inv16_apply_row<J>(cur, x);
        inv16_steps<J + 1, LS>(Lt, nxt, cur, x);
    }
}
// Lt = shared-space byte address of the block's L^T, LS = floats per scratch row
template <int LS = kLsStride>
__device__ __forceinline__ void inv16_columns(uint32_t Lt, int col, float (&x)[16]) {
#pragma unroll
    for (int r = 0; r < 16; ++r) x[r] = (r == col) ? 1.f : 0.f;
    float4 la[4], lb[4];
    inv16_load_row<0, LS>(Lt, la);
    inv16_steps<0, LS>(Lt, la, lb, x);
}

// Shared-memory carve-up and barriers of one prepass CTA (set up once; a persistent CTA runs many tiles).
struct PrepassCtx {
    uint8_t *sK, *sQ, *sV, *sA, *sB, *sC;
    float *sGam, *sBeta, *sBG, *sCF, *sWarp, *sL;
    uint64_t *bar_kq, *bar_q, *bar_v, *bar_mma;    // bar_kq: K tile landed; bar_q: Q tile; bar_v: V tile
    uint64_t* bar_mma2;                           // C = 128: the [N | G] summary MMAs (committed behind [P Ut | P W], which bar_mma covers)
    uint32_t tmem;                                // 512 TMEM columns
};
template <int D>
constexpr uint32_t prepass_smem_bytes() { return 3u * (D / 64) * kBlk + 6u * kBlk + 4u * 32 * kLsStride * 4 + 4096u; }

template <int D>
__device__ __forceinline__ void prepass_carve(uint8_t* smem, PrepassCtx& cx, uint32_t** tmem_slot) {
    constexpr uint32_t TILE = (D / 64) * kBlk;
    cx.sK = smem;
    cx.sQ = smem + TILE;
    cx.sV = smem + 2 * TILE;
    cx.sA = smem + 3 * TILE;                      // L_off -> Tm diag(beta gamma) -> Ut
    cx.sB = cx.sA + 2 * kBlk;                     // D (block-diagonal inverse) -> W      (sB directly follows sA)
    cx.sC = cx.sB + 2 * kBlk;                     // X -> Tm diag(beta) -> P
    cx.sL = reinterpret_cast<float*>(cx.sC + 2 * kBlk);        // diagonal 32x32 blocks of L^T (fp32), then of the inverse
    cx.sGam = cx.sL + 4 * 32 * kLsStride;         // [128] Gam_i (segmented for C = 64)
    cx.sBeta = cx.sGam + 128;                     // [128] beta_j
    cx.sBG = cx.sBeta + 128;                      // [128] beta_j e^{Gam_j}
    cx.sCF = cx.sBG + 128;                        // [128] e^{Gam_ref(j) - Gam_j}, ref = last row of j's 32-chunk
    cx.sWarp = cx.sCF + 128;                      // [4] per-warp sums of log alpha
    uint64_t* bars = reinterpret_cast<uint64_t*>(cx.sWarp + 4);
    cx.bar_kq = &bars[0]; cx.bar_v = &bars[1]; cx.bar_mma = &bars[2]; cx.bar_q = &bars[3]; cx.bar_mma2 = &bars[4];
    *tmem_slot = reinterpret_cast<uint32_t*>(bars + 5);
}

// One 128-token tile of one (b,h) stream.  `it` = how many tiles this CTA has run before (barrier parity),
// `ph` = running parity of bar_mma.  FUSED = false: summaries in the layouts of the three-kernel path
// (N row-major fp32 [D][D], Ol row-major [rows][D]), the call returns after the stores have read their
// staging.  FUSED = true (gdn_tc_fused.cuh, C = 128): scale * Ol is stored straight into `out` (tmOl is then
// the map of `out`; the chain workers add scale * Qt S_c to it with a TMA reduction), the stores are left
// draining while the next tile starts, and the tile's ready flag is published from inside the next tile
// once they have completed.
template <int D, int C, bool FUSED>
__device__ __forceinline__ void prepass_tile(const PrepassCtx& cx, const CUtensorMap* tmQ, const CUtensorMap* tmK,
                                             const CUtensorMap* tmV, const CUtensorMap* tmG, const CUtensorMap* tmN,
                                             const CUtensorMap* tmQt, const CUtensorMap* tmOl, const TokParams& p,
                                             int bh, int tile, uint32_t it, uint32_t& ph,
                                             unsigned int* prev_flag = nullptr, unsigned int epoch = 0,
                                             int next_bh = -1, int next_tile = -1, float2* gates = nullptr) {
    static_assert(!FUSED || C == 128, "the fused path runs C = 128");
    constexpr int NH = kPrepassNH;
    constexpr int CW = 32 / NH;                   // columns of each 32-column chunk handled per thread
    constexpr int CH = CW / 8;                    // 16-byte bf16 chunks per thread per 32-column chunk
    constexpr int NB = D / 64;
    constexpr uint32_t TILE = NB * kBlk;
    constexpr int KS = 8;                         // K = 16 steps over the 128 tokens of a tile
    constexpr int DS = D / 16;                    // K = 16 steps over the head dim
    uint8_t *sK = cx.sK, *sQ = cx.sQ, *sV = cx.sV, *sA = cx.sA, *sB = cx.sB, *sC = cx.sC;
    float *sGam = cx.sGam, *sBeta = cx.sBeta, *sBG = cx.sBG, *sCF = cx.sCF, *sWarp = cx.sWarp, *sL = cx.sL;
    uint64_t *bar_kq = cx.bar_kq, *bar_q = cx.bar_q, *bar_v = cx.bar_v, *bar_mma = cx.bar_mma;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int wq = warp & 3, hh = warp >> 2;
    const int row = wq * 32 + lane;               // token row == TMEM lane
    const int cb = hh * CW;                       // this thread's columns inside every 32-column chunk
    const uint32_t lane_base = (uint32_t)(wq * 32);
    const int b = bh / p.H, h = bh % p.H;
    const uint32_t aA = smem_u32(sA), aB = smem_u32(sB), aC = smem_u32(sC), aK = smem_u32(sK), aQ = smem_u32(sQ), aV = smem_u32(sV);
    const uint32_t par = it & 1u;

    // gates first: their global-load latency overlaps the barrier / TMEM / TMA set-up
    // (a persistent CTA passes `gates`: this row's alpha, beta of this tile, fetched during the previous tile)
    auto load_gates = [&](int gbh, int gtile) {
        const int t = gtile * 128 + row;
        float2 r = make_float2(p.log_alpha ? 0.f : 1.f, 0.f);                  // padding rows: alpha = 1, beta = 0
        if (t < p.T) { r.x = p.alpha[(long long)gbh * p.T + t]; r.y = p.beta[(long long)gbh * p.T + t]; }
        return r;
    };
    const float2 gb = (gates && it > 0) ? *gates : load_gates(bh, tile);
    float g = gb.x;
    const float beta_i = gb.y;
    if (tid == 0) {
        if (!FUSED || it == 0) {                   // FUSED, it > 0: the previous tile prefetched this tile's K
            mbar_expect_tx(bar_kq, TILE);
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) tma_load_5d(sK + nb * kBlk, tmK, bar_kq, nb * 64, h, tile * 128, 0, b);
        }
        // Q and V are requested only after the diagonal-block inversions (below): tiles landing in shared memory while
        // the inversions run slow their broadcast loads down by as much as the earlier start would gain.
    }
    // The three 128x128 operand buffers are never pre-zeroed: every phase that fills one writes whole rows
    // (data where the block structure has some, zeros elsewhere) -- see T2 (sA, sB) and the first X1 (sC).

    // ---- T0: in-tile inclusive scan of log alpha (every warp of a quadrant computes it, hh == 0 publishes) ----
    if (!p.log_alpha) g = logf(g);
    float x = g;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const float y = __shfl_up_sync(0xffffffffu, x, o);
        if (lane >= o) x += y;
    }
    if (hh == 0 && lane == 31) sts_f32(smem_u32(sWarp) + wq * 4, x);
    __syncthreads();
    const uint32_t tmem = cx.tmem;
    const uint32_t c0 = tmem, c1 = tmem + 128, c2 = tmem + 256, c3 = tmem + 384;
    float gam_i, gam_end;            // Gam_i and Gam at the end of this row's chunk
    {
        const float4 w4 = lds_f4(smem_u32(sWarp));
        const float w0 = w4.x, w1 = w4.y, w2 = w4.z, w3 = w4.w;
        if (C == 128) {
            gam_i = x + (wq > 0 ? w0 : 0.f) + (wq > 1 ? w1 : 0.f) + (wq > 2 ? w2 : 0.f);
            gam_end = w0 + w1 + w2 + w3;
        } else {
            gam_i = x + ((wq & 1) ? (wq == 1 ? w0 : w2) : 0.f);
            gam_end = wq < 2 ? (w0 + w1) : (w2 + w3);
        }
    }
    const float gam_ref = __shfl_sync(0xffffffffu, gam_i, 31);     // Gam at the last row of this 32-chunk
    if (hh == 0) {
        sts_f32(smem_u32(sGam) + row * 4, gam_i);
        sts_f32(smem_u32(sBeta) + row * 4, beta_i);
        sts_f32(smem_u32(sBG) + row * 4, beta_i * fast_exp(gam_i));
        sts_f32(smem_u32(sCF) + row * 4, fast_exp(gam_ref - gam_i));
    }
    __syncthreads();
    const int half_lo = (C == 128) ? 0 : (wq >> 1) * 2;      // first 32-column chunk of this row's chunk
    // decay factors: e^{Gam_i - Gam_j} = rf[cc] * sCF[j] for j in an earlier 32-chunk cc (both factors <= 1)
    float rf[3];
#pragma unroll
    for (int cc = 0; cc < 3; ++cc) rf[cc] = (cc < wq && cc >= half_lo) ? fast_exp(gam_i - lds_f32(smem_u32(sGam) + (cc * 32 + 31) * 4)) : 0.f;

    auto sync_then_issue = [&]() { fence_proxy_async(); tc_fence_before(); __syncthreads(); };
    auto wait_mma = [&]() { mbar_wait(bar_mma, ph); ph ^= 1; tc_fence_after(); };

    // ---- T1: K K^T -> c0 (Q K^T -> c1 follows in the shadow of the first doubling round trip) ------
    mbar_wait(bar_kq, par);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, 128, false, false);
#pragma unroll
        for (int s = 0; s < DS; ++s) {
            const uint32_t off = (s >> 2) * kBlk + (s & 3) * 32;
            umma_bf16(c0, desc_kmajor(aK + off), desc_kmajor(aK + off), id, s > 0);
        }
        // FUSED: G / N of the previous tile were staged in sA, sB, sC, which T2 overwrites once this commit
        // has been observed -- their reads must have ended first.
        // FUSED: G / N of the previous tile were staged in sA, sB, sC, which T2 overwrites once this commit has been
        // observed -- their reads must have ended first.  Waiting for the WRITES as well costs nothing more here (the
        // stores were issued a scan and an MMA ago) and lets the commit below also stand for "the previous tile's
        // summaries are complete in global memory", so that the ready flag can be released by another thread.
        if (FUSED) tma_store_wait_all();
        umma_commit(bar_mma);
    }
    wait_mma();

    // ---- T2: L (strictly lower, decay-masked) -> sA off-diagonal chunks; diagonal 32x32 block -> Ld ----
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        float v[CW];
        if (cc < 3 && cc < wq && cc >= half_lo) {
            float cf[CW];
            tmem_ldw(tmem_addr(c0, lane_base, cc * 32 + cb), v);
            ld_shared_fw(sCF + cc * 32 + cb, cf);
            const float f = beta_i * rf[cc < 3 ? cc : 0];
#pragma unroll
            for (int e = 0; e < CW; ++e) v[e] *= f * cf[e];
        } else {
#pragma unroll
            for (int e = 0; e < CW; ++e) v[e] = 0.f;
        }
        store_roww_bf16(aA, kBlk, row, cc * 32 + cb, v);
        if (cc != wq) {                            // sB = D: zero outside the diagonal block (written below)
#pragma unroll
            for (int e = 0; e < CW; ++e) v[e] = 0.f;
            store_roww_bf16(aB, kBlk, row, cc * 32 + cb, v);
        }
    }
    if (FUSED && D == 128 && it > 0 && tid == kPrepassFlagTid) tma_store_wait_all();     // this thread's share of the previous tile's stores (sC is not reused before the next CTA barrier)
    if (FUSED && prev_flag && tid == kPrepassFlagTid) {
        // The previous tile's ready flag.  A release at gpu scope takes ~800 cycles (and the fences that used to precede it
        // another ~2000): on tid 0 that sat in front of the first diagonal-block inversion of every tile.  This thread's warp
        // has nothing to do until the inversions are done.  The bulk stores were complete before the K K^T commit was issued
        // (tid 0 above), this thread observed that commit's mbarrier phase, and the release is cumulative.
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(prev_flag), "r"(epoch) : "memory");
    }
    float X[CW];                                   // this thread's columns of row `lane` of (I + Ld)^-1
    {
        // diagonal 32x32 block: ONE warp per quadrant reads it from TMEM (TMEM reads are the scarce
        // resource), masks it, shares it through shared memory and inverts it column-wise.
        float* Lq = sL + wq * 32 * kLsStride;
        if (hh == 0) {
            float v0[16], v1[16], g0[16], g1[16];
            tmem_ld16x2(tmem_addr(c0, lane_base, wq * 32), tmem_addr(c0, lane_base, wq * 32 + 16), v0, v1);
            ld_shared_f16(sGam + wq * 32, g0);
            ld_shared_f16(sGam + wq * 32 + 16, g1);
#pragma unroll
            for (int e = 0; e < 16; ++e) {
                // branch-free: clamp the exponent (rows above the diagonal would be > 0), then select
                const float m0 = (e < lane) ? beta_i : 0.f, m1 = (16 + e < lane) ? beta_i : 0.f;
                v0[e] *= m0 * fast_exp(fminf(gam_i - g0[e], 0.f));
                v1[e] *= m1 * fast_exp(fminf(gam_i - g1[e], 0.f));
            }
            // L^T into the scratch: element (r = lane, j) -> Lq[j][r]   (aL: shared-space byte address of Lq, S = row stride)
            const uint32_t aL = smem_u32(Lq);
            constexpr uint32_t S = kLsStride * 4;
#pragma unroll
            for (int e = 0; e < 16; ++e) { sts_f32(aL + e * S + lane * 4, v0[e]); sts_f32(aL + (16 + e) * S + lane * 4, v1[e]); }
            __syncwarp();
            // Blocked: L = [[L11, 0], [L21, L22]] in 16-blocks, X = [[X11, 0], [-X22 L21 X11, X22]].
            // Step 1 (this warp): lanes 0-15 invert I + L11, lanes 16-31 invert I + L22, each lane one column.
            const int o = lane & 16, col = lane & 15;
            float xc[16];
            inv16_columns(aL + o * S + o * 4, col, xc);
            __syncwarp();
            // X11 / X22 row-major over L11^T / L22^T (consumed): element (r, col) -> Lq[o + r][o + col]
#pragma unroll
            for (int r = 0; r < 16; ++r) sts_f32(aL + (o + r) * S + (o + col) * 4, xc[r]);
            __syncwarp();
            // Steps 2a, 2b (same warp, lane = row r2 x 8 columns): M = L21 X11 into the free block Lq[16 + r][c] (L^T has
            // nothing there), then X21 = -X22 M in its place, and zeros over L21^T (X's upper-right block).
            const int r2 = lane >> 1, cc0 = (lane & 1) * 8;
            float acc[8];
#pragma unroll
            for (int e = 0; e < 8; ++e) acc[e] = 0.f;
#pragma unroll
            for (int k = 0; k < 16; ++k) {
                const float a = lds_f32(aL + k * S + (16 + r2) * 4);                  // L21[r2][k] = L[16 + r2][k]
                const float4 b0 = lds_f4(aL + k * S + cc0 * 4);                       // X11[k][cc0 ..]
                const float4 b1 = lds_f4(aL + k * S + (cc0 + 4) * 4);
                acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
                acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
            }
            sts_f4(aL + (16 + r2) * S + cc0 * 4, make_float4(acc[0], acc[1], acc[2], acc[3]));
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
                const float4 b0 = lds_f4(aL + (16 + k) * S + cc0 * 4);                // M[k][cc0 ..]
                const float4 b1 = lds_f4(aL + (16 + k) * S + (cc0 + 4) * 4);
                const float a = xr[k];
                acc[0] = fmaf(a, b0.x, acc[0]); acc[1] = fmaf(a, b0.y, acc[1]); acc[2] = fmaf(a, b0.z, acc[2]); acc[3] = fmaf(a, b0.w, acc[3]);
                acc[4] = fmaf(a, b1.x, acc[4]); acc[5] = fmaf(a, b1.y, acc[5]); acc[6] = fmaf(a, b1.z, acc[6]); acc[7] = fmaf(a, b1.w, acc[7]);
            }
            __syncwarp();                                                             // every M has been read
            sts_f4(aL + (16 + r2) * S + cc0 * 4, make_float4(-acc[0], -acc[1], -acc[2], -acc[3]));
            sts_f4(aL + (16 + r2) * S + (cc0 + 4) * 4, make_float4(-acc[4], -acc[5], -acc[6], -acc[7]));
            sts_f4(aL + r2 * S + (16 + cc0) * 4, make_float4(0.f, 0.f, 0.f, 0.f));
            sts_f4(aL + r2 * S + (16 + cc0 + 4) * 4, make_float4(0.f, 0.f, 0.f, 0.f));
        }
        const uint32_t qbar = 1 + wq, qthreads = 32 * NH;
        // all NH warps of the quadrant pick up their columns of row `lane`
        asm volatile("bar.sync %0, %1;" ::"r"(qbar), "r"(qthreads) : "memory");
        ld_shared_fw(Lq + lane * kLsStride + cb, X);
    }
    store_roww_bf16(aB, kBlk, row, wq * 32 + cb, X);
    sync_then_issue();

    // One doubling level: Y = D (L_off D).  Only the blocks the level needs are computed, so the MMAs are
    // small (the operands are block-structured: D is block-diagonal, L_off strictly block-lower):
    //   level 1 (32 -> 64): Y[blk 2i+1, blk 2i] = D_{2i+1} L_{2i+1,2i} D_{2i}, i = 0, 1
    //                       X1[:, blk 2i] = L_off[:, blk 2i] D_{2i}   (N = 32, K = 32) -> c0 columns 64 i
    //                       Y [:, blk 2i] = D[:, blk 2i+1] X1[blk 2i+1, blk 2i]        -> c0 columns 64 i
    //   level 2 (64 -> 128): Y[64:128, 0:64] = T_1 L[64:128, 0:64] T_0
    //                       X1[:, 0:64] = L_off[:, 0:64] T_0        (N = 64, K = 64)   -> c0 columns 0..63
    //                       Y [:, 0:64] = D'[:, 64:128] X1[64:128, 0:64]
    // Rows outside the block a level needs hold partial sums and are never read.
    auto doubling_mmas = [&](int level) {
        if (tid == 0) {           // X1 = L_off * D  (A = sA K-major, B = sB MN-major)
            tc_fence_after();
            if (level == 1) {
                const uint32_t id = umma_idesc(128, 32, false, true);
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int s = 0; s < 2; ++s)
                        umma_bf16(c0 + 64 * i, desc_kmajor(aA + i * kBlk + s * 32), desc_mnmajor(aB + i * kBlk + (4 * i + s) * 2048, kBlk), id, s > 0);
                umma_commit(bar_mma);
            } else {
                const uint32_t id = umma_idesc(128, 64, false, true);
#pragma unroll
                for (int s = 0; s < 4; ++s)
                    umma_bf16(c0, desc_kmajor(aA + s * 32), desc_mnmajor(aB + s * 2048, kBlk), id, s > 0);
                umma_commit(bar_mma);
            }
        }
        wait_mma();
        if (level == 1) {         // whole rows: the needed block, zeros elsewhere (sC is never pre-zeroed)
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                float v[CW];
                if ((wq & 1) && cc == wq - 1) {
                    tmem_ldw(tmem_addr(c0, lane_base, cc * 32 + cb), v);
                } else {
#pragma unroll
                    for (int e = 0; e < CW; ++e) v[e] = 0.f;
                }
                store_roww_bf16(aC, kBlk, row, cc * 32 + cb, v);
            }
        } else if (wq >= 2) {
            float v0[CW], v1[CW];
            tmem_ldw2(tmem_addr(c0, lane_base, cb), tmem_addr(c0, lane_base, 32 + cb), v0, v1);
            store_roww_bf16(aC, kBlk, row, cb, v0);
            store_roww_bf16(aC, kBlk, row, 32 + cb, v1);
        }
        sync_then_issue();
        if (tid == 0) {           // Y = D * X1  (A = sB K-major, B = sC MN-major)
            tc_fence_after();
            if (level == 1) {
                const uint32_t id = umma_idesc(128, 32, false, true);
#pragma unroll
                for (int i = 0; i < 2; ++i)
#pragma unroll
                    for (int s = 2; s < 4; ++s)
                        umma_bf16(c0 + 64 * i, desc_kmajor(aB + i * kBlk + s * 32), desc_mnmajor(aC + i * kBlk + (4 * i + s) * 2048, kBlk), id, s > 2);
            } else {
                const uint32_t id = umma_idesc(128, 64, false, true);
#pragma unroll
                for (int s = 0; s < 4; ++s)
                    umma_bf16(c0, desc_kmajor(aB + kBlk + s * 32), desc_mnmajor(aC + (4 + s) * 2048, kBlk), id, s > 0);
            }
            umma_commit(bar_mma);
            if (level == (C == 128 ? 2 : 1)) {
                // Q K^T -> c1: not needed before the P mask, so it runs in the shadow of the last doubling read-out
                // (the next commit covers it); the Q tile was requested two round trips ago
                mbar_wait(bar_q, par);
                tc_fence_after();
                const uint32_t idq = umma_idesc(128, 128, false, false);
#pragma unroll
                for (int s = 0; s < DS; ++s) {
                    const uint32_t off = (s >> 2) * kBlk + (s & 3) * 32;
                    umma_bf16(c1, desc_kmajor(aQ + off), desc_kmajor(aK + off), idq, s > 0);
                }
            }
        }
        wait_mma();
    };

    if (tid == 64) {                               // sQ, sV are free: the previous tile's stores were complete before the K K^T commit
        mbar_expect_tx(bar_q, TILE);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_5d(sQ + nb * kBlk, tmQ, bar_q, nb * 64, h, tile * 128, 0, b);
        mbar_expect_tx(bar_v, TILE);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_5d(sV + nb * kBlk, tmV, bar_v, nb * 64, h, tile * 128, 0, b);
    }
    // ---- T3/T4: 32 -> 64 blocks: D' = D - mask(D L_off D) ------------------------------------------
    doubling_mmas(1);
    float Dlow[CW];                                // block (wq, wq-1) of the 64x64 inverse, odd wq
#pragma unroll
    for (int j = 0; j < CW; ++j) Dlow[j] = 0.f;
    if (wq & 1) {
        float v[CW];
        tmem_ldw(tmem_addr(c0, lane_base, (wq - 1) * 32 + cb), v);
#pragma unroll
        for (int j = 0; j < CW; ++j) Dlow[j] = -v[j];
        store_roww_bf16(aB, kBlk, row, (wq - 1) * 32 + cb, Dlow);
    }
    float Tlow[2 * CW];                            // rows >= 64, this thread's columns of chunks 0 and 1
#pragma unroll
    for (int j = 0; j < 2 * CW; ++j) Tlow[j] = 0.f;
    if (C == 128) {
        sync_then_issue();
        doubling_mmas(2);
        if (wq >= 2) {
            float v0[CW], v1[CW];
            tmem_ldw2(tmem_addr(c0, lane_base, cb), tmem_addr(c0, lane_base, 32 + cb), v0, v1);
#pragma unroll
            for (int j = 0; j < CW; ++j) { Tlow[j] = -v0[j]; Tlow[CW + j] = -v1[j]; }
        }
    }
    // ---- scaled copies of Tm: sA = Tm diag(beta gamma), sC = Tm diag(beta) -------------------------
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        if (cc <= wq && cc >= half_lo) {
            float tm[CW], sbg[CW], sbt[CW], va[CW], vc[CW];
#pragma unroll
            for (int e = 0; e < CW; ++e) {
                if (cc == wq) tm[e] = X[e];
                else if ((wq & 1) && cc == wq - 1) tm[e] = Dlow[e];
                else if (C == 128 && wq >= 2 && cc < 2) tm[e] = Tlow[cc * CW + e];
                else tm[e] = 0.f;
            }
            ld_shared_fw(sBG + cc * 32 + cb, sbg);
            ld_shared_fw(sBeta + cc * 32 + cb, sbt);
#pragma unroll
            for (int e = 0; e < CW; ++e) { va[e] = tm[e] * sbg[e]; vc[e] = tm[e] * sbt[e]; }
            store_roww_bf16(aA, kBlk, row, cc * 32 + cb, va);
            store_roww_bf16(aC, kBlk, row, cc * 32 + cb, vc);
        }
    }
    sync_then_issue();

    // ---- T7: W = Tm diag(beta gamma) K -> c2,  Ut = Tm diag(beta) V -> c3 ---------------------------
    mbar_wait(bar_v, par);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, D, false, true);
#pragma unroll
        for (int s = 0; s < KS; ++s)
            umma_bf16(c2, desc_kmajor(aA + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aK + s * 2048, kBlk), id, s > 0);
#pragma unroll
        for (int s = 0; s < KS; ++s)
            umma_bf16(c3, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aV + s * 2048, kBlk), id, s > 0);
        umma_commit(bar_mma);
    }
    wait_mma();

    // ---- round trip 6: W -> sB, Ut -> sA, P -> sC, Kt in place -------------------------------------
#pragma unroll
    for (int cc = 0; cc < D / 32; ++cc) {
        float w[CW], u[CW];
        tmem_ldw2(tmem_addr(c2, lane_base, cc * 32 + cb), tmem_addr(c3, lane_base, cc * 32 + cb), w, u);
        store_roww_bf16(aB, kBlk, row, cc * 32 + cb, w);
        store_roww_bf16(aA, kBlk, row, cc * 32 + cb, u);
    }
#pragma unroll
    for (int cc = 0; cc < 4; ++cc) {
        if (cc <= wq && cc >= half_lo) {
            float v[CW], f[CW];
            tmem_ldw(tmem_addr(c1, lane_base, cc * 32 + cb), v);
            if (cc == wq) {                        // same 32-chunk: direct exponentials, diagonal included
                float gj[CW];
                ld_shared_fw(sGam + wq * 32 + cb, gj);
#pragma unroll
                for (int e = 0; e < CW; ++e) f[e] = ((cb + e <= lane) ? 1.f : 0.f) * fast_exp(fminf(gam_i - gj[e], 0.f));
            } else {
                ld_shared_fw(sCF + cc * 32 + cb, f);
                const float r = (cc == 0) ? rf[0] : (cc == 1 ? rf[1] : rf[2]);
#pragma unroll
                for (int e = 0; e < CW; ++e) f[e] *= r;
            }
#pragma unroll
            for (int e = 0; e < CW; ++e) v[e] *= f[e];
            store_roww_bf16(aC, kBlk, row, cc * 32 + cb, v);
        }
    }
    {
        const float ks = fast_exp(gam_end - gam_i);
#pragma unroll
        for (int c2i = 0; c2i < D / (8 * NH); ++c2i) {
            const int ch = c2i * NH + hh;
            const uint32_t addr = aK + swz_chunk_off(row, ch, kBlk);
            float f[8];
            unpack8(ld_shared_v4(addr), f);
            st_shared_v4(addr, pack_bf16(f[0] * ks, f[1] * ks), pack_bf16(f[2] * ks, f[3] * ks),
                         pack_bf16(f[4] * ks, f[5] * ks), pack_bf16(f[6] * ks, f[7] * ks));
        }
    }
    sync_then_issue();

    // ---- T8: [N | G] = Kt^T [Ut | W] -> c0.., [P Ut | P W] -> c2.. (B operand = sA then sB, N = 2D) ----
    //      column layout of both results: [0, D) from Ut, [D, 2D) from W.  For D = 128 they take 256 columns
    //      each: [N|G] -> c0,c1 and [PUt|PW] -> c2,c3.
    const float gamma_i = fast_exp(gam_i);
    constexpr uint32_t LBO2 = (D == 128) ? kBlk : 2 * kBlk;     // distance between the 64-column blocks of [Ut | W]
    constexpr uint32_t SBLK = (uint32_t)D * 128;                 // one [D][64] bf16 or [D][32] fp32 summary block
    const int m = (D == 128) ? row : (16 * wq + lane);           // summary row held by this thread
    const bool m_ok = (D == 128) || (lane < 16);
    auto issue_summary = [&](int hf) {                           // tid 0
        tc_fence_after();
        const uint32_t idg = umma_idesc(D, 2 * D, true, true);
        const int s_lo = (C == 128) ? 0 : hf * 4, s_hi = (C == 128) ? KS : hf * 4 + 4;
        const uint32_t acc = (hf == 0) ? c0 : c2;
        for (int s = s_lo; s < s_hi; ++s)
            umma_bf16(acc, desc_mnmajor(aK + s * 2048, kBlk), desc_mnmajor(aA + s * 2048, LBO2), idg, s > s_lo);
        if (hf == 0) {
            const uint32_t idp = umma_idesc(128, 2 * D, false, true);
#pragma unroll
            for (int s = 0; s < KS; ++s)
                umma_bf16(c2, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aA + s * 2048, LBO2), idp, s > 0);
        }
        umma_commit(bar_mma);
    };
    // The results leave through shared memory (the operand buffers, free once the MMAs have completed) and
    // TMA stores: full-line writes issued by one thread instead of 32 half-used sectors per warp store.
    //   [PUt | PW] at `acc` (lane = token row) -> Qt = gamma Q - P W in place in sQ, Ol = P Ut -> odst
    auto stage_QO = [&](uint32_t acc, uint32_t odst) {
#pragma unroll
        for (int cc = 0; cc < D / 32; ++cc) {
            float pu[CW], pw[CW];
            tmem_ldw2(tmem_addr(acc, lane_base, cc * 32 + cb), tmem_addr(acc, lane_base, D + cc * 32 + cb), pu, pw);
#pragma unroll
            for (int q4 = 0; q4 < CH; ++q4) {
                const uint32_t off = swz_chunk_off(row, cc * 4 + hh * CH + q4, kBlk);
                float f[8];
                unpack8(ld_shared_v4(aQ + off), f);
#pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = gamma_i * f[e] - pw[8 * q4 + e];
                st_shared_v4(aQ + off, pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
                if (FUSED) {                       // this is the local part of the output itself: out = scale (Ol + Qt S_c)
#pragma unroll
                    for (int e = 0; e < 8; ++e) pu[8 * q4 + e] *= p.scale;
                }
                st_shared_v4(odst + off, pack_bf16(pu[8 * q4], pu[8 * q4 + 1]), pack_bf16(pu[8 * q4 + 2], pu[8 * q4 + 3]),
                             pack_bf16(pu[8 * q4 + 4], pu[8 * q4 + 5]), pack_bf16(pu[8 * q4 + 6], pu[8 * q4 + 7]));
            }
        }
    };
    //   [N | G] at `acc` (lane = summary row m) -> G bf16 as [D][64] blocks at gdst, N fp32 as [D][32] blocks at ndst
    //   (FUSED: N in bf16 as well, [D][64] blocks like G: half the summary traffic; the chain adds it to its fp32 state)
    auto stage_NG = [&](uint32_t acc, uint32_t gdst, uint32_t ndst) {
#pragma unroll
        for (int cc = 0; cc < D / 32; ++cc) {
            float nv[CW], gv[CW];
            tmem_ldw2(tmem_addr(acc, lane_base, cc * 32 + cb), tmem_addr(acc, lane_base, D + cc * 32 + cb), nv, gv);
            if (m_ok) {
                store_roww_bf16(gdst, SBLK, m, cc * 32 + cb, gv);
                if (FUSED) {
                    store_roww_bf16(ndst, SBLK, m, cc * 32 + cb, nv);
                } else {
#pragma unroll
                    for (int q4 = 0; q4 < CW / 4; ++q4) {
                        const uint32_t noff = cc * SBLK + (uint32_t)m * 128u + (uint32_t)((((cb >> 2) + q4) ^ (m & 7)) << 4);
                        st_shared_v4(ndst + noff, __float_as_uint(nv[4 * q4]), __float_as_uint(nv[4 * q4 + 1]),
                                     __float_as_uint(nv[4 * q4 + 2]), __float_as_uint(nv[4 * q4 + 3]));
                    }
                }
            }
        }
    };
    auto store_QO = [&](const uint8_t* odst) {                   // tid 0
        const int r0 = (int)(((long long)bh * p.NT + tile) * 128);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            tma_store_2d(tmQt, sQ + nb * kBlk, nb * 64, r0);
            if (FUSED) tma_store_5d(tmOl, odst + nb * kBlk, nb * 64, h, tile * 128, 0, b);    // tmOl = map of `out` (rows past T are clipped)
            else tma_store_2d(tmOl, odst + nb * kBlk, nb * 64, r0);
        }
    };
    // j_lo .. j_hi: which [D][32] blocks of N go with this call (FUSED, d = 128: the last two, staged in sC, are stored
    // by the flag thread as a group of its own, so that tid 0's wait in front of the next K K^T commit is shorter)
    auto store_NG = [&](const uint8_t* gsrc, const uint8_t* nsrc, int chunk, int j_lo = 0, int j_hi = D / 32, bool with_g = true) {
        const int z = bh * p.NC + chunk;
        if (with_g) {
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) tma_store_3d(tmG, gsrc + nb * SBLK, nb * 64, 0, z);
        }
        if (FUSED) {
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) tma_store_3d(tmN, nsrc + nb * SBLK, nb * 64, 0, z);       // bf16 [D][64] blocks
        } else {
            for (int j = j_lo; j < j_hi; ++j) tma_store_3d(tmN, nsrc + j * SBLK, j * 32, 0, z);
        }
    };
    auto publish_staging = [&]() { fence_proxy_async(); tc_fence_before(); __syncthreads(); };

    if (C == 128) {
        // [P Ut | P W] first with a commit of its own: Qt / Ol are staged (and, d = 128, sent off) while [N | G] still runs
        if (tid == 0) {
            tc_fence_after();
            const uint32_t idp = umma_idesc(128, 2 * D, false, true), idg = umma_idesc(D, 2 * D, true, true);
#pragma unroll
            for (int s = 0; s < KS; ++s)
                umma_bf16(c2, desc_kmajor(aC + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aA + s * 2048, LBO2), idp, s > 0);
            umma_commit(bar_mma);
#pragma unroll
            for (int s = 0; s < KS; ++s)
                umma_bf16(c0, desc_mnmajor(aK + s * 2048, kBlk), desc_mnmajor(aA + s * 2048, LBO2), idg, s > 0);
            umma_commit(cx.bar_mma2);
        }
    } else {
        if (tid == 0) issue_summary(0);
    }
    if (gates && next_bh >= 0) *gates = load_gates(next_bh, next_tile);       // lands while the summary MMAs run
    wait_mma();
    if (C == 128) {
        stage_QO(c2, aV);                          // Qt in place in sQ, Ol -> sV: neither is an operand of [N | G]
        if (FUSED && D == 128) {
            // d = 128 leaves 160 KB per tile and the next tile's K K^T commit waits for these stores: Qt / Ol (64 KB) set
            // off while G / N are still being computed and staged
            publish_staging();
            if (tid == 0) { store_QO(sV); tma_store_commit(); }
        }
        mbar_wait(cx.bar_mma2, par);
        tc_fence_after();
    }
    if (FUSED && tid == 0 && next_bh >= 0) {
        // sK is free (the summary MMAs were its last readers): fetch the next tile's K ahead of this tile's
        // stores, so the next K K^T does not queue behind them
        mbar_expect_tx(bar_kq, TILE);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_5d(sK + nb * kBlk, tmK, bar_kq, nb * 64, next_bh % p.H, next_tile * 128, 0, next_bh / p.H);
    }
    if (C == 128) {
        // everything is free now: Qt in place, Ol -> sV, G -> sA, N -> sB (+ sC)
        stage_NG(c0, aA, aB);
        if (tid == 0) p.gam[(long long)bh * p.NC + tile] = fast_exp(gam_end);
        publish_staging();
        if (tid == 0) {
            if (!(FUSED && D == 128)) store_QO(sV);
            if (FUSED) tma_store_commit();         // group 1: Qt, Ol (sQ, sV); group 2: G, N (sA, sB, sC)
            store_NG(sA, sB, tile);                // FUSED: N is bf16 and fits sB (d = 128: 32 KB)
            tma_store_commit();
            if (!FUSED) tma_store_wait_read();     // FUSED: the next tile waits where it reuses the staging
        }
    } else {
        // first half: drain [PUt | PW] (c2), send Qt / Ol off, then reuse c2 for the second chunk's [N | G]
        stage_QO(c2, aV);
        if (tid == 0 || tid == 64) p.gam[(long long)bh * p.NC + 2 * tile + (tid >> 6)] = fast_exp(gam_end);
        publish_staging();
        if (tid == 0) {
            store_QO(sV);
            tma_store_commit();
            issue_summary(1);
            if (D == 128) tma_store_wait_read();                 // sQ, sV are the staging of the second N below
        }
        wait_mma();
        if (D == 128) __syncthreads();
        // chunk 2t: G -> sC, N -> sA (+ sB);  chunk 2t+1: G -> sK, N -> sB (D = 64) or sQ + sV (D = 128)
        const uint32_t aN1 = (D == 64) ? aB : aQ;
        uint8_t* sN1 = (D == 64) ? sB : sQ;
        stage_NG(c0, aC, aA);
        stage_NG(c2, aK, aN1);
        publish_staging();
        if (tid == 0) {
            store_NG(sC, sA, 2 * tile);
            store_NG(sK, sN1, 2 * tile + 1);
            tma_store_commit();
            tma_store_wait_read();
        }
    }

}

template <int D, int C>
__global__ void __launch_bounds__(kPrepassThreads, 1)
gdn_tok_prepass(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
                const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmG,
                const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmQt,
                const __grid_constant__ CUtensorMap tmOl, const TokParams p) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    PrepassCtx cx;
    uint32_t* tmem_slot;
    prepass_carve<D>(smem, cx, &tmem_slot);
    if (threadIdx.x == 0) {
        mbar_init(cx.bar_kq, 1); mbar_init(cx.bar_q, 1); mbar_init(cx.bar_v, 1); mbar_init(cx.bar_mma, 1); mbar_init(cx.bar_mma2, 1);
        mbar_fence_init();
    }
    if (threadIdx.x < 32) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    cx.tmem = *tmem_slot;
    pdl_launch_dependents();
    uint32_t ph = 0;
    prepass_tile<D, C, false>(cx, &tmQ, &tmK, &tmV, &tmG, &tmN, &tmQt, &tmOl, p, blockIdx.x / p.NT, blockIdx.x % p.NT, 0u, ph);
    tc_fence_before();
    __syncthreads();
    if (threadIdx.x < 32) tmem_dealloc(cx.tmem, 512);
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

constexpr int kChainThreads = 192;     // warps 0-3: state rows (epilogue); warp 4: MMA issuer; warp 5: TMA producer

template <int D>
__device__ __forceinline__ void chain_body(const CUtensorMap* tmGp, const CUtensorMap* tmNp, const CUtensorMap* tmScp,
                                           const TokParams& p, const int cta) {
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
    const int NT_COL = p.col_tiles ? p.col_tiles : D / 64;
    const int ct = cta % NT_COL, bh = cta / NT_COL;
    const int n0 = ct * 64;
    const bool worker = warp < 4;
    const int m = (D == 128) ? tid : (16 * warp + lane);              // state row of a worker thread
    const bool m_ok = worker && ((D == 128) || (lane < 16));
    uint64_t* bar_mma = &bars[STAGES];

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) mbar_init(&bars[s], 1);
        mbar_init(bar_mma, 1);
        mbar_fence_init();
    }
    if (tid == 160) { tma_prefetch_desc(tmGp); tma_prefetch_desc(tmNp); tma_prefetch_desc(tmScp); }   // descriptor fetch off the first loads' path
    if (warp == 0) tmem_alloc(tmem_slot, 64);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_launch_dependents();
    // Only the summaries (G, N, gamma) come from the previous kernel: the TMA producer waits for it before its first load and
    // the state rows before they read gamma.  The carried state S_in is older than that (the previous call's kernels are
    // complete before this call's first kernel passes its own wait), so its load and the first operand copy overlap the
    // previous kernel's tail.
    if (warp >= 4) pdl_wait();

    auto ent = [&](int c) { return p.rev ? p.NCa - 1 - c : c; };      // summary entry of step c / snapshot slot of state c
    auto issue_loads = [&](int c) {
        const int st = c % STAGES;
        uint8_t* base = sStage + st * L::STAGE;
        mbar_expect_tx(&bars[st], L::STAGE);
        const int z = bh * p.NCa + ent(c);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_3d(base + nb * (D * 128), tmGp, &bars[st], nb * 64, 0, z);
        tma_load_3d(base + L::G_BYTES, tmNp, &bars[st], n0, 0, z);
        tma_load_3d(base + L::G_BYTES + D * 128, tmNp, &bars[st], n0 + 32, 0, z);
    };
    if (warp == 5 && lane == 0)
        for (int c = 0; c < STAGES && c < p.NC; ++c) issue_loads(c);

    // state row m, columns n0..n0+63, fp32 master copy in registers
    float S[64];
    if (p.zvec) {
#pragma unroll
        for (int i = 0; i < 64; ++i) S[i] = 0.f;
        if (m_ok && m < p.dr && ct == 0 && p.z_vec_in) S[0] = p.z_vec_in[(long long)bh * p.dr + m];
    } else if (m_ok && m < p.dr && p.S_in) {
        const float4* src = reinterpret_cast<const float4*>(p.S_in + ((long long)bh * p.dr + m) * p.dr + n0);
#pragma unroll
        for (int i = 0; i < 16; ++i) {
            const float4 f = (n0 + 4 * i < p.dr) ? src[i] : make_float4(0.f, 0.f, 0.f, 0.f);
            S[4 * i] = f.x; S[4 * i + 1] = f.y; S[4 * i + 2] = f.z; S[4 * i + 3] = f.w;
        }
    } else {
#pragma unroll
        for (int i = 0; i < 64; ++i) S[i] = 0.f;
    }
    // publish S (bf16) as the next MMA's B operand (shared buffer `buf`)
    auto publish_smem = [&](int buf) {
        if (m_ok) {
            const uint32_t sbase = smem_u32(sS + buf * L::S_BYTES);
#pragma unroll
            for (int ch = 0; ch < 8; ++ch)
                st_shared_v4(sbase + swz_chunk_off(m, ch, 0), pack_bf16(S[8 * ch], S[8 * ch + 1]), pack_bf16(S[8 * ch + 2], S[8 * ch + 3]),
                             pack_bf16(S[8 * ch + 4], S[8 * ch + 5]), pack_bf16(S[8 * ch + 6], S[8 * ch + 7]));
        }
    };
    if (worker) { publish_smem(0); pdl_wait(); }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();

    if (warp == 4) {
        // ===== MMA issuer: D[tmem] = G_c (A, K-major) * S_c (B, MN-major), one commit per chunk =====
        const uint32_t id = umma_idesc(D, 64, false, true);
        for (int c = 0; c < p.NC; ++c) {
            const int st = c % STAGES;
            if (lane == 0) {
                mbar_wait(&bars[st], (uint32_t)(c / STAGES) & 1u);
                tc_fence_after();
                const uint32_t aG = smem_u32(sStage + st * L::STAGE), aS = smem_u32(sS + (c & 1) * L::S_BYTES);
#pragma unroll
                for (int s = 0; s < D / 16; ++s)
                    umma_bf16(tmem, desc_kmajor(aG + (s >> 2) * (D * 128) + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), id, s > 0);
                umma_commit(bar_mma);
            }
            __syncwarp();
            tc_fence_before();
            __syncthreads();
        }
    } else if (warp == 5) {
        // ===== TMA producer: refill a stage as soon as the step that used it has ended, and write the bf16
        //       operand tile sS (= state at the start of chunk c) to the workspace for kernel 3 with one TMA
        //       store straight from shared memory (no per-thread global stores on the chain) =====
        const int sstride = p.snap_stride ? p.snap_stride : p.NSc;
        auto store_snapshot = [&](int c) {           // sS[c & 1] holds the state at the start of chunk c
            const int slot = ent(c) + p.snap_off;
            if (p.snap_add && slot > 0) tma_reduce_add_3d(tmScp, sS + (c & 1) * L::S_BYTES, n0, 0, bh * sstride + slot);
            else tma_store_3d(tmScp, sS + (c & 1) * L::S_BYTES, n0, 0, bh * sstride + slot);
            tma_store_commit();
        };
        if (lane == 0 && !(p.snap_add && p.rev)) store_snapshot(0);      // (the reverse scan starts from zero: nothing to add)
        for (int c = 0; c < p.NC; ++c) {
            if (lane == 0) tma_store_wait_read();    // snapshot c has left sS[c & 1] before step c+1 may overwrite it
            __syncthreads();                          // end of step c: sS[(c+1) & 1] published, stage c % STAGES free
            if (lane == 0) {
                if (c + 1 < p.NSc) store_snapshot(c + 1);
                if (c + STAGES < p.NC) issue_loads(c + STAGES);
            }
        }
        if (lane == 0) tma_store_wait_read();        // the snapshots have left shared memory; their writes complete with the kernel
    } else {
        // ===== state rows: S <- (gamma_c S + N_c) - G_c S =====
        uint32_t ph_mma = 0;
        float gamma_c = p.NC > 0 ? p.gam[(long long)bh * p.NCa + ent(0)] : 0.f;
        for (int c = 0; c < p.NC; ++c) {
            const int st = c % STAGES;
            uint8_t* base = sStage + st * L::STAGE;
            const float gamma_next = (c + 1 < p.NC) ? p.gam[(long long)bh * p.NCa + ent(c + 1)] : 0.f;
            mbar_wait(&bars[st], (uint32_t)(c / STAGES) & 1u);
            if (m_ok) {                                // state-independent part while the MMA runs
#pragma unroll
                for (int cc = 0; cc < 2; ++cc) {
                    const uint32_t nbase = smem_u32(base + L::G_BYTES + cc * (D * 128));
#pragma unroll
                    for (int ch = 0; ch < 8; ++ch) {
                        const uint4 u = ld_shared_v4(nbase + swz_chunk_off(m, ch, 0));
                        const int i0 = cc * 32 + ch * 4;
                        S[i0 + 0] = fmaf(gamma_c, S[i0 + 0], __uint_as_float(u.x));
                        S[i0 + 1] = fmaf(gamma_c, S[i0 + 1], __uint_as_float(u.y));
                        S[i0 + 2] = fmaf(gamma_c, S[i0 + 2], __uint_as_float(u.z));
                        S[i0 + 3] = fmaf(gamma_c, S[i0 + 3], __uint_as_float(u.w));
                    }
                }
            }
            mbar_wait(bar_mma, ph_mma); ph_mma ^= 1;
            tc_fence_after();
            {
                float v[64];
                tmem_ld64(tmem_addr(tmem, warp * 32, 0), v);
#pragma unroll
                for (int i = 0; i < 64; ++i) S[i] -= v[i];
            }
            publish_smem((c + 1) & 1);
            fence_proxy_async();
            tc_fence_before();
            __syncthreads();
            gamma_c = gamma_next;
        }
        if (p.zvec) {
            if (m_ok && m < p.dr && ct == 0 && p.z_vec_out) p.z_vec_out[(long long)bh * p.dr + m] = S[0];
        } else if (p.S_out) {
            // The state rows leave through shared memory (the operand stages are idle now; 16-byte chunks XOR-ed with the row
            // against bank conflicts) so that a warp writes whole 256-byte row segments: row-per-thread stores (32 lines per
            // request) took 1.5 us here, and the next kernel waits for this one to complete.
            const uint32_t stg = smem_u32(sStage);
            if (m_ok) {
#pragma unroll
                for (int i = 0; i < 16; ++i)
                    st_shared_v4(stg + (uint32_t)m * 256u + (uint32_t)((i ^ (m & 15)) << 4), __float_as_uint(S[4 * i]), __float_as_uint(S[4 * i + 1]),
                                 __float_as_uint(S[4 * i + 2]), __float_as_uint(S[4 * i + 3]));
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            for (int idx = tid; idx < D * 16; idx += 128) {
                const int row = idx >> 4, c = idx & 15;
                if (row < p.dr && n0 + 4 * c < p.dr) {
                    const uint4 u = ld_shared_v4(stg + (uint32_t)row * 256u + (uint32_t)((c ^ (row & 15)) << 4));
                    st_global_v4(p.S_out + ((long long)bh * p.dr + row) * p.dr + n0 + 4 * c, u.x, u.y, u.z, u.w);
                }
            }
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 64);
}

template <int D>
__global__ void __launch_bounds__(kChainThreads, 1)
gdn_tok_chain(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmN,
              const __grid_constant__ CUtensorMap tmSc, const TokParams p) {
    chain_body<D>(&tmG, &tmN, &tmSc, p, (int)blockIdx.x);
}

// Both scans of the bidirectional frame path in ONE launch (they share the summaries and do not depend on each other,
// Alg. 1 l.9-17): CTAs [0, n_fwd) run the forward scan `pf` (snapshots -> tmScF), the rest the reverse scan `pr`.
template <int D>
__global__ void __launch_bounds__(kChainThreads, 1)
gdn_tok_chain_bidir(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmN,
                    const __grid_constant__ CUtensorMap tmScF, const __grid_constant__ CUtensorMap tmScR,
                    const TokParams pf, const TokParams pr, const int n_fwd) {
    if ((int)blockIdx.x < n_fwd) chain_body<D>(&tmG, &tmN, &tmScF, pf, (int)blockIdx.x);
    else chain_body<D>(&tmG, &tmN, &tmScR, pr, (int)blockIdx.x - n_fwd);
}

// Every scan of the normalised frame path in ONE launch: the matrix pass (forward, and reverse with GDN_FLAG_BIDIR) and the z
// pass (the same two, on its own summaries and snapshots, first column tile only).  They are independent of one another; as
// separate launches on two streams the readout behind them had two dependencies and could not be a programmatic dependent.
// Set s takes the next n[s] CTAs (n[s] = 0: absent).
struct ChainSets { TokParams p[4]; int n[4]; };

template <int D>
__global__ void __launch_bounds__(kChainThreads, 1)
gdn_tok_chain_multi(const __grid_constant__ CUtensorMap tmG, const __grid_constant__ CUtensorMap tmN,
                    const __grid_constant__ CUtensorMap tmScF, const __grid_constant__ CUtensorMap tmScR,
                    const __grid_constant__ CUtensorMap tmGz, const __grid_constant__ CUtensorMap tmNz,
                    const __grid_constant__ CUtensorMap tmSczF, const __grid_constant__ CUtensorMap tmSczR, const ChainSets cs) {
    int cta = (int)blockIdx.x, s = 0;
    while (s < 3 && cta >= cs.n[s]) { cta -= cs.n[s]; ++s; }
    const TokParams p = cs.p[s];
    const CUtensorMap* g = s < 2 ? &tmG : &tmGz;
    const CUtensorMap* n = s < 2 ? &tmN : &tmNz;
    const CUtensorMap* sc = s == 0 ? &tmScF : (s == 1 ? &tmScR : (s == 2 ? &tmSczF : &tmSczR));
    chain_body<D>(g, n, sc, p, cta);
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
    pdl_wait();                                    // the chain's state snapshots are complete
    const long long row = ((long long)bh * p.NT + tile) * 128 + tid;
    if (tid == 0) {
        mbar_expect_tx(&bars[0], QT_BYTES + NS * S_BYTES);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) tma_load_2d(sQt + nb * kBlk, &tmQt, &bars[0], nb * 64, (int)(((long long)bh * p.NT + tile) * 128));
#pragma unroll
        for (int s = 0; s < NS; ++s)
#pragma unroll
            for (int nb = 0; nb < NB; ++nb)
                tma_load_3d(sS + s * S_BYTES + nb * (D * 128), &tmSc, &bars[0], nb * 64, 0, bh * p.NSc + tile * NS + s);
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
