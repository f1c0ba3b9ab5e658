// gdn_tc_frame.cuh -- frame-wise (G = tokens per frame) Gated DeltaNet forward on tcgen05 tensor cores:
// the paper's own variant (Eq. 4-5, Alg. 1), re-designed for sm_100a.
//
//   Phase A  gdn_frm_summaries : per (b,h,f) and token split, [Gram | A] = (sqrt(beta) K)^T [sqrt(beta) K | sqrt(beta) V]
//                                token-contraction MMAs (M = d, N = 2d, K = tokens) fed by a TMA ring;
//                                both operands are MN-major views of the TMA tiles, no transposes.
//            gdn_frm_reduce    : fixed-order sum of the token-split partials -> G_f = alpha_f Gram_f (bf16),
//                                N_f = A_f (fp32), gamma_f = alpha_f           (deterministic, no atomics)
//   Phase B  gdn_tok_chain     : S_f = alpha_f S_{f-1} - G_f S_{f-1} + N_f  -- the same one-MMA-per-step chain
//                                kernel as the token-wise path (Eq. 5: S_f = alpha_f (I - Gram_f) S_{f-1} + A_f)
//   Phase C  gdn_frm_readout   : O_f = scale * Q_f S_f  (every token of frame f reads the post-update state, Eq. 22)
//
// Tokens beyond the end of a frame inside a 128-token tile are zero-filled by the 5-D tensor map
// (d, H, G, F, B) and get beta = 0: they contribute nothing and are never stored.
#pragma once
#include <cuda.h>

#include "gdn_tc_token.cuh"

namespace gdn {

struct FrmParams {
    const float* alpha;          // [BH][F]
    const float* beta;           // [BH][T]
    void* out;                   // [B][T][H][D] bf16
    float* part;                 // [BH*F][NSPLIT][D][2D] fp32 partial summaries
    __nv_bfloat16* Gw;           // [BH][F][D][D]
    float* Nw;                   // [BH][F][D][D]
    float* gam;                  // [BH][F]
    int B, H, T, G, F, NSPLIT, TPF;   // TPF = 128-token tiles per frame
    int NSc;                     // snapshot slots per (b,h) = F + 1
    long long o_ts;
    float scale;
    int log_alpha;
};

namespace frm {

using namespace tc;
using tok::kBlk;
using tok::st_global_v4;

constexpr int kSumThreads = 192;       // warps 0-3: beta scaling + epilogue; warp 4: MMA issuer; warp 5: TMA producer

template <int D>
struct SumSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t STAGE = 2u * NB * kBlk;                 // K tile then V tile (contiguous: one N = 2D operand)
    static constexpr int STAGES = (D == 128) ? 3 : 5;
    static constexpr uint32_t TOTAL = STAGES * STAGE + 512 + 1024;
};

// ---------------------------------------------------------------------------------------------------
// Phase A.  grid = BH*F*NSPLIT, block = 192.
// ---------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kSumThreads, 1)
gdn_frm_summaries(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV, const FrmParams p) {
    using L = SumSmem<D>;
    constexpr int NB = L::NB;
    constexpr int STAGES = L::STAGES;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + STAGES * L::STAGE);   // full[S], scaled[S], empty[S], done
    uint64_t* bar_full = bars;
    uint64_t* bar_scaled = bars + STAGES;
    uint64_t* bar_empty = bars + 2 * STAGES;
    uint64_t* bar_done = bars + 3 * STAGES;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 3 * STAGES + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int split = blockIdx.x % p.NSPLIT;
    const int bhf = blockIdx.x / p.NSPLIT;
    const int f = bhf % p.F, bh = bhf / p.F;
    const int b = bh / p.H, h = bh % p.H;
    // contiguous range of 128-token tiles of this frame handled by this split
    const int per = (p.TPF + p.NSPLIT - 1) / p.NSPLIT;
    const int tile_lo = split * per;
    const int tile_hi = min(p.TPF, tile_lo + per);
    const int ntiles = max(0, tile_hi - tile_lo);

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_scaled[s], 128); mbar_init(&bar_empty[s], 1); }
        mbar_init(bar_done, 1);
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(tmem_slot, 2 * D);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;

    if (warp == 5) {
        // ===== TMA producer =====
        if (lane == 0) {
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES;
                if (i >= STAGES) mbar_wait(&bar_empty[st], (uint32_t)((i / STAGES) - 1) & 1u);
                uint8_t* base = smem + st * L::STAGE;
                mbar_expect_tx(&bar_full[st], L::STAGE);
                const int n0 = (tile_lo + i) * 128;
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) {
                    tma_load_5d(base + nb * kBlk, &tmK, &bar_full[st], nb * 64, h, n0, f, b);
                    tma_load_5d(base + (NB + nb) * kBlk, &tmV, &bar_full[st], nb * 64, h, n0, f, b);
                }
            }
        }
    } else if (warp == 4) {
        // ===== MMA issuer: [Gram | A] += K'^T [K' | V']  (A and B both MN-major views of the stage) =====
        if (lane == 0) {
            const uint32_t id = umma_idesc(D, 2 * D, true, true);
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES;
                mbar_wait(&bar_scaled[st], (uint32_t)(i / STAGES) & 1u);
                tc_fence_after();
                const uint32_t a = smem_u32(smem + st * L::STAGE);
#pragma unroll
                for (int s = 0; s < 8; ++s)
                    umma_bf16(tmem, desc_mnmajor(a + s * 2048, kBlk), desc_mnmajor(a + s * 2048, kBlk), id, (i > 0 || s > 0) ? 1u : 0u);
                umma_commit(&bar_empty[st]);
            }
            umma_commit(bar_done);
        }
    } else {
        // ===== beta scaling (thread = token row of the tile), then the epilogue =====
        const int row = tid;
        for (int i = 0; i < ntiles; ++i) {
            const int st = i % STAGES;
            const int n = (tile_lo + i) * 128 + row;
            float sb = 0.f;
            if (n < p.G) sb = sqrtf(p.beta[(long long)bh * p.T + (long long)f * p.G + n]);
            mbar_wait(&bar_full[st], (uint32_t)(i / STAGES) & 1u);
            const uint32_t base = smem_u32(smem + st * L::STAGE) + (uint32_t)row * 128u;
#pragma unroll
            for (int blk = 0; blk < 2 * NB; ++blk) {
#pragma unroll
                for (int c = 0; c < 8; ++c) {
                    // the scale is per row, so any order of the row's 16-byte chunks works: rotate by the
                    // row index to keep the 8 lanes of a quarter-warp on distinct banks
                    const uint32_t addr = base + blk * kBlk + (uint32_t)(((c + row) & 7) << 4);
                    float x[8];
                    unpack8(ld_shared_v4(addr), x);
                    st_shared_v4(addr, pack_bf16(x[0] * sb, x[1] * sb), pack_bf16(x[2] * sb, x[3] * sb),
                                 pack_bf16(x[4] * sb, x[5] * sb), pack_bf16(x[6] * sb, x[7] * sb));
                }
            }
            fence_proxy_async();
            mbar_arrive(&bar_scaled[st]);
        }
        // epilogue: partial [Gram | A] of this split -> workspace (fp32)
        const int m = (D == 128) ? tid : (16 * warp + lane);
        const bool m_ok = (D == 128) || (lane < 16);
        float* dst = p.part + (((long long)bhf * p.NSPLIT + split) * D + m) * (2 * D);
        if (ntiles > 0) {
            mbar_wait(bar_done, 0);
            tc_fence_after();
#pragma unroll 1
            for (int cc = 0; cc < 2 * D / 32; ++cc) {
                float v[32];
                tmem_ld32(tmem_addr(tmem, warp * 32, cc * 32), v);
                if (m_ok) {
#pragma unroll
                    for (int q4 = 0; q4 < 8; ++q4)
                        st_global_v4(dst + cc * 32 + q4 * 4, __float_as_uint(v[4 * q4]), __float_as_uint(v[4 * q4 + 1]),
                                     __float_as_uint(v[4 * q4 + 2]), __float_as_uint(v[4 * q4 + 3]));
                }
            }
        } else if (m_ok) {
            for (int cc = 0; cc < 2 * D / 4; ++cc) st_global_v4(dst + cc * 4, 0, 0, 0, 0);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 2 * D);
}

// ---------------------------------------------------------------------------------------------------
// Fixed-order reduction of the split partials.  grid = (BH*F, kReduceSlices), block = 256.
//   G_f = alpha_f * Gram_f (bf16),  N_f = A_f (fp32),  gamma_f = alpha_f
// ---------------------------------------------------------------------------------------------------
constexpr int kReduceSlices = 8;       // row slices per (b,h,f): enough CTAs to pull the partials at full bandwidth

template <int D>
__global__ void __launch_bounds__(256)
gdn_frm_reduce(const FrmParams p) {
    const int bhf = blockIdx.x;
    float a = p.alpha[bhf];
    if (p.log_alpha) a = expf(a);
    if (threadIdx.x == 0 && blockIdx.y == 0) p.gam[bhf] = a;
    const float4* src = reinterpret_cast<const float4*>(p.part + (long long)bhf * p.NSPLIT * D * 2 * D);
    constexpr int ROW4 = 2 * D / 4;                 // float4 per summary row
    constexpr int PER = D * ROW4 / kReduceSlices;
    for (int e = blockIdx.y * PER + threadIdx.x; e < (blockIdx.y + 1) * PER; e += blockDim.x) {
        float4 acc = src[e];
        for (int s = 1; s < p.NSPLIT; ++s) {
            const float4 v = src[(long long)s * D * ROW4 + e];
            acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
        }
        const int m = e / ROW4, c4 = e % ROW4;
        if (c4 < D / 4) {
            __nv_bfloat16* g = p.Gw + ((long long)bhf * D + m) * D + c4 * 4;
            uint2 u;
            u.x = pack_bf16(a * acc.x, a * acc.y);
            u.y = pack_bf16(a * acc.z, a * acc.w);
            *reinterpret_cast<uint2*>(g) = u;
        } else {
            float* n = p.Nw + ((long long)bhf * D + m) * D + (c4 - D / 4) * 4;
            *reinterpret_cast<float4*>(n) = acc;
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// Phase C.  grid = BH*F*TPF, block = 128.   O = scale * Q_f S_f   (S_f = snapshot slot f + 1)
// ---------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(128)
gdn_frm_readout(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmSc, const FrmParams p) {
    constexpr int NB = D / 64;
    constexpr uint32_t Q_BYTES = NB * kBlk;
    constexpr uint32_t S_BYTES = (uint32_t)D * D * 2;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sQ = smem;
    uint8_t* sS = smem + Q_BYTES;
    uint64_t* bars = reinterpret_cast<uint64_t*>(sS + S_BYTES);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 2);

    const int tid = threadIdx.x, warp = tid >> 5;
    const int tile = blockIdx.x % p.TPF;
    const int bhf = blockIdx.x / p.TPF;
    const int f = bhf % p.F, bh = bhf / p.F;
    const int b = bh / p.H, h = bh % p.H;
    if (tid == 0) {
        mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_fence_init();
        mbar_expect_tx(&bars[0], Q_BYTES + S_BYTES);
#pragma unroll
        for (int nb = 0; nb < NB; ++nb) {
            tma_load_5d(sQ + nb * kBlk, &tmQ, &bars[0], nb * 64, h, tile * 128, f, b);
            tma_load_3d(sS + nb * (D * 128), &tmSc, &bars[0], nb * 64, 0, bh * p.NSc + f + 1);
        }
    }
    if (warp == 0) tmem_alloc(tmem_slot, D);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    mbar_wait(&bars[0], 0);
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(128, D, false, true);
        const uint32_t aQ = smem_u32(sQ), aS = smem_u32(sS);
#pragma unroll
        for (int s = 0; s < D / 16; ++s)
            umma_bf16(tmem, desc_kmajor(aQ + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aS + s * 2048, D * 128), id, s > 0);
        umma_commit(&bars[1]);
    }
    mbar_wait(&bars[1], 0);
    tc_fence_after();
    const int n = tile * 128 + tid;
    const long long t = (long long)f * p.G + n;
    __nv_bfloat16* dst = reinterpret_cast<__nv_bfloat16*>(p.out) + ((long long)b * p.T + t) * p.o_ts + (long long)h * D;
#pragma unroll
    for (int cc = 0; cc < D / 32; ++cc) {
        float v[32];
        tmem_ld32(tmem_addr(tmem, warp * 32, cc * 32), v);
        if (n < p.G) {
#pragma unroll
            for (int q4 = 0; q4 < 4; ++q4)
                st_global_v4(dst + cc * 32 + q4 * 8, pack_bf16(p.scale * v[8 * q4], p.scale * v[8 * q4 + 1]),
                             pack_bf16(p.scale * v[8 * q4 + 2], p.scale * v[8 * q4 + 3]),
                             pack_bf16(p.scale * v[8 * q4 + 4], p.scale * v[8 * q4 + 5]),
                             pack_bf16(p.scale * v[8 * q4 + 6], p.scale * v[8 * q4 + 7]));
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, D);
}

}  // namespace frm
}  // namespace gdn
