// gdn_tc_fused.cuh -- token-wise (G = 1, C = 128) Gated DeltaNet forward as ONE persistent kernel.
//
// Same mathematics as gdn_tc_token.cuh (chunkwise WY/UT form of PAPER.md Eq. 17-19 at N = 1, per-chunk
// affine summaries).  What changes is the schedule: instead of three kernels that each drain the GPU,
// one grid of ~#SM CTAs is split into two roles that run concurrently and hand tiles over through L2:
//
//   prepass workers (blockIdx >= NWC)  run prepass_tile<D,128,true> over the 128-token tiles in
//       chunk-major order (tile c of every head of the current head group, then tile c+1, ...), write
//       G_c, N_c, gamma_c, Qt, Ol to the workspace and release a per-tile ready flag;
//   chain workers (blockIdx < NWC)     own one (b,h, 64-column tile of S) unit at a time: they acquire the
//       flag of chunk c, pull G_c / Qt by TMA, run the ONE chain MMA of the step
//       S_{c+1} = gamma_c S_c - G_c S_c + N_c (fp32 master state in registers, 256 threads) and, off the
//       critical path, the output MMA O_c = scale (Qt_c S_c + Ol_c), whose tile leaves by TMA store.
//
// The S_c snapshots and the separate output kernel of the three-kernel path disappear; the summaries are
// consumed from L2 shortly after they were written.  Chain workers never block prepass workers, and a
// prepass worker's tile list is static, so every CTA makes progress even if the grid were not co-resident.
#pragma once
#include <cuda.h>

#include "gdn_tc_token.cuh"

namespace gdn {

struct FusedParams {
    TokParams t;
    unsigned int* flags;         // [BH][NT] epoch of the last call that published the tile
    unsigned int epoch;          // this call's epoch (> every earlier one)
    int NWC;                     // chain-worker CTAs = HPR * (D / 64)
    int HPR;                     // heads per round (head group)
    int total_tiles;             // BH * NT
};

namespace fused {

using namespace tc;
using tok::kBlk;

constexpr int kThreads = tok::kPrepassThreads;      // 512

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
// orders async-proxy accesses (TMA) of any state space with this thread's generic-proxy accesses
__device__ __forceinline__ void fence_proxy_async_all() { asm volatile("fence.proxy.async;" ::: "memory"); }

template <int D>
struct ChainSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t G_BYTES = (uint32_t)D * D * 2;          // NB blocks of [D][64] bf16
    static constexpr uint32_t Q_BYTES = 128u * D * 2;                 // NB blocks of [128][64] bf16
    static constexpr uint32_t S_BYTES = (uint32_t)D * 128;            // [D][64] bf16
    static constexpr int GST = (D == 128) ? 3 : 4;
    static constexpr int QST = (D == 128) ? 3 : 4;
    static constexpr uint32_t OFF_Q = GST * G_BYTES;
    static constexpr uint32_t OFF_S = OFF_Q + QST * Q_BYTES;
    static constexpr uint32_t OFF_BAR = OFF_S + 2 * S_BYTES;
    static constexpr uint32_t TOTAL = OFF_BAR + 256;
};

template <int D>
constexpr uint32_t fused_smem_bytes() {
    return (ChainSmem<D>::TOTAL > tok::prepass_smem_bytes<D>() ? ChainSmem<D>::TOTAL : tok::prepass_smem_bytes<D>()) + 1024u;
}

// ---------------------------------------------------------------------------------------------------
// chain worker.  warps 0-7: state rows (thread = row m x 32 columns); 8-11: output epilogue (thread = token
// row); 12: MMA issuer; 13: flag poller + TMA producer; 14-15: idle.
// ---------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void chain_role(uint8_t* smem, const CUtensorMap* tmG, const CUtensorMap* tmQt,
                                           const CUtensorMap* tmO, const FusedParams& fp) {
    using L = ChainSmem<D>;
    constexpr int NB = L::NB, GST = L::GST, QST = L::QST, NCT = D / 64;
    const TokParams& p = fp.t;
    uint8_t* sG = smem;
    uint8_t* sQ = smem + L::OFF_Q;
    uint8_t* sS = smem + L::OFF_S;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* g_full = bars;                  // [GST] TMA: G_c landed
    uint64_t* g_empty = g_full + GST;         // [GST] chain MMA of the step has completed
    uint64_t* q_full = g_empty + GST;         // [QST] TMA: Qt tile landed
    uint64_t* q_empty = q_full + QST;         // [QST] the out tile staged in the buffer has left
    uint64_t* mma_chain = q_empty + QST;      // chain MMA complete
    uint64_t* s_ready = mma_chain + 1;        // bf16 state operand published (8 warps)
    uint64_t* out_full = s_ready + 1;         // [2] output MMA complete
    uint64_t* out_free = out_full + 2;        // [2] output accumulator drained (4 warps)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(out_free + 2);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < GST; ++s) { mbar_init(&g_full[s], 1); mbar_init(&g_empty[s], 1); }
        for (int s = 0; s < QST; ++s) { mbar_init(&q_full[s], 1); mbar_init(&q_empty[s], 1); }
        mbar_init(mma_chain, 1);
        mbar_init(s_ready, 8);
        for (int s = 0; s < 2; ++s) { mbar_init(&out_full[s], 1); mbar_init(&out_free[s], 4); }
        mbar_fence_init();
    }
    if (warp == 0) tmem_alloc(tmem_slot, 256);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const uint32_t acc_chain = tmem;
    const int NT = p.NT;
    const int nunits = p.B * p.H * NCT;

    if (warp == 13) {
        // ===== flag poller + TMA producer =====
        if (lane == 0) {
            uint32_t gs = 0;
            for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
                const int bh = u / NCT;
                for (int c = 0; c < NT; ++c, ++gs) {
                    const unsigned int* f = fp.flags + (long long)bh * NT + c;
                    while (ld_acquire_gpu(f) < fp.epoch) __nanosleep(64);
                    fence_proxy_async_all();
                    const int gst = gs % GST, qst = gs % QST;
                    if (gs >= (uint32_t)GST) mbar_wait(&g_empty[gst], ((gs / GST) - 1) & 1u);
                    mbar_expect_tx(&g_full[gst], L::G_BYTES);
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb)
                        tma_load_3d(sG + gst * L::G_BYTES + nb * (D * 128), tmG, &g_full[gst], nb * 64, 0, bh * p.NC + c);
                    if (gs >= (uint32_t)QST) mbar_wait(&q_empty[qst], ((gs / QST) - 1) & 1u);
                    mbar_expect_tx(&q_full[qst], L::Q_BYTES);
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb)
                        tma_load_2d(sQ + qst * L::Q_BYTES + nb * kBlk, tmQt, &q_full[qst], nb * 64, (bh * NT + c) * 128);
                }
            }
        }
    } else if (warp == 12) {
        // ===== MMA issuer =====
        if (lane == 0) {
            const uint32_t idc = umma_idesc(D, 64, false, true);
            const uint32_t ido = umma_idesc(128, 64, false, true);
            uint32_t gs = 0;
            for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
                for (int c = 0; c < NT; ++c, ++gs) {
                    const int gst = gs % GST, qst = gs % QST;
                    const uint32_t aS = smem_u32(sS + (gs & 1) * L::S_BYTES);
                    // chain: acc = G_c (A, K-major) * S_c (B, MN-major)
                    mbar_wait(&g_full[gst], (gs / GST) & 1u);
                    mbar_wait(s_ready, gs & 1u);
                    tc_fence_after();
                    const uint32_t aG = smem_u32(sG + gst * L::G_BYTES);
#pragma unroll
                    for (int s = 0; s < D / 16; ++s)
                        umma_bf16(acc_chain, desc_kmajor(aG + (s >> 2) * (D * 128) + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), idc, s > 0);
                    umma_commit(mma_chain);
                    umma_commit(&g_empty[gst]);
                    // output: acc_out = Qt_c (A, K-major) * S_c
                    mbar_wait(&q_full[qst], (gs / QST) & 1u);
                    if (gs >= 2) mbar_wait(&out_free[gs & 1], ((gs >> 1) - 1) & 1u);
                    tc_fence_after();
                    const uint32_t aQ = smem_u32(sQ + qst * L::Q_BYTES);
                    const uint32_t acc_out = tmem + 64 + 64 * (gs & 1);
#pragma unroll
                    for (int s = 0; s < D / 16; ++s)
                        umma_bf16(acc_out, desc_kmajor(aQ + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), ido, s > 0);
                    umma_commit(&out_full[gs & 1]);
                }
            }
        }
    } else if (warp < 8) {
        // ===== state rows: S <- (gamma_c S + N_c) - G_c S =====
        const int wq = warp & 3, half = warp >> 2;
        const int m = (D == 128) ? (wq * 32 + lane) : (16 * wq + lane);     // state row (M = 64 uses lanes 0-15 of a quadrant)
        const bool m_ok = (D == 128) || (lane < 16);
        const int mm = m_ok ? m : 0;
        float S[32], Nr[32];
        uint32_t gs = 0;
        for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
            const int bh = u / NCT, ct = u % NCT;
            const int col0 = ct * 64 + half * 32;
            if (m_ok && p.S_in) {
                const float4* src = reinterpret_cast<const float4*>(p.S_in + ((long long)bh * D + m) * D + col0);
#pragma unroll
                for (int i = 0; i < 8; ++i) { const float4 f = __ldcg(src + i); S[4 * i] = f.x; S[4 * i + 1] = f.y; S[4 * i + 2] = f.z; S[4 * i + 3] = f.w; }
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) S[i] = 0.f;
            }
            auto publish = [&](uint32_t buf) {
                if (m_ok) {
                    const uint32_t sbase = smem_u32(sS + buf * L::S_BYTES);
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch)
                        st_shared_v4(sbase + swz_chunk_off(m, half * 4 + ch, 0), pack_bf16(S[8 * ch], S[8 * ch + 1]), pack_bf16(S[8 * ch + 2], S[8 * ch + 3]),
                                     pack_bf16(S[8 * ch + 4], S[8 * ch + 5]), pack_bf16(S[8 * ch + 6], S[8 * ch + 7]));
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(s_ready);
            };
            // chunk-major N_c: [(col / 4) * D + row] float4
            auto load_N = [&](int c) {
                const float4* src = reinterpret_cast<const float4*>(p.Nw + ((long long)bh * p.NC + c) * D * D) + (col0 >> 2) * D + mm;
#pragma unroll
                for (int i = 0; i < 8; ++i) { const float4 f = __ldcg(src + i * D); Nr[4 * i] = f.x; Nr[4 * i + 1] = f.y; Nr[4 * i + 2] = f.z; Nr[4 * i + 3] = f.w; }
            };
            publish(gs & 1);
            mbar_wait(&g_full[gs % GST], (gs / GST) & 1u);      // ordered after the poller's acquire of flag (bh, 0)
            load_N(0);
            float gamma_c = __ldcg(p.gam + (long long)bh * p.NC);
            for (int c = 0; c < NT; ++c, ++gs) {
#pragma unroll
                for (int i = 0; i < 32; ++i) S[i] = fmaf(gamma_c, S[i], Nr[i]);          // state-independent half, during the MMA
                if (c + 1 < NT) {
                    mbar_wait(&g_full[(gs + 1) % GST], ((gs + 1) / GST) & 1u);
                    load_N(c + 1);
                    gamma_c = __ldcg(p.gam + (long long)bh * p.NC + c + 1);
                }
                mbar_wait(mma_chain, gs & 1u);
                tc_fence_after();
                {
                    float v[32];
                    tmem_ld32(tmem_addr(acc_chain, wq * 32, half * 32), v);
#pragma unroll
                    for (int i = 0; i < 32; ++i) S[i] -= v[i];
                }
                tc_fence_before();
                if (c + 1 < NT) publish((gs + 1) & 1);
            }
            if (m_ok) {
                float4* dst = reinterpret_cast<float4*>(p.S_out + ((long long)bh * D + m) * D + col0);
#pragma unroll
                for (int i = 0; i < 8; ++i) dst[i] = make_float4(S[4 * i], S[4 * i + 1], S[4 * i + 2], S[4 * i + 3]);
            }
        }
    } else if (warp < 12) {
        // ===== output epilogue: out = scale (acc_out + Ol), staged in the Qt buffer, TMA store =====
        const int ew = warp - 8;
        const int row = ew * 32 + lane;
        uint32_t gs = 0;
        for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
            const int bh = u / NCT, ct = u % NCT;
            const int b = bh / p.H, h = bh % p.H;
            for (int c = 0; c < NT; ++c, ++gs) {
                const int qst = gs % QST;
                mbar_wait(&q_full[qst], (gs / QST) & 1u);       // ordered after the poller's acquire of flag (bh, c)
                uint4 ol[8];
                {
                    const uint4* src = reinterpret_cast<const uint4*>(p.Ol + ((long long)bh * NT + c) * 128 * D) + (ct * 8) * 128 + row;
#pragma unroll
                    for (int i = 0; i < 8; ++i) ol[i] = __ldcg(src + i * 128);
                }
                mbar_wait(&out_full[gs & 1], (gs >> 1) & 1u);
                tc_fence_after();
                float v[64];
                tmem_ld64(tmem_addr(tmem + 64 + 64 * (gs & 1), ew * 32, 0), v);
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&out_free[gs & 1]);
                const uint32_t stg = smem_u32(sQ + qst * L::Q_BYTES);
#pragma unroll
                for (int ch = 0; ch < 8; ++ch) {
                    float f[8];
                    unpack8(ol[ch], f);
#pragma unroll
                    for (int e = 0; e < 8; ++e) f[e] = p.scale * (v[8 * ch + e] + f[e]);
                    st_shared_v4(stg + swz_chunk_off(row, ch, 0), pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
                }
                fence_proxy_async();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (warp == 8 && lane == 0) {
                    tma_store_5d(tmO, sQ + qst * L::Q_BYTES, ct * 64, h, c * 128, 0, b);
                    tma_store_commit();
                    tma_store_wait_read();
                    mbar_arrive(&q_empty[qst]);
                }
            }
        }
        if (warp == 8 && lane == 0) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 256);
}

// ---------------------------------------------------------------------------------------------------
// prepass worker: persistent loop over its static tile list
// ---------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void prepass_role(uint8_t* smem, const CUtensorMap* tmQ, const CUtensorMap* tmK, const CUtensorMap* tmV,
                                             const CUtensorMap* tmG, const CUtensorMap* tmQt, const FusedParams& fp) {
    const TokParams& p = fp.t;
    tok::PrepassCtx cx;
    uint32_t* tmem_slot;
    tok::prepass_carve<D>(smem, cx, &tmem_slot);
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(cx.bar_kq, 1); mbar_init(cx.bar_v, 1); mbar_init(cx.bar_mma, 1);
        mbar_fence_init();
    }
    if (tid < 32) tmem_alloc(tmem_slot, 512);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    cx.tmem = *tmem_slot;
    const int w = blockIdx.x - fp.NWC, nwp = gridDim.x - fp.NWC;
    const int BH = p.B * p.H, NT = p.NT;
    const int round_tiles = fp.HPR * NT;
    uint32_t it = 0, ph = 0;
    for (int i = w; i < fp.total_tiles; i += nwp, ++it) {
        // chunk-major inside a head group, so the chain workers of the group can follow closely
        const int r = i / round_tiles, il = i - r * round_tiles;
        const int hr = min(fp.HPR, BH - r * fp.HPR);
        const int tile = il / hr, bh = r * fp.HPR + il % hr;
        tok::prepass_tile<D, 128, true>(cx, tmQ, tmK, tmV, tmG, nullptr, tmQt, nullptr, p, bh, tile, it, ph);
        if (tid == 0) {
            tma_store_wait_all();                  // the tile's summaries are complete in global memory
            fence_proxy_async_all();
            __threadfence();
            st_release_gpu(fp.flags + (long long)bh * NT + tile, fp.epoch);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(cx.tmem, 512);
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1)
gdn_tok_fused(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
              const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmG,
              const __grid_constant__ CUtensorMap tmQt, const __grid_constant__ CUtensorMap tmO, const FusedParams fp) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    if ((int)blockIdx.x < fp.NWC) chain_role<D>(smem, &tmG, &tmQt, &tmO, fp);
    else prepass_role<D>(smem, &tmQ, &tmK, &tmV, &tmG, &tmQt, fp);
}

}  // namespace fused
}  // namespace gdn
