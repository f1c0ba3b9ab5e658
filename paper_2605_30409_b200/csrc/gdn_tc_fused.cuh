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
// the same for global memory only: the flag acquire (generic proxy) before the TMA loads of what the flag guards
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }


template <int D>
struct ChainSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t G_BYTES = (uint32_t)D * D * 2;          // NB blocks of [D][64] bf16
    static constexpr uint32_t N_BYTES = (uint32_t)D * 64 * 2;         // one block of [D][64] bf16 (this CTA's 64 state columns)
    static constexpr uint32_t GN_BYTES = G_BYTES + N_BYTES;
    static constexpr uint32_t Q_BYTES = 128u * D * 2;                 // NB blocks of [128][64] bf16; block 0 then stages the out tile
    static constexpr uint32_t S_BYTES = (uint32_t)D * 128;            // [D][64] bf16
    // d = 64: six stages each (the chain CTA has the SM to itself: 216 KB): a step moves 48 KB through one SM's TMA path, and
    // with three stages in flight that path ran at the latency-bound ~50 GB/s (config 2: 41.6 -> 41.15 us)
    static constexpr int GST = (D == 128) ? 2 : 6;
    static constexpr int QST = (D == 128) ? 2 : 6;
    static constexpr int NSB = (D == 128) ? 2 : 3;                    // bf16 state operand buffers
    static constexpr uint32_t OFF_Q = GST * GN_BYTES;
    static constexpr uint32_t OFF_S = OFF_Q + QST * Q_BYTES;
    static constexpr uint32_t OFF_BAR = OFF_S + NSB * S_BYTES;
    static constexpr uint32_t OFF_GAM = OFF_BAR + 384;                // [GST] gamma_c of the chunk in the stage
    static constexpr uint32_t TOTAL = OFF_BAR + 512;
};

template <int D>
constexpr uint32_t fused_smem_bytes() {
    return (ChainSmem<D>::TOTAL > tok::prepass_smem_bytes<D>() ? ChainSmem<D>::TOTAL : tok::prepass_smem_bytes<D>()) + 1024u;
}

// ---------------------------------------------------------------------------------------------------
// chain worker.  warps 0-7: state rows (thread = row m x 32 columns); 8-11: output epilogue (thread = token
// row); 12: chain MMA issuer; 13: flag poller + TMA producer of the chain's operands; 14: output MMA issuer; 15: flag
// poller + TMA producer of the output's Qt tiles.
// The chain (warps 0-7) and the output (warps 8-11) only meet at the bf16 state operand buffers: the output
// of chunk c reads S_c while the chain is already up to NSB - 1 steps further on.
// ---------------------------------------------------------------------------------------------------
template <int D>
__device__ __forceinline__ void chain_role(uint8_t* smem, const CUtensorMap* tmG, const CUtensorMap* tmN, const CUtensorMap* tmQt,
                                           const CUtensorMap* tmO, const FusedParams& fp) {
    using L = ChainSmem<D>;
    constexpr int NB = L::NB, GST = L::GST, QST = L::QST, NSB = L::NSB, NCT = D / 64;
    const TokParams& p = fp.t;
    uint8_t* sG = smem;
    uint8_t* sQ = smem + L::OFF_Q;
    uint8_t* sS = smem + L::OFF_S;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* g_full = bars;                  // [GST] TMA: G_c and N_c landed (gamma_c written before the arm)
    uint64_t* g_empty = g_full + GST;         // [GST] chain MMA of the step has completed and the 8 state warps have read gamma_c, N_c
    uint64_t* q_full = g_empty + GST;         // [QST] TMA: Qt tile landed
    uint64_t* q_empty = q_full + QST;         // [QST] the out tile staged in the buffer has left
    uint64_t* s_ready = q_empty + QST;        // [NSB] bf16 state operand published (8 warps)
    uint64_t* s_free = s_ready + NSB;         // [NSB] the output MMA that read the buffer has completed
    uint64_t* mma_chain = s_free + NSB;       // chain MMA complete
    uint64_t* out_full = mma_chain + 1;       // [2] output MMA complete
    uint64_t* out_free = out_full + 2;        // [2] output accumulator drained (4 warps)
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(out_free + 2);
    float* sGamma = reinterpret_cast<float*>(smem + L::OFF_GAM);
    const uint32_t a_issued = smem_u32(smem + L::OFF_GAM + 64);       // chain MMAs issued so far (shared-space word)
    auto issued_ld = [&]() { uint32_t v; asm volatile("ld.volatile.shared.u32 %0, [%1];" : "=r"(v) : "r"(a_issued) : "memory"); return v; };
    auto issued_st = [&](uint32_t v) { asm volatile("st.volatile.shared.u32 [%0], %1;" ::"r"(a_issued), "r"(v) : "memory"); };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    if (tid == 0) {
        for (int s = 0; s < GST; ++s) { mbar_init(&g_full[s], 1); mbar_init(&g_empty[s], 9); }
        for (int s = 0; s < QST; ++s) { mbar_init(&q_full[s], 1); mbar_init(&q_empty[s], 1); }
        for (int s = 0; s < NSB; ++s) { mbar_init(&s_ready[s], 8); mbar_init(&s_free[s], 1); }
        mbar_init(mma_chain, 1);
        for (int s = 0; s < 2; ++s) { mbar_init(&out_full[s], 1); mbar_init(&out_free[s], 4); }
        mbar_fence_init();
        issued_st(0u);
    }
    if (warp == 0) tmem_alloc(tmem_slot, 256);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    // The kernel is launched as a programmatic dependent of whatever precedes it in the stream (normally the previous call's
    // launch of this kernel): its CTAs take the SMs as the previous grid's CTAs leave, set themselves up, and wait here,
    // before their first global access, until that grid has completed.
    pdl_launch_dependents();
    pdl_wait();
    const uint32_t acc_chain = tmem;
    const int NT = p.NT;
    const int nunits = p.B * p.H * NCT;

    if (warp == 13 || warp == 15) {
        // ===== flag pollers + TMA producers: warp 13 feeds the chain (G_c, N_c, gamma_c), warp 15 the output (Qt).  Two
        // producers, because the Qt ring also stages the outgoing tiles and recycles at the pace of the output path: in one
        // in-order producer a late q_empty held back the NEXT chunk's G / N and with it the serial chain.
        // The 32 lanes poll the flags of the next 32 chunks together (one L2 round trip for all of them);
        // the elected lane issues the loads of every chunk in the ready prefix.
        const bool feed_chain = warp == 13;
        uint32_t gs = 0;
        for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
            const int bh = u / NCT, ct = u % NCT;
            int ready = 0, base = 0;                         // chunks [0, ready) of this unit are published
            float gam_l = 0.f;                               // gamma of chunk base + lane (valid below `ready`)
            for (int c = 0; c < NT; ++c, ++gs) {
                while (c >= ready) {
                    base = ready;
                    const int idx = base + lane;
                    const bool ok = idx < NT && ld_acquire_gpu(fp.flags + (long long)bh * NT + idx) >= fp.epoch;
                    const uint32_t m = __ballot_sync(0xffffffffu, ok);
                    ready += (m == 0xffffffffu) ? 32 : (__ffs(~m) - 1);      // length of the ready prefix
                    if (feed_chain && idx < ready) {         // accepted exactly once per chunk
                        gam_l = __ldcg(p.gam + (long long)bh * p.NC + idx);
                        if (GST < 3) {                       // shallow ring: have the summaries waiting in L2
                            fence_proxy_async_global();
                            const int z = bh * p.NC + idx;
#pragma unroll
                            for (int nb = 0; nb < NB; ++nb) tma_prefetch_3d(tmG, nb * 64, 0, z);
                            tma_prefetch_3d(tmN, ct * 64, 0, z);
                        }
                    }
                    if (c >= ready) __nanosleep(32);
                }
                const float gam_c = __shfl_sync(0xffffffffu, gam_l, c - base);
                if (lane == 0) {
                    fence_proxy_async_global();
                    if (feed_chain) {
                        const int gst = gs % GST;
                        if (gs >= (uint32_t)GST) mbar_wait(&g_empty[gst], ((gs / GST) - 1) & 1u);
                        sts_f32(smem_u32(sGamma) + gst * 4, gam_c);      // visible to the waiters of g_full through the arrive below
                        mbar_expect_tx(&g_full[gst], L::GN_BYTES);
                        uint8_t* gb = sG + gst * L::GN_BYTES;
                        const int z = bh * p.NC + c;
#pragma unroll
                        for (int nb = 0; nb < NB; ++nb) tma_load_3d(gb + nb * (D * 128), tmG, &g_full[gst], nb * 64, 0, z);
                        tma_load_3d(gb + L::G_BYTES, tmN, &g_full[gst], ct * 64, 0, z);
                    } else {
                        const int qst = gs % QST;
                        if (gs >= (uint32_t)QST) mbar_wait(&q_empty[qst], ((gs / QST) - 1) & 1u);
                        mbar_expect_tx(&q_full[qst], L::Q_BYTES);
                        uint8_t* qb = sQ + qst * L::Q_BYTES;
#pragma unroll
                        for (int nb = 0; nb < NB; ++nb) tma_load_2d(qb + nb * kBlk, tmQt, &q_full[qst], nb * 64, (bh * NT + c) * 128);
                    }
                }
                __syncwarp();
            }
        }
    } else if (warp == 12) {
        // ===== chain MMA issuer: acc = G_c (A, K-major) * S_c (B, MN-major), the moment the operand is published.
        // Nothing else is issued by this thread: its commit covers the chain MMA only, and no output MMA's issue sits
        // between a publication and the chain MMA that waits for it.  Issued under elect.sync: with a plain `lane == 0`
        // every tcgen05.mma sits in a ~70-cycle "waterfall" loop (ELECT / R2UR / BRA.U.ANY) because ptxas cannot keep
        // its operands in uniform registers -- on this serial chain that is exposed latency (~450 cycles per step).
        if (elect_one()) {
            const uint32_t idc = umma_idesc(D, 64, false, true);
            const uint32_t total = (uint32_t)((nunits - (int)blockIdx.x + fp.NWC - 1) / fp.NWC) * (uint32_t)NT;   // steps of this CTA
            for (uint32_t gs = 0; gs < total; ++gs) {
                const int gst = gs % GST, sb = gs % NSB;
                mbar_wait(&g_full[gst], (gs / GST) & 1u);
                mbar_wait(&s_ready[sb], (gs / NSB) & 1u);
                tc_fence_after();
                const uint32_t aG = smem_u32(sG + gst * L::GN_BYTES), aS = smem_u32(sS + sb * L::S_BYTES);
#pragma unroll
                for (int s = 0; s < D / 16; ++s)
                    umma_bf16(acc_chain, desc_kmajor(aG + (s >> 2) * (D * 128) + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), idc, s > 0);
                umma_commit(mma_chain);
                umma_commit(&g_empty[gst]);
                issued_st(gs + 1);                                   // the output issuer lets the chain MMA of a step go first
            }
        }
    } else if (warp == 14) {
        // ===== output MMA issuer: acc_out = Qt_c (A) * S_c (B), in the shadow of the chain's TMEM -> register ->
        // shared-memory round trip; may lag the chain by up to NSB - 1 steps (s_free gates the reuse of an operand buffer).
        if (lane == 0) {
            const uint32_t ido = umma_idesc(128, 64, false, true);
            const uint32_t total = (uint32_t)((nunits - (int)blockIdx.x + fp.NWC - 1) / fp.NWC) * (uint32_t)NT;
            for (uint32_t o = 0; o < total; ++o) {
                const int qst = o % QST, sb = o % NSB;
                mbar_wait(&s_ready[sb], (o / NSB) & 1u);             // S_o is published
                mbar_wait(&q_full[qst], (o / QST) & 1u);
                if (o >= 2) mbar_wait(&out_free[o & 1], ((o >> 1) - 1) & 1u);
                while (issued_ld() <= o) {}
                tc_fence_after();
                const uint32_t aQ = smem_u32(sQ + qst * L::Q_BYTES), aS = smem_u32(sS + sb * L::S_BYTES);
                const uint32_t acc_out = tmem + 64 + 64 * (o & 1);
#pragma unroll
                for (int s = 0; s < D / 16; ++s)
                    umma_bf16(acc_out, desc_kmajor(aQ + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aS + s * 2048, 0), ido, s > 0);
                umma_commit(&out_full[o & 1]);
                umma_commit(&s_free[sb]);
            }
        }
    } else if (warp < 8) {
        // ===== state rows: S <- (gamma_c S + N_c) - G_c S =====
        const int wq = warp & 3, half = warp >> 2;
        const int m = (D == 128) ? (wq * 32 + lane) : (16 * wq + lane);     // state row (M = 64 uses lanes 0-15 of a quadrant)
        const bool m_ok = (D == 128) || (lane < 16);
        const int mm = m_ok ? m : 0;
        float S[32];
        uint32_t gs = 0;                                                    // steps done; also the index of the next publication
        for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
            const int bh = u / NCT, ct = u % NCT;
            const int col0 = ct * 64 + half * 32;
            if (m_ok && m < p.dr && p.S_in) {
                const float4* src = reinterpret_cast<const float4*>(p.S_in + ((long long)bh * p.dr + m) * p.dr + col0);
#pragma unroll
                for (int i = 0; i < 8; ++i) {
                    const float4 f = (col0 + 4 * i < p.dr) ? __ldcg(src + i) : make_float4(0.f, 0.f, 0.f, 0.f);
                    S[4 * i] = f.x; S[4 * i + 1] = f.y; S[4 * i + 2] = f.z; S[4 * i + 3] = f.w;
                }
            } else {
#pragma unroll
                for (int i = 0; i < 32; ++i) S[i] = 0.f;
            }
            // publication `pi` (= the state at the start of step pi) goes to operand buffer pi % NSB
            auto publish = [&](uint32_t pi) {
                const uint32_t sb = pi % NSB;
                if (pi >= (uint32_t)NSB) mbar_wait(&s_free[sb], ((pi / NSB) - 1) & 1u);   // output MMA of step pi - NSB is done with it
                if (m_ok) {
                    const uint32_t sbase = smem_u32(sS + sb * L::S_BYTES);
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch)
                        st_shared_v4(sbase + swz_chunk_off(m, half * 4 + ch, 0), pack_bf16(S[8 * ch], S[8 * ch + 1]), pack_bf16(S[8 * ch + 2], S[8 * ch + 3]),
                                     pack_bf16(S[8 * ch + 4], S[8 * ch + 5]), pack_bf16(S[8 * ch + 6], S[8 * ch + 7]));
                }
                fence_proxy_async();
                __syncwarp();
                if (lane == 0) mbar_arrive(&s_ready[sb]);
            };
            publish(gs);
            for (int c = 0; c < NT; ++c, ++gs) {
                const int gst = gs % GST;
                mbar_wait(&g_full[gst], (gs / GST) & 1u);
                // N_c's 64-column block of this CTA has been read for the only time (no other CTA loads these lines; the next
                // call rewrites them): dropped from L2 without a write-back to DRAM (config 3: DRAM writes 170 -> 123 MB, the
                // call 178.4 -> 176.3 us).  G_c and Qt_c are read by both column CTAs of a head; dropping them from the last
                // reader (a counter per tile, 4 discards per output-epilogue thread and step) brought the writes down to
                // 57 MB but cost time where the chain is the bound (config 5: 180 -> 210 us): not done.
                if (half == 0 && m_ok) {
                    const char* nl = reinterpret_cast<const char*>(p.Nw) + ((((long long)bh * p.NC + c) * D + m) * D + ct * 64) * 2;
                    asm volatile("discard.global.L2 [%0], 128;" ::"l"(nl) : "memory");
                }
                const float gamma_c = lds_f32(smem_u32(sGamma) + gst * 4);
                {   // state-independent half, while the MMA runs: S <- gamma_c S + N_c
                    const uint32_t nbase = smem_u32(sG + gst * L::GN_BYTES + L::G_BYTES);
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch) {
                        float f[8];
                        unpack8(ld_shared_v4(nbase + swz_chunk_off(mm, half * 4 + ch, 0)), f);
#pragma unroll
                        for (int e = 0; e < 8; ++e) S[8 * ch + e] = fmaf(gamma_c, S[8 * ch + e], f[e]);
                    }
                }
                __syncwarp();
                if (lane == 0) mbar_arrive(&g_empty[gst]);                   // gamma_c and N_c of the stage have been read
                mbar_wait(mma_chain, gs & 1u);
                tc_fence_after();
                {
                    float v[32];
                    tmem_ld32(tmem_addr(acc_chain, wq * 32, half * 32), v);
#pragma unroll
                    for (int i = 0; i < 32; ++i) S[i] -= v[i];
                }
                tc_fence_before();
                if (c + 1 < NT) publish(gs + 1);
            }
            if (m_ok && m < p.dr) {
                float4* dst = reinterpret_cast<float4*>(p.S_out + ((long long)bh * p.dr + m) * p.dr + col0);
#pragma unroll
                for (int i = 0; i < 8; ++i)
                    if (col0 + 4 * i < p.dr) dst[i] = make_float4(S[4 * i], S[4 * i + 1], S[4 * i + 2], S[4 * i + 3]);
            }
        }
    } else if (warp < 12) {
        // ===== output epilogue: out += scale * acc_out (the prepass already stored scale * Ol there): the tile is
        //       staged as bf16 in block 0 of the Qt buffer and leaves as a TMA reduction (add) =====
        const int ew = warp - 8;
        const int row = ew * 32 + lane;
        uint32_t gs = 0;
        int prev_qst = -1;
        for (int u = blockIdx.x; u < nunits; u += fp.NWC) {
            const int bh = u / NCT, ct = u % NCT;
            const int b = bh / p.H, h = bh % p.H;
            for (int c = 0; c < NT; ++c, ++gs) {
                const int qst = gs % QST;
                mbar_wait(&out_full[gs & 1], (gs >> 1) & 1u);         // implies q_full of the stage
                tc_fence_after();
                const uint32_t stg = smem_u32(sQ + qst * L::Q_BYTES);
#pragma unroll
                for (int hf = 0; hf < 2; ++hf) {
                    float v[32];
                    tmem_ld32(tmem_addr(tmem + 64 + 64 * (gs & 1), ew * 32, hf * 32), v);
                    if (hf == 1) {
                        tc_fence_before();
                        __syncwarp();
                        if (lane == 0) mbar_arrive(&out_free[gs & 1]);
                    }
#pragma unroll
                    for (int ch = 0; ch < 4; ++ch)
                        st_shared_v4(stg + swz_chunk_off(row, hf * 4 + ch, 0),
                                     pack_bf16(p.scale * v[8 * ch], p.scale * v[8 * ch + 1]), pack_bf16(p.scale * v[8 * ch + 2], p.scale * v[8 * ch + 3]),
                                     pack_bf16(p.scale * v[8 * ch + 4], p.scale * v[8 * ch + 5]), pack_bf16(p.scale * v[8 * ch + 6], p.scale * v[8 * ch + 7]));
                }
                fence_proxy_async();
                asm volatile("bar.sync 1, 128;" ::: "memory");
                if (warp == 8 && lane == 0) {
                    // the slot goes back to the producer once the reduction has READ it: checked one step later, so that this
                    // thread (and with it the next step's barrier) does not sit out the read of the tile it has just sent
                    // (deep ring only: with two slots the late release starves the producer -- config 5 180 -> 270 us)
                    tma_reduce_add_5d(tmO, sQ + qst * L::Q_BYTES, ct * 64, h, c * 128, 0, b);
                    tma_store_commit();
                    if (QST >= 4) {
                        tma_store_wait_read_but1();
                        if (prev_qst >= 0) mbar_arrive(&q_empty[prev_qst]);
                        prev_qst = qst;
                    } else {
                        tma_store_wait_read();
                        mbar_arrive(&q_empty[qst]);
                    }
                }
            }
        }
        if (warp == 8 && lane == 0) {
            tma_store_wait_read();
            if (prev_qst >= 0) mbar_arrive(&q_empty[prev_qst]);
            tma_store_wait_all();
        }
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
                                             const CUtensorMap* tmG, const CUtensorMap* tmN, const CUtensorMap* tmQt,
                                             const CUtensorMap* tmOl, const FusedParams& fp) {
    const TokParams& p = fp.t;
    tok::PrepassCtx cx;
    uint32_t* tmem_slot;
    tok::prepass_carve<D>(smem, cx, &tmem_slot);
    const int tid = threadIdx.x;
    if (tid == 0) {
        mbar_init(cx.bar_kq, 1); mbar_init(cx.bar_q, 1); mbar_init(cx.bar_v, 1); mbar_init(cx.bar_mma, 1); mbar_init(cx.bar_mma2, 1);
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
    unsigned int* pending = nullptr;
    float2 gates = make_float2(0.f, 0.f);          // this thread's alpha, beta of the next tile (prefetched a tile ahead)
    auto tile_of = [&](int i, int& bh, int& tile) {
        // chunk-major inside a head group, so the chain workers of the group can follow closely
        const int r = i / round_tiles, il = i - r * round_tiles;
        const int hr = min(fp.HPR, BH - r * fp.HPR);
        tile = il / hr; bh = r * fp.HPR + il % hr;
    };
    // (see chain_role)  The first tile's operands are the caller's: asked into L2 while the previous grid finishes.
    pdl_launch_dependents();
    if (tid == 0 && w < fp.total_tiles) {
        constexpr int NBp = D / 64;
        int bh0, t0;
        tile_of(w, bh0, t0);
#pragma unroll
        for (int nb = 0; nb < NBp; ++nb) {
            tma_prefetch_5d(tmK, nb * 64, bh0 % p.H, t0 * 128, 0, bh0 / p.H);
            tma_prefetch_5d(tmQ, nb * 64, bh0 % p.H, t0 * 128, 0, bh0 / p.H);
            tma_prefetch_5d(tmV, nb * 64, bh0 % p.H, t0 * 128, 0, bh0 / p.H);
        }
    }
    pdl_wait();
    for (int i = w; i < fp.total_tiles; i += nwp, ++it) {
        int bh, tile, nbh = -1, ntile = -1;
        tile_of(i, bh, tile);
        if (i + nwp < fp.total_tiles) tile_of(i + nwp, nbh, ntile);
        // the previous tile's ready flag is published inside this tile, once its stores have completed
        tok::prepass_tile<D, 128, true>(cx, tmQ, tmK, tmV, tmG, tmN, tmQt, tmOl, p, bh, tile, it, ph, pending, fp.epoch, nbh, ntile, &gates);
        pending = fp.flags + (long long)bh * NT + tile;
    }
    if (D == 128 && tid == tok::kPrepassFlagTid && pending) tma_store_wait_all();      // this thread's share of the last tile's stores
    __syncthreads();
    if (tid == 0 && pending) {
        tma_store_wait_all();                      // the last tile's summaries are complete in global memory ...
        st_release_gpu(pending, fp.epoch);         // ... and the release orders them (and this thread's gamma store) before the flag
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(cx.tmem, 512);
}

template <int D>
__global__ void __launch_bounds__(kThreads, 1)
gdn_tok_fused(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK,
              const __grid_constant__ CUtensorMap tmV, const __grid_constant__ CUtensorMap tmG,
              const __grid_constant__ CUtensorMap tmN, const __grid_constant__ CUtensorMap tmQt,
              const __grid_constant__ CUtensorMap tmO, const FusedParams fp) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    if ((int)blockIdx.x < fp.NWC) chain_role<D>(smem, &tmG, &tmN, &tmQt, &tmO, fp);
    else prepass_role<D>(smem, &tmQ, &tmK, &tmV, &tmG, &tmN, &tmQt, &tmO, fp);
}

}  // namespace fused
}  // namespace gdn
