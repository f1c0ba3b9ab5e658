// gdn_tc_fused64.cuh -- token-wise (G = 1) Gated DeltaNet forward, d = 64, as ONE persistent kernel of light CTAs with a
// TWO-LEVEL (segment-parallel) scan over the per-chunk affine maps.
//
// Chunks of C = 64 tokens; chunk c of a stream acts on the state as the affine map
//     S_{c+1} = gamma_c S_c - G_c S_c + N_c,        O_c = scale (Qt_c S_c + Ol_c),
// with (G_c, N_c, gamma_c, Qt_c, Ol_c) state-independent (t64::tile64).  Affine maps compose (Eq. 5:
// S_f = alpha_f P_f S_{f-1} + A_f; the columns of the state are independent, L419-L423), so the chunks of a stream are cut
// into NS segments and each segment k >= 1 is scanned FROM THE IDENTITY MAP while segment 0 is scanned from state_in:
//     prefix map of chunk c in segment k:   S_c = gacc_c S_k - Gacc_c S_k + B_c        (S_k = state at the segment start)
//     Gacc_{c+1} = gamma_c Gacc_c + gacc_c G_c - G_c Gacc_c,   B_{c+1} = gamma_c B_c - G_c B_c + N_c,   gacc_{c+1} = gamma_c gacc_c
// (the identity part of the map is kept as the fp32 scalar gacc, so only the small correction Gacc is rounded to bf16).
// Level 2 is the same step over the NS segment maps, and the outputs are a parallel fix-up once S_k is known.
//
// All CTAs have the footprint of a tile worker (128 threads, ~56 KB, 128 TMEM columns; four per SM).  Roles by blockIdx:
//   chain CTAs (the first NCH):  P(bh)     plain scan of segment 0 from state_in, then the NS-1 level-2 steps; leaves
//                                          S_c (bf16) per chunk, S_k (fp32) per segment, state_out;
//                                B(bh,k)   the B part of segment k from zero  -> B_c per chunk, B_k of the whole segment;
//                                A(bh,k)   the Gacc part of segment k from zero -> Gacc_c, gacc_c per chunk, and per segment.
//     One step = ONE M = 64 MMA G_c x (bf16 state) with the fp32 master copy of the state row in registers.
//   workers (the rest): a dynamic queue (one atomic counter) of tile tasks (segments interleaved, so that all chain CTAs
//     of a stream advance together) followed by output tasks, segment-major:
//       segment 0:   O_c = scale (Qt_c S_c + Ol_c)                                   one MMA
//       segment k:   S_c = gacc_c S_k - Gacc_c S_k + B_c, then the same              two MMAs
//     `out` is written exactly once, by a TMA store of the finished tile.
// Hand-over is by epoch-stamped release/acquire flags in global memory (never reset).  Tile tasks wait for nothing,
// chain CTAs wait for tile tasks (and level 2 for the segment scans), output tasks wait for chain CTAs: no cycle.
#pragma once
#include <cuda.h>

#include "gdn_tc_tile64.cuh"

namespace gdn {

struct F64Params {
    TokParams t;                 // alpha, beta, S_in, S_out, out, gam, B, H, T, NC (chunks of 64 per stream), scale, log_alpha
    int NS, LSEG;                // segments per stream, chunks per segment (the last segment may be shorter)
    int NCH;                     // chain CTAs = BH * (1 + 2 (NS - 1))
    int zG, zN, zSc, zGA, zGs, zBs;     // first [64][64] bf16 slot of each array in the 3-D workspace map
    long long rQt, rOl;          // first row of Qt / Ol in the 2-D workspace map
    float* gacc;                 // [BH][NC]  gacc_c (prefix inside its segment)
    float* gseg;                 // [BH][NS]  gamma of the whole segment
    float* SegS;                 // [BH][NS][64][64] fp32 state at the start of segment k >= 1
    unsigned int *f_tile, *f_snap, *f_snapA;      // [BH][NC]
    unsigned int *f_segA, *f_segB, *f_segS;       // [BH][NS]
    unsigned int epoch;
    unsigned int* ctr;           // [0] task counter, [1] finished CTAs (the last one resets both)
    int n_tile_tasks, n_out_tasks;
};

namespace f64 {

using namespace tc;
using t64::kTile;

__device__ __forceinline__ unsigned int ld_acquire_gpu(const unsigned int* p) {
    unsigned int v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_gpu(unsigned int* p, unsigned int v) {
    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(p), "r"(v) : "memory");
}
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void wait_flag(const unsigned int* f, unsigned int epoch) {
    while (ld_acquire_gpu(f) < epoch) __nanosleep(20);
}
__device__ __forceinline__ void tma_store_wait_but1() { asm volatile("cp.async.bulk.wait_group 1;" ::: "memory"); }

// shared-memory carve-up of a chain CTA (same allocation as a tile worker)
constexpr uint32_t C_STAGE = 2 * kTile;               // G_c | N_c (bf16 [64][64] each)
constexpr uint32_t C_OFF_SB = 2 * C_STAGE;            // two bf16 state operand buffers
constexpr uint32_t C_OFF_GAM = C_OFF_SB + 2 * kTile;  // gamma of the chunk in each stage

// ---------------------------------------------------------------------------------------------------
// chain CTA.  Thread (warp w, lane l < 16) owns state row m = 16 w + l (the TMEM lanes of an M = 64 accumulator);
// thread 0 is also the producer (flag polling, TMA) and the MMA issuer.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_role(uint8_t* smem, uint32_t tmem, uint64_t* bars, const CUtensorMap* tmM3, const F64Params& fp, int unit) {
    const TokParams& p = fp.t;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int BH = p.B * p.H, NS = fp.NS, NC = p.NC;
    int bh, type, k;                                  // type 0 = P, 1 = B, 2 = A
    if (unit < BH) { bh = unit; type = 0; k = 0; }
    else { const int u = unit - BH; bh = u / (2 * (NS - 1)); const int r = u % (2 * (NS - 1)); k = 1 + (r >> 1); type = 1 + (r & 1); }
    const int c_lo = k * fp.LSEG, c_hi = min(c_lo + fp.LSEG, NC);
    const int m = 16 * warp + lane;
    const bool act = lane < 16;
    const uint32_t aSt = smem_u32(smem), aSb = smem_u32(smem + C_OFF_SB), aGam = smem_u32(smem + C_OFF_GAM);
    uint64_t *full = &bars[0], *bar_mma = &bars[2];
    const unsigned int ep = fp.epoch;

    float S[64];
#pragma unroll
    for (int j = 0; j < 64; ++j) S[j] = 0.f;
    if (type == 0 && act && p.S_in) {
        const float4* src = reinterpret_cast<const float4*>(p.S_in + ((long long)bh * 64 + m) * 64);
#pragma unroll
        for (int q = 0; q < 16; ++q) { const float4 f = __ldcg(src + q); S[4 * q] = f.x; S[4 * q + 1] = f.y; S[4 * q + 2] = f.z; S[4 * q + 3] = f.w; }
    }
    float gacc = 1.f;
    auto publish = [&](int buf) {                     // bf16 copy of the state rows -> MN-major B operand `buf`
        if (act) {
            const uint32_t base = aSb + buf * kTile;
#pragma unroll
            for (int c = 0; c < 8; ++c)
                st_shared_v4(base + swz_chunk_off(m, c, 0), pack_bf16(S[8 * c], S[8 * c + 1]), pack_bf16(S[8 * c + 2], S[8 * c + 3]),
                             pack_bf16(S[8 * c + 4], S[8 * c + 5]), pack_bf16(S[8 * c + 6], S[8 * c + 7]));
        }
        fence_proxy_async();
    };
    // thread 0: wait for the flags of an entry, then pull its operands into stage `st`
    auto issue_load = [&](int st, int zg, int zn, const unsigned int* f0, const unsigned int* f1, const float* gsrc) {
        wait_flag(f0, ep);
        if (f1) wait_flag(f1, ep);
        sts_f32(aGam + st * 4, __ldcg(gsrc));
        fence_proxy_async_global();
        mbar_expect_tx(&full[st], zn >= 0 ? 2 * kTile : kTile);
        tma_load_3d(smem + st * C_STAGE, tmM3, &full[st], 0, 0, zg);
        if (zn >= 0) tma_load_3d(smem + st * C_STAGE + kTile, tmM3, &full[st], 0, 0, zn);
    };
    uint32_t nstep = 0;                               // steps done (stage / operand buffer / parity bookkeeping)
    // One step on the entry loaded in stage nstep & 1.  add_g: the additive term is gacc G_c (type A) instead of N_c.
    // Thread 0, behind the MMA issue: stores the operand buffer (= the state BEFORE this entry) as snapshot `snap_z`,
    // releases the flag of the previous snapshot (whose store has had a whole step to complete), pulls the next entry.
    auto step = [&](bool add_g, int snap_z, unsigned int* prev_flag, float* gacc_dst, bool has_next, int nzg, int nzn,
                    const unsigned int* nf0, const unsigned int* nf1, const float* ngsrc) {
        const int st = nstep & 1;
        mbar_wait(&full[st], (nstep >> 1) & 1u);
        if (tid == 0) {
            tc_fence_after();
            const uint32_t id = umma_idesc(64, 64, false, true);
            const uint32_t aG = aSt + st * C_STAGE, aB = aSb + (nstep & 1) * kTile;
#pragma unroll
            for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aG + s * 32), desc_mnmajor(aB + s * 2048, 0), id, s > 0);
            umma_commit(bar_mma);
            if (gacc_dst) *gacc_dst = gacc;
            if (snap_z >= 0) { tma_store_3d(tmM3, smem + C_OFF_SB + (nstep & 1) * kTile, 0, 0, snap_z); tma_store_commit(); }
            if (prev_flag) {
                if (snap_z >= 0) tma_store_wait_but1(); else tma_store_wait_all();
                st_release_gpu(prev_flag, ep);
            }
            if (has_next) issue_load(st ^ 1, nzg, nzn, nf0, nf1, ngsrc);
        }
        const float gamma = lds_f32(aGam + st * 4);
        if (act) {                                    // state-independent half, while the MMA runs
            const uint32_t src = aSt + st * C_STAGE + (add_g ? 0u : kTile);
            const float w = add_g ? gacc : 1.f;
#pragma unroll
            for (int c = 0; c < 8; ++c) {
                float f[8];
                unpack8(ld_shared_v4(src + swz_chunk_off(m, c, 0)), f);
#pragma unroll
                for (int e = 0; e < 8; ++e) S[8 * c + e] = fmaf(gamma, S[8 * c + e], w * f[e]);
            }
        }
        gacc *= gamma;
        mbar_wait(bar_mma, nstep & 1u);
        tc_fence_after();
#pragma unroll
        for (int hc = 0; hc < 2; ++hc) {
            float v[32];
            tmem_ld32(tmem_addr(tmem, warp * 32, hc * 32), v);
#pragma unroll
            for (int j = 0; j < 32; ++j) S[hc * 32 + j] -= v[j];
        }
        tc_fence_before();
        ++nstep;
        publish(nstep & 1);
        __syncthreads();
    };

    // ---- the chunks of this CTA's segment ----
    const bool add_g = type == 2;
    const int zsnap0 = (type == 2 ? fp.zGA : fp.zSc) + bh * NC;
    unsigned int* fsnap = (type == 2 ? fp.f_snapA : fp.f_snap) + (long long)bh * NC;
    const unsigned int* ftile = fp.f_tile + (long long)bh * NC;
    const float* gam = p.gam + (long long)bh * NC;
    const int zg0 = fp.zG + bh * NC, zn0 = fp.zN + bh * NC;
    if (tid == 0) issue_load(0, zg0 + c_lo, add_g ? -1 : zn0 + c_lo, ftile + c_lo, nullptr, gam + c_lo);
    publish(0);
    __syncthreads();
    for (int c = c_lo; c < c_hi; ++c) {
        const bool nx = c + 1 < c_hi;
        step(add_g, zsnap0 + c, c > c_lo ? fsnap + c - 1 : nullptr, add_g ? fp.gacc + (long long)bh * NC + c : nullptr,
             nx, zg0 + c + 1, add_g ? -1 : zn0 + c + 1, ftile + c + 1, nullptr, gam + c + 1);
    }
    if (tid == 0) { tma_store_wait_all(); st_release_gpu(fsnap + c_hi - 1, ep); }

    if (type != 0) {
        // the map of the whole segment: Gacc / B at its end (the operand buffer holds it in bf16), gamma of the segment
        if (tid == 0) {
            const int idx = bh * NS + k;
            tma_store_3d(tmM3, smem + C_OFF_SB + (nstep & 1) * kTile, 0, 0, (type == 2 ? fp.zGs : fp.zBs) + idx);
            tma_store_commit();
            if (type == 2) fp.gseg[idx] = gacc;
            tma_store_wait_all();
            st_release_gpu((type == 2 ? fp.f_segA : fp.f_segB) + idx, ep);
        }
        return;
    }
    // ---- level 2 (type P): S_{k+1} = gseg_k S_k - Gs_k S_k + Bs_k over the segment maps ----
    for (int kk = 1; kk < NS; ++kk) {
        const int idx = bh * NS + kk;
        if (act) {
            float4* dst = reinterpret_cast<float4*>(fp.SegS + ((long long)idx * 64 + m) * 64);
#pragma unroll
            for (int q = 0; q < 16; ++q) __stcg(dst + q, make_float4(S[4 * q], S[4 * q + 1], S[4 * q + 2], S[4 * q + 3]));
        }
        __syncthreads();
        if (tid == 0) {
            __threadfence();
            st_release_gpu(fp.f_segS + idx, ep);
            issue_load(nstep & 1, fp.zGs + idx, fp.zBs + idx, fp.f_segA + idx, fp.f_segB + idx, fp.gseg + idx);
        }
        step(false, -1, nullptr, nullptr, false, 0, 0, nullptr, nullptr, nullptr);
    }
    if (act && p.S_out) {
        float4* dst = reinterpret_cast<float4*>(p.S_out + ((long long)bh * 64 + m) * 64);
#pragma unroll
        for (int q = 0; q < 16; ++q) dst[q] = make_float4(S[4 * q], S[4 * q + 1], S[4 * q + 2], S[4 * q + 3]);
    }
}

// ---------------------------------------------------------------------------------------------------
// output task (worker CTA): chunk c of stream bh, segment k.  Thread (warp w, lane l < 16) owns token row 16 w + l.
//   shared memory (offsets of t64): Qt -> OFF_Q, Ol -> OFF_V (the finished tile is staged over it), state operand -> OFF_K,
//   Gacc_c -> OFF_PT, B_c -> OFF_X.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void output_task(uint8_t* smem, uint32_t tmem, uint64_t* bars, const CUtensorMap* tmM3, const CUtensorMap* tmR2,
                                            const CUtensorMap* tmO, const F64Params& fp, int bh, int c, int k, uint32_t& pl, uint32_t& ph) {
    const TokParams& p = fp.t;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int NC = p.NC, NS = fp.NS;
    const int m = 16 * warp + lane;
    const bool act = lane < 16;
    const uint32_t aS = smem_u32(smem + t64::OFF_K), aQ = smem_u32(smem + t64::OFF_Q), aO = smem_u32(smem + t64::OFF_V);
    const uint32_t aGA = smem_u32(smem + t64::OFF_PT), aB = smem_u32(smem + t64::OFF_X);
    uint64_t *bar_ld = &bars[0], *bar_mma = &bars[2];
    const unsigned int ep = fp.epoch;
    const long long ci = (long long)bh * NC + c;
    const bool comp = k > 0;
    if (tid == 0) {
        tma_store_wait_read();                        // the previous task's stores have left the staging buffers
        wait_flag(fp.f_snap + ci, ep);
        if (comp) wait_flag(fp.f_snapA + ci, ep);
        fence_proxy_async_global();
        const int r0 = (int)(ci * 64);
        mbar_expect_tx(bar_ld, (comp ? 4u : 3u) * kTile);
        tma_load_2d(smem + t64::OFF_Q, tmR2, bar_ld, 0, (int)(fp.rQt + r0));
        tma_load_2d(smem + t64::OFF_V, tmR2, bar_ld, 0, (int)(fp.rOl + r0));
        if (comp) {
            tma_load_3d(smem + t64::OFF_PT, tmM3, bar_ld, 0, 0, fp.zGA + (int)ci);
            tma_load_3d(smem + t64::OFF_X, tmM3, bar_ld, 0, 0, fp.zSc + (int)ci);
        } else {
            tma_load_3d(smem + t64::OFF_K, tmM3, bar_ld, 0, 0, fp.zSc + (int)ci);
        }
        if (comp) wait_flag(fp.f_segS + (long long)bh * NS + k, ep);
    }
    auto sync_then_issue = [&]() { fence_proxy_async(); tc_fence_before(); __syncthreads(); };
    auto wait_mma = [&]() { mbar_wait(bar_mma, ph); ph ^= 1; tc_fence_after(); };
    if (comp) {
        // S_c = gacc_c S_k - Gacc_c S_k + B_c: S_k (fp32, global) -> registers and bf16 operand; one MMA; fp32 combination
        __syncthreads();                              // thread 0 has seen the flag of S_k
        float S[64];
        const float4* src = reinterpret_cast<const float4*>(fp.SegS + (((long long)bh * NS + k) * 64 + (act ? m : 0)) * 64);
#pragma unroll
        for (int q = 0; q < 16; ++q) { const float4 f = __ldcg(src + q); S[4 * q] = f.x; S[4 * q + 1] = f.y; S[4 * q + 2] = f.z; S[4 * q + 3] = f.w; }
        const float ga = __ldcg(fp.gacc + ci);
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc)
                st_shared_v4(aS + swz_chunk_off(m, cc, 0), pack_bf16(S[8 * cc], S[8 * cc + 1]), pack_bf16(S[8 * cc + 2], S[8 * cc + 3]),
                             pack_bf16(S[8 * cc + 4], S[8 * cc + 5]), pack_bf16(S[8 * cc + 6], S[8 * cc + 7]));
        }
        mbar_wait(bar_ld, pl);
        sync_then_issue();
        if (tid == 0) {
            tc_fence_after();
            const uint32_t id = umma_idesc(64, 64, false, true);
#pragma unroll
            for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aGA + s * 32), desc_mnmajor(aS + s * 2048, 0), id, s > 0);
            umma_commit(bar_mma);
        }
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) {
                float f[8];
                unpack8(ld_shared_v4(aB + swz_chunk_off(m, cc, 0)), f);
#pragma unroll
                for (int e = 0; e < 8; ++e) S[8 * cc + e] = fmaf(ga, S[8 * cc + e], f[e]);
            }
        }
        wait_mma();
#pragma unroll
        for (int hc = 0; hc < 2; ++hc) {
            float v[32];
            tmem_ld32(tmem_addr(tmem, warp * 32, hc * 32), v);
#pragma unroll
            for (int j = 0; j < 32; ++j) S[hc * 32 + j] -= v[j];
        }
        tc_fence_before();
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc)
                st_shared_v4(aS + swz_chunk_off(m, cc, 0), pack_bf16(S[8 * cc], S[8 * cc + 1]), pack_bf16(S[8 * cc + 2], S[8 * cc + 3]),
                             pack_bf16(S[8 * cc + 4], S[8 * cc + 5]), pack_bf16(S[8 * cc + 6], S[8 * cc + 7]));
        }
        sync_then_issue();
    } else {
        mbar_wait(bar_ld, pl);
    }
    pl ^= 1u;
    // O_c = scale (Qt_c S_c + Ol_c)
    if (tid == 0) {
        tc_fence_after();
        const uint32_t id = umma_idesc(64, 64, false, true);
#pragma unroll
        for (int s = 0; s < 4; ++s) umma_bf16(tmem + 64, desc_kmajor(aQ + s * 32), desc_mnmajor(aS + s * 2048, 0), id, s > 0);
        umma_commit(bar_mma);
    }
    wait_mma();
#pragma unroll
    for (int hc = 0; hc < 2; ++hc) {
        float v[32];
        tmem_ld32(tmem_addr(tmem + 64, warp * 32, hc * 32), v);
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 4; ++cc) {
                const uint32_t off = swz_chunk_off(m, hc * 4 + cc, 0);
                float f[8];
                unpack8(ld_shared_v4(aO + off), f);
#pragma unroll
                for (int e = 0; e < 8; ++e) f[e] = p.scale * (v[8 * cc + e] + f[e]);
                st_shared_v4(aO + off, pack_bf16(f[0], f[1]), pack_bf16(f[2], f[3]), pack_bf16(f[4], f[5]), pack_bf16(f[6], f[7]));
            }
        }
    }
    fence_proxy_async();
    tc_fence_before();
    __syncthreads();
    if (tid == 0) {
        tma_store_5d(tmO, smem + t64::OFF_V, 0, bh % p.H, c * 64, 0, bh / p.H);
        tma_store_commit();
    }
}

// ---------------------------------------------------------------------------------------------------
// the kernel: grid = 4 CTAs per SM (or fewer when there is less work)
// ---------------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(t64::kThreads, 4)
gdn_tok_fused64(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                const __grid_constant__ CUtensorMap tmO, const __grid_constant__ CUtensorMap tmM3, const __grid_constant__ CUtensorMap tmR2,
                const F64Params fp) {
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + t64::OFF_BAR);
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bars + 4);
    int* s_task = reinterpret_cast<int*>(bars + 5);
    const int tid = threadIdx.x;
    if (tid == 0) {
        for (int s = 0; s < 4; ++s) mbar_init(&bars[s], 1);
        mbar_fence_init();
    }
    if (tid < 32) tmem_alloc(tmem_slot, 128);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    const TokParams& p = fp.t;
    const int BH = p.B * p.H;
    if ((int)blockIdx.x < fp.NCH) {
        chain_role(smem, tmem, bars, &tmM3, fp, (int)blockIdx.x);
    } else {
        t64::Tile64Maps mp{&tmQ, &tmK, &tmV, &tmM3, &tmM3, &tmR2, &tmR2, fp.zG, fp.zN, (long long)p.NC * 64, fp.rQt, fp.rOl};
        uint32_t pl = 0, ph = 0;
        const int total = fp.n_tile_tasks + fp.n_out_tasks;
        for (;;) {
            if (tid == 0) *s_task = (int)atomicAdd(fp.ctr, 1u);
            __syncthreads();
            const int task = *s_task;
            __syncthreads();
            if (task >= total) break;
            const int tt = task < fp.n_tile_tasks ? task : task - fp.n_tile_tasks;
            int bh, c, k;
            if (task < fp.n_tile_tasks) {             // segments interleaved: (j, k, bh)
                const int j = tt / (fp.NS * BH), r = tt % (fp.NS * BH);
                k = r / BH; bh = r % BH; c = k * fp.LSEG + j;
            } else {                                  // segment-major: (k, j, bh)
                k = tt / (fp.LSEG * BH);
                const int r = tt % (fp.LSEG * BH);
                bh = r % BH; c = k * fp.LSEG + r / BH;
            }
            if (c >= p.NC) continue;                  // the last segment is shorter
            if (task < fp.n_tile_tasks) {
                if (tid == 0) tma_store_wait_read();  // an output task before this one may still be reading its staging
                t64::tile64<true>(smem, tmem, bars, mp, p, bh, c, pl, ph);
                if (tid == 0) {
                    tma_store_wait_all();
                    st_release_gpu(fp.f_tile + (long long)bh * p.NC + c, fp.epoch);
                }
            } else {
                output_task(smem, tmem, bars, &tmM3, &tmR2, &tmO, fp, bh, c, k, pl, ph);
            }
        }
        if (tid == 0) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(tmem, 128);
    if (tid == 0) {
        __threadfence();
        if (atomicAdd(fp.ctr + 1, 1u) == gridDim.x - 1) { fp.ctr[0] = 0u; fp.ctr[1] = 0u; __threadfence(); }
    }
}

}  // namespace f64
}  // namespace gdn
