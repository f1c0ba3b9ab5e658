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
//                                          S_c (bf16) per chunk, S_k (bf16) per segment, state_out (fp32);
//                                B(bh,k)   the B part of segment k from zero  -> B_c per chunk, B_k of the whole segment;
//                                A(bh,k)   the Gacc part of segment k from zero -> Gacc_c, gacc_c per chunk, and per segment.
//     One step = ONE M = 64 MMA G_c x (bf16 state) with the fp32 master copy of the state row in registers.
//   workers (the rest): a static round-robin list of tile tasks (segments interleaved, so that all chain CTAs of a
//     stream advance together) followed by output tasks, segment-major:
//       segment 0:   O_c = scale (Qt_c S_c + Ol_c)                                   one MMA
//       segment k:   S_c = gacc_c S_k - Gacc_c S_k + B_c, then the same              two MMAs
//     `out` is written exactly once, by a TMA store of the finished tile.
// Hand-over is by epoch-stamped release/acquire flags in global memory (never reset).  Tile tasks wait for nothing,
// chain CTAs wait for tile tasks (and level 2 for the segment scans), output tasks wait for chain CTAs: no cycle.
#pragma once
#include <cuda.h>

#include "gdn_tc_tile64.cuh"

namespace gdn {

struct F64Params;
__host__ __device__ inline int f64_seg_lo(int L0, int L1, int k) { return k == 0 ? 0 : L0 + (k - 1) * L1; }

struct F64Params {
    TokParams t;                 // alpha, beta, S_in, S_out, out, B, H, T, NC (chunks of 64 per stream), scale, log_alpha
    int NS, L0, L1;              // segments per stream; segment 0 has L0 chunks, the others L1 <= L0 (the last one may be
                                 // shorter): segment 0 is longer by about the latency of publishing a segment map, so that the
                                 // maps of the other segments are waiting when its scan arrives at level 2
    int NCH;                     // chain CTAs = BH * (1 + 2 (NS - 1))
    int zG, zN, zSc, zGA, zGs, zBs, zSk;   // first [64][64] bf16 slot of each array in the 3-D workspace map
    long long rQt, rOl;          // first row of Qt / Ol in the 2-D workspace map
    // flag words: low half = epoch of the call that published the item, high half = an fp32 payload
    unsigned long long *f_tile;  // [BH][NC]  tile summaries of chunk c complete; payload gamma_c
    unsigned long long *f_snap;  // [BH][NC]  S_c (segment 0) / B_c (segment k >= 1) stored
    unsigned long long *f_snapA; // [BH][NC]  Gacc_c stored; payload gacc_c
    unsigned long long *f_segA;  // [BH][NS]  Gacc of the whole segment stored; payload gamma of the segment
    unsigned long long *f_segB;  // [BH][NS]  B of the whole segment stored
    unsigned long long *f_segS;  // [BH][NS]  S_k (state at the start of segment k) stored
    unsigned int epoch;
    int n_tile_tasks, n_out_tasks;
};

namespace f64 {



using namespace tc;
using t64::kTile;

__device__ __forceinline__ unsigned long long ld_acquire64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release64(unsigned long long* p, unsigned long long v) {
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ unsigned long long flag_word(unsigned int epoch, float payload) {
    return ((unsigned long long)__float_as_uint(payload) << 32) | (unsigned long long)epoch;
}
__device__ __forceinline__ bool flag_ready(unsigned long long w, unsigned int epoch) { return (unsigned int)w >= epoch; }
__device__ __forceinline__ float flag_payload(unsigned long long w) { return __uint_as_float((unsigned int)(w >> 32)); }
// (Polling with relaxed loads followed by one fence.acq_rel.gpu measured 5 us SLOWER on config 2 than acquire loads.)
__device__ __forceinline__ void acquire_after_poll() {}
// (and relaxed loads with no fence at all, which the memory model does not cover, gained 0.8 us: not taken)
#define ld_relaxed64 ld_acquire64
__device__ __forceinline__ unsigned long long wait_flag(const unsigned long long* f, unsigned int epoch, unsigned int ns = 20) {
    unsigned long long w = ld_relaxed64(f);
    while (!flag_ready(w, epoch)) { __nanosleep(ns); w = ld_relaxed64(f); }
    return w;
}
// Waiting that may last long (output tasks waiting for a chain CTA): poll with RELAXED loads and a long sleep, then take
// the value with one acquire load.  An acquire load invalidates the SM's L1 every time; chain CTAs share the SM.
__device__ __forceinline__ unsigned long long wait_flag_quiet(const unsigned long long* f, unsigned int epoch) {
    unsigned long long w;
    for (;;) {
        asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(w) : "l"(f) : "memory");
        if (flag_ready(w, epoch)) break;
        __nanosleep(500);
    }
    return ld_acquire64(f);
}
__device__ __forceinline__ void fence_proxy_async_global() { asm volatile("fence.proxy.async.global;" ::: "memory"); }
__device__ __forceinline__ void tma_store_wait_but1() { asm volatile("cp.async.bulk.wait_group 1;" ::: "memory"); }

// shared-memory carve-up of a chain CTA (same allocation as a tile worker)
constexpr uint32_t C_STAGE = 2 * kTile;               // G | N of an entry (bf16 [64][64] each)
constexpr uint32_t C_OFF_SB = 2 * C_STAGE;            // two bf16 state operand buffers
constexpr uint32_t C_OFF_GAM = C_OFF_SB + 2 * kTile;  // gamma of the entry in each stage
constexpr uint32_t C_OFF_GH = C_OFF_GAM + 16;         // gamma of every entry done (replayed for the flag payloads), up to 1024 entries

// ---------------------------------------------------------------------------------------------------
// chain CTA.  Warp w owns state rows 16 w .. 16 w + 15 (the TMEM lanes of an M = 64 accumulator), spread over all of its
// 32 threads in the 16x256b fragment layout: 32 state values per thread, no idle lanes.
// The CTA walks a list of ENTRIES (G, N, gamma): the chunks of its segment and, for P, the maps of the segments 1..NS-1
// behind them (level 2).  Before entry e the bf16 operand buffer holds the state that entry e acts on; it is stored as
// the snapshot of that entry.  The chores of a step are spread over three warps so that none of them delays its warp's share
// of the state update: thread 0 issues the MMA, thread 32 stores the snapshot and releases the flag of the previous one,
// thread 64 pulls entry e+1 (its flag word was requested a step earlier, so nothing waits for L2).
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void chain_role(uint8_t* smem, uint32_t tmem, uint64_t* bars, const CUtensorMap* tmM3, const F64Params& fp, int unit) {
    const TokParams& p = fp.t;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int BH = p.B * p.H, NS = fp.NS, NC = p.NC;
    int bh, type, k;                                  // type 0 = P, 1 = B, 2 = A
    if (unit < BH) { bh = unit; type = 0; k = 0; }
    else { const int u = unit - BH; bh = u / (2 * (NS - 1)); const int r = u % (2 * (NS - 1)); k = 1 + (r >> 1); type = 1 + (r & 1); }
    const int c_lo = f64_seg_lo(fp.L0, fp.L1, k), c_hi = min(c_lo + (k == 0 ? fp.L0 : fp.L1), NC);
    const int nchunk = c_hi - c_lo, n = nchunk + (type == 0 ? NS - 1 : 0);
    const int r0 = 16 * warp + (lane >> 2), r1 = r0 + 8, qd = lane & 3;
    const bool add_g = type == 2;
    const uint32_t aSt = smem_u32(smem), aSb = smem_u32(smem + C_OFF_SB), aGam = smem_u32(smem + C_OFF_GAM);
    uint64_t *full = &bars[0], *bar_mma = &bars[2];
    const unsigned int ep = fp.epoch;
    const long long cb = (long long)bh * NC, sb = (long long)bh * NS;
    // entry e -> operands, readiness flags, snapshot slot and flag
    auto e_zg = [&](int e) { return e < nchunk ? fp.zG + (int)cb + c_lo + e : fp.zGs + (int)sb + (e - nchunk + 1); };
    auto e_zn = [&](int e) { return add_g ? -1 : (e < nchunk ? fp.zN + (int)cb + c_lo + e : fp.zBs + (int)sb + (e - nchunk + 1)); };
    auto e_f0 = [&](int e) { return e < nchunk ? fp.f_tile + cb + c_lo + e : fp.f_segA + sb + (e - nchunk + 1); };
    auto e_f1 = [&](int e) -> const unsigned long long* { return e < nchunk ? nullptr : fp.f_segB + sb + (e - nchunk + 1); };
    auto e_snap_z = [&](int e) { return e < nchunk ? (add_g ? fp.zGA : fp.zSc) + (int)cb + c_lo + e : fp.zSk + (int)sb + (e - nchunk + 1); };
    auto e_snap_f = [&](int e) { return e < nchunk ? (add_g ? fp.f_snapA : fp.f_snap) + cb + c_lo + e : fp.f_segS + sb + (e - nchunk + 1); };

    // S[4j], S[4j+1] = state (r0, 8j + 2qd + {0,1});  S[4j+2], S[4j+3] = the same columns of row r1 (tmem_ld_16x64's layout)
    float S[32];
#pragma unroll
    for (int j = 0; j < 32; ++j) S[j] = 0.f;
    if (type == 0 && p.S_in) {
        const float* s0 = p.S_in + ((long long)bh * 64 + r0) * 64 + 2 * qd;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const float2 a = __ldcg(reinterpret_cast<const float2*>(s0 + 8 * j)), b = __ldcg(reinterpret_cast<const float2*>(s0 + 8 * 64 + 8 * j));
            S[4 * j] = a.x; S[4 * j + 1] = a.y; S[4 * j + 2] = b.x; S[4 * j + 3] = b.y;
        }
    }
    // byte offset, inside a swizzled bf16 [64][64] tile, of this thread's column pair in 8-column block j of row r0 / r1;
    // the eight rows of a warp's access hit eight different 16-byte slots: no bank conflicts
    uint32_t o0[8], o1[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) { o0[j] = swz_chunk_off(r0, j, 0) + 4 * qd; o1[j] = swz_chunk_off(r1, j, 0) + 4 * qd; }
    float gacc = 1.f;                                 // gamma accumulated over the entries done so far
    auto publish = [&](int buf) {                     // bf16 copy of the state -> MN-major B operand `buf`
        const uint32_t base = aSb + buf * kTile;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            sts_b32(base + o0[j], pack_bf16(S[4 * j], S[4 * j + 1]));
            sts_b32(base + o1[j], pack_bf16(S[4 * j + 2], S[4 * j + 3]));
        }
        fence_proxy_async();
    };
    // thread 64: entry e is ready (w0 = its first flag word); pull it into stage e & 1
    auto issue_load = [&](int e, unsigned long long w0) {
        const int st = e & 1;
        sts_f32(aGam + st * 4, flag_payload(w0));
        fence_proxy_async_global();
        const int zn = e_zn(e);
        mbar_expect_tx(&full[st], zn >= 0 ? 2 * kTile : kTile);
        tma_load_3d(smem + st * C_STAGE, tmM3, &full[st], 0, 0, e_zg(e));
        if (zn >= 0) tma_load_3d(smem + st * C_STAGE + kTile, tmM3, &full[st], 0, 0, zn);
    };
    unsigned long long nf0 = 0ull, nf1 = 0ull;       // thread 64: flag words of entry e + 1, requested during step e - 1
    if (tid == 64) {
        unsigned long long w0 = wait_flag(e_f0(0), ep);
        if (e_f1(0)) wait_flag(e_f1(0), ep);
        acquire_after_poll();
        issue_load(0, w0);
        if (n > 1) { nf0 = ld_relaxed64(e_f0(1)); nf1 = e_f1(1) ? ld_relaxed64(e_f1(1)) : ~0ull; }
    }
    publish(0);
    __syncthreads();
    auto gam_hist = [&](int e) { return lds_f32(aGam + 16 + (e < 1024 ? e : 1023) * 4); };
    int released = 0;                                 // thread 32: snapshot flags released so far, and gacc before that entry
    float ga_rel = 1.f;
    for (int e = 0; e < n; ++e) {
        const int st = e & 1;
        if (tid == 32) {
            // Snapshot of the state entry e acts on (independent of the entry's operands: issued before waiting for them).
            // Its buffer is rewritten at the end of step e + 1: by then the store must have READ it (checked one step
            // later, cheap).  Flags need COMPLETE stores and a gpu-scope fence, which on a state warp costs more than it
            // buys during the scan (per-step release 55.4 us, batches of four 51.2, none 49.6 on config 2): a chain CTA
            // releases its chunk snapshots when its chunks are done.  The segment-0 CTA does so when it ENTERS level 2
            // (the outputs of segment 0 then run beside level 2) and releases every S_k one step after storing it.
            tma_store_3d(tmM3, smem + C_OFF_SB + st * kTile, 0, 0, e_snap_z(e));
            tma_store_commit();
            asm volatile("cp.async.bulk.wait_group.read 1;" ::: "memory");
            if (type == 0 && e >= nchunk) {
                asm volatile("cp.async.bulk.wait_group 1;" ::: "memory");
                __threadfence();
                for (; released < e; ++released) {
                    asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(e_snap_f(released)), "l"(flag_word(ep, ga_rel)) : "memory");
                    ga_rel *= gam_hist(released);
                }
            }
        }
        mbar_wait(&full[st], (uint32_t)(e >> 1) & 1u);
        if (warp == 0) {
            // issued under elect.sync: with a plain `tid == 0` every tcgen05.mma sits in a ~70-cycle "waterfall" loop
            // (ptxas cannot keep its operands in uniform registers), which on this serial chain is exposed latency
            if (elect_one()) {
                tc_fence_after();
                const uint32_t id = umma_idesc(64, 64, false, true);
                const uint32_t aG = aSt + st * C_STAGE, aB = aSb + st * kTile;
#pragma unroll
                for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aG + s * 32), desc_mnmajor(aB + s * 2048, 0), id, s > 0);
                umma_commit(bar_mma);
            }
            __syncwarp();
            } else if (tid == 64) {
            if (e + 1 < n) {                          // stage (e + 1) & 1 was released by the barrier that ended step e - 1
                while (!flag_ready(nf0, ep)) { __nanosleep(40); nf0 = ld_relaxed64(e_f0(e + 1)); }
                while (!flag_ready(nf1, ep)) { __nanosleep(40); nf1 = ld_relaxed64(e_f1(e + 1)); }
                acquire_after_poll();
                issue_load(e + 1, nf0);
                if (e + 2 < n) { nf0 = ld_relaxed64(e_f0(e + 2)); nf1 = e_f1(e + 2) ? ld_relaxed64(e_f1(e + 2)) : ~0ull; }
            }
        }
        const float gamma = lds_f32(aGam + st * 4);
        {                                             // state-independent half, while the MMA runs
            const uint32_t src = aSt + st * C_STAGE + (add_g ? 0u : kTile);
            const float w = add_g ? gacc : 1.f;
#pragma unroll
            for (int j = 0; j < 8; ++j) {
                const uint32_t a = lds_b32(src + o0[j]), b = lds_b32(src + o1[j]);
                S[4 * j] = fmaf(gamma, S[4 * j], w * bf16lo(a));
                S[4 * j + 1] = fmaf(gamma, S[4 * j + 1], w * bf16hi(a));
                S[4 * j + 2] = fmaf(gamma, S[4 * j + 2], w * bf16lo(b));
                S[4 * j + 3] = fmaf(gamma, S[4 * j + 3], w * bf16hi(b));
            }
        }
        if (tid == 32 && e < 1024) sts_f32(aGam + 16 + e * 4, gamma);
        gacc *= gamma;
        mbar_wait(bar_mma, (uint32_t)e & 1u);
        tc_fence_after();
        {
            float v[32];
            tmem_ld_16x64(tmem_addr(tmem, warp * 32, 0), v);
#pragma unroll
            for (int j = 0; j < 32; ++j) S[j] -= v[j];
        }
        tc_fence_before();
        publish((e + 1) & 1);
        __syncthreads();
    }
    if (tid == 32) {
        tma_store_wait_all();
        __threadfence();                              // the remaining snapshot flags: one fence, then relaxed stores
        for (; released < n; ++released) {            // (payload: gacc before the entry, replayed from the gamma history)
            asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(e_snap_f(released)), "l"(flag_word(ep, ga_rel)) : "memory");
            ga_rel *= gam_hist(released);
        }
        if (type != 0) {
            // the map of the whole segment: Gacc / B at its end (the operand buffer holds it in bf16), gamma of the segment
            tma_store_3d(tmM3, smem + C_OFF_SB + (n & 1) * kTile, 0, 0, (add_g ? fp.zGs : fp.zBs) + (int)sb + k);
            tma_store_commit();
            tma_store_wait_all();
            st_release64((add_g ? fp.f_segA : fp.f_segB) + sb + k, flag_word(ep, gacc));
        }
    }
    if (type == 0 && p.S_out) {
        float* d0 = p.S_out + ((long long)bh * 64 + r0) * 64 + 2 * qd;
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            *reinterpret_cast<float2*>(d0 + 8 * j) = make_float2(S[4 * j], S[4 * j + 1]);
            *reinterpret_cast<float2*>(d0 + 8 * 64 + 8 * j) = make_float2(S[4 * j + 2], S[4 * j + 3]);
        }
    }
}

// ---------------------------------------------------------------------------------------------------
// output task (worker CTA): chunk c of stream bh, segment k.  Thread (warp w, lane l < 16) owns token row 16 w + l.
//   shared memory (offsets of t64): Qt -> OFF_Q, Ol -> OFF_V (the finished tile is staged over it), state operand
//   (S_c, or S_k then S_c) -> OFF_K, Gacc_c -> OFF_PT, B_c -> OFF_X.
// ---------------------------------------------------------------------------------------------------
__device__ __forceinline__ void output_task(uint8_t* smem, uint32_t tmem, uint64_t* bars, const CUtensorMap* tmM3, const CUtensorMap* tmR2,
                                            const CUtensorMap* tmO, const F64Params& fp, int bh, int c, int k, uint32_t& pl, uint32_t& ph,
                                            unsigned long long* pend_flag, unsigned long long pend_val) {
    const TokParams& p = fp.t;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int NC = p.NC, NS = fp.NS;
    const int m = 16 * warp + lane;
    const bool act = lane < 16;
    const uint32_t aS = smem_u32(smem + t64::OFF_K), aQ = smem_u32(smem + t64::OFF_Q), aO = smem_u32(smem + t64::OFF_V);
    const uint32_t aGA = smem_u32(smem + t64::OFF_PT), aB = smem_u32(smem + t64::OFF_X), aVec = smem_u32(smem + t64::OFF_VEC);
    uint64_t *bar_ld = &bars[0], *bar_st = &bars[1], *bar_mma = &bars[2];      // both load barriers complete once per task (as in a tile task)
    const unsigned int ep = fp.epoch;
    const long long ci = (long long)bh * NC + c;
    const bool comp = k > 0;
    if (tid == 0) {
        tma_store_wait_read();                        // the previous task's stores have left the staging buffers
        if (pend_flag) { tma_store_wait_all(); st_release64(pend_flag, pend_val); }
        // the tile's own operands first (they do not depend on S_k), then the state operand on a barrier of its own
        wait_flag_quiet(fp.f_snap + ci, ep);
        if (comp) sts_f32(aVec, flag_payload(wait_flag_quiet(fp.f_snapA + ci, ep)));
        fence_proxy_async_global();
        const int r0 = (int)(ci * 64);
        mbar_expect_tx(bar_ld, (comp ? 4u : 2u) * kTile);
        tma_load_2d(smem + t64::OFF_Q, tmR2, bar_ld, 0, (int)(fp.rQt + r0));
        tma_load_2d(smem + t64::OFF_V, tmR2, bar_ld, 0, (int)(fp.rOl + r0));
        if (comp) {
            tma_load_3d(smem + t64::OFF_PT, tmM3, bar_ld, 0, 0, fp.zGA + (int)ci);
            tma_load_3d(smem + t64::OFF_X, tmM3, bar_ld, 0, 0, fp.zSc + (int)ci);
            wait_flag_quiet(fp.f_segS + (long long)bh * NS + k, ep);
            fence_proxy_async_global();
        }
        mbar_expect_tx(bar_st, kTile);
        tma_load_3d(smem + t64::OFF_K, tmM3, bar_st, 0, 0, comp ? fp.zSk + bh * NS + k : fp.zSc + (int)ci);
        mbar_wait(bar_ld, pl);
        mbar_wait(bar_st, pl);
    }
    // Only thread 0 polls (flags, then the load barrier); the others sleep in the CTA barrier instead of spinning on the
    // mbarrier: this CTA shares its SM with chain CTAs whose steps are the critical path.
    __syncthreads();
    auto wait_mma = [&]() { mbar_wait(bar_mma, ph); ph ^= 1; tc_fence_after(); };
    mbar_wait(bar_ld, pl);
    mbar_wait(bar_st, pl);
    pl ^= 1u;
    if (comp) {
        // S_c = gacc_c S_k - Gacc_c S_k + B_c: one MMA on the bf16 S_k, fp32 combination, S_c (bf16) over S_k
        if (tid == 0) {
            tc_fence_after();
            const uint32_t id = umma_idesc(64, 64, false, true);
#pragma unroll
            for (int s = 0; s < 4; ++s) umma_bf16(tmem, desc_kmajor(aGA + s * 32), desc_mnmajor(aS + s * 2048, 0), id, s > 0);
            umma_commit(bar_mma);
        }
        const float ga = lds_f32(aVec);
        float S[64];
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc) {
                float f[8], g[8];
                unpack8(ld_shared_v4(aS + swz_chunk_off(m, cc, 0)), f);
                unpack8(ld_shared_v4(aB + swz_chunk_off(m, cc, 0)), g);
#pragma unroll
                for (int e = 0; e < 8; ++e) S[8 * cc + e] = fmaf(ga, f[e], g[e]);
            }
        }
        wait_mma();
#pragma unroll
        for (int hc = 0; hc < 4; ++hc) {
            float v[16];
            tmem_ld16(tmem_addr(tmem, warp * 32, hc * 16), v);
#pragma unroll
            for (int j = 0; j < 16; ++j) S[hc * 16 + j] -= v[j];
        }
        tc_fence_before();
        if (act) {
#pragma unroll
            for (int cc = 0; cc < 8; ++cc)
                st_shared_v4(aS + swz_chunk_off(m, cc, 0), pack_bf16(S[8 * cc], S[8 * cc + 1]), pack_bf16(S[8 * cc + 2], S[8 * cc + 3]),
                             pack_bf16(S[8 * cc + 4], S[8 * cc + 5]), pack_bf16(S[8 * cc + 6], S[8 * cc + 7]));
        }
        fence_proxy_async();
        tc_fence_before();
        __syncthreads();
    }
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
    // Roles: the first NCH CTAs are chain CTAs (the block scheduler hands CTAs to SMs in index order, so they are resident
    // before any worker and spread over distinct SMs), the rest are workers.
    const int my_unit = (int)blockIdx.x < fp.NCH ? (int)blockIdx.x : -1;
    if (my_unit >= 0) {
        chain_role(smem, tmem, bars, &tmM3, fp, my_unit);
    } else {
        t64::Tile64Maps mp{&tmQ, &tmK, &tmV, &tmM3, &tmM3, &tmR2, &tmR2, fp.zG, fp.zN, (long long)p.NC * 64, fp.rQt, fp.rOl};
        uint32_t pl = 0, ph = 0;
        const int total = fp.n_tile_tasks + fp.n_out_tasks;
        // task -> (is tile task, stream, chunk, segment); chunk >= NC: nothing to do (the last segment is shorter)
        auto decode = [&](int task, bool& tile, int& bh, int& c, int& k) {
            tile = task < fp.n_tile_tasks;
            const int tt = tile ? task : task - fp.n_tile_tasks;
            int j;
            if (tile) {                               // segments interleaved: (j, k, bh)
                j = tt / (fp.NS * BH);
                const int r = tt % (fp.NS * BH);
                k = r / BH; bh = r % BH;
            } else {                                  // segment-major: (k, j, bh)
                k = tt / (fp.L0 * BH);
                const int r = tt % (fp.L0 * BH);
                bh = r % BH; j = r / BH;
            }
            c = f64_seg_lo(fp.L0, fp.L1, k) + j;
            if (j >= (k == 0 ? fp.L0 : fp.L1)) c = p.NC;
        };
        unsigned long long* pend_flag = nullptr;      // flag of this CTA's last tile task, released inside the next task
        unsigned long long pend_val = 0ull;
        const uint32_t aRaw = smem_u32(smem + t64::OFF_RAW);
        int raw_sel = 0;                              // raw gate buffer of the current task
        bool have_cur = false, first_tile = true;
        // static round-robin over the workers: waves of tile tasks complete in task order (the chain CTAs consume them
        // in that order), and the task after this one is known in advance (its inputs are prefetched during this one).
        // (A dynamic queue -- one atomic counter, the next task claimed a task ahead -- measured 15 us slower on config 2.)
        const int nworkers = (int)gridDim.x - fp.NCH;
        int task = (int)blockIdx.x - fp.NCH;
        while (task < total) {
            const int next = task + nworkers;
            bool tile, ntile = false;
            int bh, c, k, nbh = 0, nc = 0, nk = 0;
            decode(task, tile, bh, c, k);
            if (next < total) decode(next, ntile, nbh, nc, nk);
            const bool have_next = next < total && ntile && nc < p.NC;
            if (have_next) {
                // the next chunk's gates -> the other raw buffer with 4-byte asynchronous copies (padding rows:
                // alpha = 1, beta = 0), its K / Q / V tiles -> L2
                if (tid < 128) {
                    const int j = tid & 63, t = nc * 64 + j;
                    const bool is_b = tid >= 64;
                    const uint32_t dst = aRaw + (uint32_t)(raw_sel ^ 1) * 512u + (uint32_t)tid * 4u;
                    if (t < p.T) {
                        const float* src = (is_b ? p.beta : p.alpha) + (long long)nbh * p.T + t;
                        asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
                    } else {
                        sts_f32(dst, is_b ? 0.f : (p.log_alpha ? 0.f : 1.f));
                    }
                    asm volatile("cp.async.commit_group;" ::: "memory");
                }
                if (tid == 0) {
                    const int b = nbh / p.H, h = nbh % p.H;
                    tma_prefetch_5d(&tmK, 0, h, nc * 64, 0, b);
                    tma_prefetch_5d(&tmQ, 0, h, nc * 64, 0, b);
                    tma_prefetch_5d(&tmV, 0, h, nc * 64, 0, b);
                }
            }
            if (c < p.NC) {
                if (tile) {
                    if (tid == 0) tma_store_wait_read();  // the previous task's stores have left the staging buffers
                    float gam_c = 0.f;
                    t64::tile64<true>(smem, tmem, bars, mp, p, bh, c, pl, ph, have_cur ? aRaw + (uint32_t)raw_sel * 512u : 0u, pend_flag, pend_val, &gam_c);
                    pend_flag = fp.f_tile + (long long)bh * p.NC + c;
                    pend_val = flag_word(fp.epoch, gam_c);
                    if (first_tile) {                 // the chain CTAs are waiting for the first wave: publish it at once
                        if (tid == 0) { tma_store_wait_all(); st_release64(pend_flag, pend_val); }
                        pend_flag = nullptr;
                        first_tile = false;
                    }
                } else {
                    output_task(smem, tmem, bars, &tmM3, &tmR2, &tmO, fp, bh, c, k, pl, ph, pend_flag, pend_val);
                    pend_flag = nullptr;
                }
            }
            asm volatile("cp.async.wait_all;" ::: "memory");
            raw_sel ^= 1;
            have_cur = have_next;
            task = next;
            __syncthreads();
        }
        if (tid == 0) {
            tma_store_wait_all();
            if (pend_flag) st_release64(pend_flag, pend_val);
        }
    }
    tc_fence_before();
    __syncthreads();
    if (tid < 32) tmem_dealloc(tmem, 128);
}

}  // namespace f64
}  // namespace gdn
