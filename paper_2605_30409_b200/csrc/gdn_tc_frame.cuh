// gdn_tc_frame.cuh -- frame-wise (G = tokens per frame) Gated DeltaNet forward on tcgen05 tensor cores:
// the paper's own variant (Eq. 4-5, Alg. 1), re-designed for sm_100a.
//
//   Phase A  gdn_frm_summaries : per (b,h,f) and token split, [Gram | A] = (diag(beta) K)^T [K | V]
//                                token-contraction MMAs (M = d, N = 2d, K = tokens) fed by a TMA ring.  The B
//                                operand [K | V] is the TMA tile itself; only the A operand diag(beta) K is a
//                                thread-written copy.  Both are MN-major views, no transposes.
//                                Token splits of a frame leave fp32 partials in the workspace; the LAST split CTA
//                                to finish (a counter per frame) sums them in fixed split order -> G_f = alpha_f
//                                Gram_f (bf16), N_f = A_f (fp32), gamma_f = alpha_f: deterministic, no atomics on
//                                data, no separate reduction launch.
//   Phase B  gdn_tok_chain     : S_f = alpha_f S_{f-1} - G_f S_{f-1} + N_f  -- the same one-MMA-per-step chain
//                                kernel as the token-wise path (Eq. 5: S_f = alpha_f (I - Gram_f) S_{f-1} + A_f)
//   (bidirectional scan, Alg. 1 l.9-21: forward and reverse scan in ONE launch; both ADD their snapshots into slots that
//    Phase A zeroes (TMA reduction), so Phase C reads S^hist = S> + S< with no second output pass, L122)
//   Phase C  gdn_frm_readout   : O_f = scale * Q_f S_f  (every token of frame f reads the post-update state, Eq. 22)
//                                persistent CTAs over contiguous tile ranges: TMA ring for Q, S_f reloaded only when
//                                the frame changes, two TMEM accumulators, bf16 tiles leave by TMA store.
//
// Tokens beyond the end of a frame inside a 128-token tile are zero-filled by the 5-D tensor map
// (d, H, G, F, B) and get beta = 0: they contribute nothing; on the way out the same map clips them.
#pragma once
#include <cuda.h>

#include "gdn_tc_token.cuh"

namespace gdn {

struct FrmParams {
    const float* alpha;          // [BH][F]
    const float* beta;           // [BH][T]
    void* out;                   // [B][T][H][D] bf16
    float* part;                 // [BH*F][NSPLIT][D][2D] fp32 partial summaries (NSPLIT > 1)
    unsigned int* counters;      // [BH*F] split CTAs that have delivered their partial (self-resetting)
    __nv_bfloat16* Gw;           // [BH][F][D][D]
    float* Nw;                   // [BH][F][D][D]
    float* gam;                  // [BH][F]
    int B, H, T, G, F, NSPLIT, TPF;   // TPF = 128-token tiles per frame
    int NSc;                     // snapshot slots per (b,h) = F + 1
    int total_tiles;             // BH * F * TPF (readout)
    long long o_ts;
    float scale;
    int log_alpha;
    // normaliser (Eq. 20-22): the vector state z is run through the SAME Phase A and scan kernels as column 0 of a
    // matrix state ("the z path is the matrix path with v = 1", SURVEY pin 13): zpass = 1 replaces V by a constant block whose
    // column 0 is one, so N_f[:, 0] = K^T beta = b_f and Gram is that of the un-rotated keys.  The readout of the MATRIX pass
    // forms den = q_raw . z_f itself (den_mode 1): z_f is column 0 of the z pass's state snapshots z_sc, the q_raw tile of a
    // token tile rides in the last slot of the Q ring, and out = scale Q S / (den + eps).
    int zpass;
    int den_mode;                // readout: 0 = plain, 1 = normalised
    float eps;
    const __nv_bfloat16* z_sc;   // [BH][NSc][D][D] bf16 snapshots of the z pass (slot f + 1 = the state frame f reads)
    // Phase A, bidirectional path: slot f + 1 of these snapshots [BH][NSc][D][D] is zeroed (this CTA's column block): both
    // scans add their states into it (TokParams::snap_add).  NULL = off.
    __nv_bfloat16* zero_sc;
    // output gate (Eq. 23, the Hadamard product G (.) Y): multiplied in the readout's epilogue, before the
    // bf16 rounding of the tile.  gate [B][T][H][dr] bf16, token stride g_ts; NULL = no gate.
    const __nv_bfloat16* gate;
    long long g_ts;
    int dr;                      // real head dim (112 when padded to D = 128): channels >= dr are clipped by the store
    // readout: q_rot / q_raw when they are the plan's OWN feature buffers (gdn_forward_chunk_full; dense [B][T][H][D]): a tile that
    // has been consumed is dropped from L2 (discard.global.L2), so the dead intermediate is never written back to DRAM.
    // NULL = the caller's memory, left alone.
    const __nv_bfloat16* drop_q;
    const __nv_bfloat16* drop_qr;
};

namespace frm {

using namespace tc;
using tok::kBlk;
using tok::st_global_v4;

constexpr int kSumThreads = 192;       // warps 0-3: beta scaling + epilogue; warp 4: MMA issuer; warp 5: TMA producer

// NC = column split of the summary [Gram | A] across CTAs (d = 128: 2).  CTA j of a frame computes the 64-column
// block j of Gram and of A over the tokens of its split: it loads K whole (the A operand is diag(beta) K with all d
// features) plus V block j, and its B operand is [K block j | V block j].  No CTA adds to another one's columns,
// so without a token split there are no partials and no reduction at all.
template <int D>
constexpr int sum_nc() { return D == 128 ? 2 : 1; }

template <int D>
struct SumSmem {
    static constexpr int NB = D / 64;
    static constexpr int NC = sum_nc<D>();
    static constexpr uint32_t KTILE = NB * kBlk;                      // [128 tokens][D] bf16
    static constexpr int VB = NB / NC;                                // V blocks of this CTA
    static constexpr uint32_t STAGE = KTILE + VB * kBlk;              // K tile, then this CTA's V block(s)
    static constexpr int STAGES = (D == 128) ? 3 : 4;
    static constexpr int SCB = 2;                                     // diag(beta) K copies (the A operand)
    static constexpr uint32_t OFF_SC = STAGES * STAGE;
    static constexpr uint32_t OFF_ONE = OFF_SC + SCB * KTILE;         // z pass: constant [128][64] block standing in for V
    static constexpr uint32_t OFF_BAR = OFF_ONE + kBlk;
    static constexpr uint32_t TOTAL = OFF_BAR + 512 + 1024;
};

// ---------------------------------------------------------------------------------------------------
// Phase A.  grid = BH*F*NSPLIT*NC, block = 192.
// ---------------------------------------------------------------------------------------------------
template <int D>
__global__ void __launch_bounds__(kSumThreads, 1)
gdn_frm_summaries(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV, const FrmParams p) {
    using L = SumSmem<D>;
    constexpr int NB = L::NB, NC = L::NC;
    constexpr int STAGES = L::STAGES, SCB = L::SCB;
    constexpr int NW = 2 * D / NC;                // accumulator columns of this CTA: [Gram cols | A cols]
    constexpr int HW = D / NC;                    // columns of each of the two halves
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* bar_full = bars;                    // [STAGES] TMA: K and V tiles landed
    uint64_t* bar_empty = bar_full + STAGES;      // [STAGES] the MMAs that read the stage have completed
    uint64_t* bar_scaled = bar_empty + STAGES;    // [SCB] diag(beta) K written (4 warps)
    uint64_t* bar_sfree = bar_scaled + SCB;       // [SCB] the MMAs that read the copy have completed
    uint64_t* bar_done = bar_sfree + SCB;
    uint8_t* sSc = smem + L::OFF_SC;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_done + 1);
    uint32_t* last_flag = tmem_slot + 1;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int j = blockIdx.x % NC;                // column block
    const int split = (blockIdx.x / NC) % p.NSPLIT;
    const int bhf = blockIdx.x / (NC * p.NSPLIT);
    const int f = bhf % p.F, bh = bhf / p.F;
    const int b = bh / p.H, h = bh % p.H;
    // contiguous range of 128-token tiles of this frame handled by this split
    const int per = (p.TPF + p.NSPLIT - 1) / p.NSPLIT;
    const int tile_lo = split * per;
    const int tile_hi = min(p.TPF, tile_lo + per);
    const int ntiles = max(0, tile_hi - tile_lo);

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_empty[s], 1); }
        for (int s = 0; s < SCB; ++s) { mbar_init(&bar_scaled[s], 4); mbar_init(&bar_sfree[s], 1); }
        mbar_init(bar_done, 1);
        mbar_fence_init();
    }
    if (tid == 160) { tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV); }      // descriptor fetch off the first loads' path
    if (warp == 0) tmem_alloc(tmem_slot, NW);
    const bool zp = p.zpass != 0;
    if (zp && tid < 128) {
        // row `tid` of the constant block: column 0 = 1 (first column block only), everything else 0
        const uint32_t one = smem_u32(smem + L::OFF_ONE);
#pragma unroll
        for (int c = 0; c < 8; ++c) st_shared_v4(one + swz_chunk_off(tid, c, 0), (c == 0 && j == 0) ? 0x00003F80u : 0u, 0u, 0u, 0u);
        fence_proxy_async();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();                                    // no-op unless launched as a dependent of the front-end kernel (gdn_forward_chunk_full)
    pdl_launch_dependents();

    if (warp == 5) {
        // ===== TMA producer =====
        if (elect_one()) {
            // The ring holds what fits in shared memory (three tiles); the DRAM latency of a tile (~3500 cycles measured from
            // issue to arrival with the ring alone) is taken earlier, by an L2 prefetch kPF tiles ahead of the load.
            constexpr int kPF = 3;
            const uint64_t pol = l2_policy_evict_first();      // K and V are streamed (K is read by the sibling column CTA within a tile time)
            auto prefetch = [&](int i) {
                const int n0 = (tile_lo + i) * 128;
                if (j == 0) {                     // the column CTAs of a frame read the same K: one of them prefetches it
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) tma_prefetch_5d(&tmK, nb * 64, h, n0, f, b);
                }
                if (zp) return;
                if (NC == 1) {
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) tma_prefetch_5d(&tmV, nb * 64, h, n0, f, b);
                } else {
                    tma_prefetch_5d(&tmV, j * 64, h, n0, f, b);
                }
            };
            for (int i = STAGES; i < min(ntiles, STAGES + kPF); ++i) prefetch(i);
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES;
                if (i >= STAGES) mbar_wait(&bar_empty[st], (uint32_t)((i / STAGES) - 1) & 1u);
                if (i + kPF < ntiles && i >= STAGES) prefetch(i + kPF);
                uint8_t* base = smem + st * L::STAGE;
                mbar_expect_tx(&bar_full[st], zp ? L::KTILE : L::STAGE);
                const int n0 = (tile_lo + i) * 128;
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(base + nb * kBlk, &tmK, &bar_full[st], nb * 64, h, n0, f, b, pol);
                if (zp) continue;                  // no V: the constant block stands in
                if (NC == 1) {
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(base + (NB + nb) * kBlk, &tmV, &bar_full[st], nb * 64, h, n0, f, b, pol);
                } else {
                    tma_load_5d_hint(base + NB * kBlk, &tmV, &bar_full[st], j * 64, h, n0, f, b, pol);
                }
            }
        }
    } else if (warp == 4) {
        // ===== MMA issuer: [Gram | A] += (beta K)^T [K | V]  (A = the scaled copy, B = the stage's 64-column blocks; MN-major) =====
        if (elect_one()) {
            const uint32_t id = umma_idesc(D, NW, true, true);
            // B: all of K then all of V (NC = 1), or K block j then the V block (NC = 2)
            const uint32_t b_off = (NC == 1) ? 0u : (uint32_t)j * kBlk;
            const uint32_t b_lbo = (NC == 1) ? kBlk : (uint32_t)(NB - j) * kBlk;
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES, sb = i % SCB;
                mbar_wait(&bar_full[st], (uint32_t)(i / STAGES) & 1u);
                mbar_wait(&bar_scaled[sb], (uint32_t)(i / SCB) & 1u);
                tc_fence_after();
                const uint32_t a = smem_u32(sSc + sb * L::KTILE), bq = smem_u32(smem + st * L::STAGE) + b_off;
                // z pass: the block after the K block(s) of this CTA is the constant block (any distance is a legal LBO)
                const uint32_t lbo = zp ? smem_u32(smem + L::OFF_ONE) - (bq + (uint32_t)(NB / NC - 1) * kBlk) : b_lbo;
#pragma unroll
                for (int s = 0; s < 8; ++s)
                    umma_bf16(tmem, desc_mnmajor(a + s * 2048, kBlk), desc_mnmajor(bq + s * 2048, lbo), id, (i > 0 || s > 0) ? 1u : 0u);
                umma_commit(&bar_empty[st]);
                umma_commit(&bar_sfree[sb]);
            }
            umma_commit(bar_done);
        }
    } else {
        // ===== diag(beta) K copy (thread = token row of the tile), then the epilogue =====
        const int row = tid;
        const float* beta_f = p.beta + (long long)bh * p.T + (long long)f * p.G;
        auto load_beta = [&](int i) { const int n = (tile_lo + i) * 128 + row; return (i < ntiles && n < p.G) ? __ldg(beta_f + n) : 0.f; };
        float b_next = load_beta(0);               // one tile ahead: the global-load latency stays off the per-tile path
        for (int i = 0; i < ntiles; ++i) {
            const int st = i % STAGES, sb = i % SCB;
            const float bt = b_next;
            b_next = load_beta(i + 1);
            if (i >= SCB) mbar_wait(&bar_sfree[sb], (uint32_t)((i / SCB) - 1) & 1u);
            mbar_wait(&bar_full[st], (uint32_t)(i / STAGES) & 1u);
            const uint32_t src = smem_u32(smem + st * L::STAGE) + (uint32_t)row * 128u;
            const uint32_t dst = smem_u32(sSc + sb * L::KTILE) + (uint32_t)row * 128u;
            const Bf16Scale bs = bf16_scale(bt);
#pragma unroll
            for (int blk = 0; blk < NB; ++blk) {
                // the scale is per row, so the copy keeps every 16-byte chunk where the swizzle put it; rotating
                // the chunk order by the row index keeps the 8 lanes of a quarter-warp on distinct banks.  All eight
                // loads of a block are issued before the first use (the asm loads are not reordered by the compiler:
                // one load at a time left the warp, alone on its scheduler, waiting out every shared-memory latency).
                uint4 x[8];
#pragma unroll
                for (int c = 0; c < 8; ++c) x[c] = ld_shared_v4(src + blk * kBlk + (uint32_t)(((c + row) & 7) << 4));
#pragma unroll
                for (int c = 0; c < 8; ++c)
                    st_shared_v4(dst + blk * kBlk + (uint32_t)(((c + row) & 7) << 4), bf16x2_scale(x[c].x, bs), bf16x2_scale(x[c].y, bs),
                                 bf16x2_scale(x[c].z, bs), bf16x2_scale(x[c].w, bs));
            }
            fence_proxy_async();
            __syncwarp();
            if (lane == 0) mbar_arrive(&bar_scaled[sb]);
        }
    }

    // ---- epilogue (warps 0-3; thread = summary row m).  Accumulator column c: half c / HW (0 = Gram, 1 = A),
    //      global column j * HW + c % HW --------------------------------------------------------------------
    const int m = (D == 128) ? tid : (16 * warp + lane);
    const bool m_ok = warp < 4 && ((D == 128) || (lane < 16));
    float a_f = p.alpha[bhf];
    if (p.log_alpha) a_f = expf(a_f);
    if (p.zero_sc && warp < 4 && split == 0) {
        __nv_bfloat16* zb = p.zero_sc + (((long long)bh * p.NSc + f + 1) * D) * D + j * HW;
        for (int idx = tid; idx < D * (HW / 8); idx += 128) st_global_v4(zb + (long long)(idx / (HW / 8)) * D + (idx % (HW / 8)) * 8, 0u, 0u, 0u, 0u);
    }
    if (p.NSPLIT == 1) {
        // no token split: G_f = alpha_f Gram_f (bf16), N_f = A_f (fp32).  The rows leave TMEM one per thread; written to global
        // memory like that, every store instruction of a warp touches 32 different lines (measured: ~6 us for 128 KB).  They
        // are staged in shared memory instead (the ring is idle by now; 16-byte chunks XOR-ed with the row index against bank
        // conflicts) and copied out with whole 128- / 256-byte row segments per quarter / half warp.
        static_assert(HW == 64, "staging layout: 64 columns per half");
        constexpr int R = D;                       // summary rows
        if (warp < 4) {
            mbar_wait(bar_done, 0);
            tc_fence_after();
            const uint32_t stgG = smem_u32(smem), stgN = stgG + R * 128;
#pragma unroll 1
            for (int cc = 0; cc < NW / 32; ++cc) {
                float v[32];
                tmem_ld32(tmem_addr(tmem, warp * 32, cc * 32), v);
                if (m_ok) {
                    if (cc < HW / 32) {
#pragma unroll
                        for (int q4 = 0; q4 < 4; ++q4)
                            st_shared_v4(stgG + m * 128 + (uint32_t)(((cc * 4 + q4) ^ (m & 7)) << 4), pack_bf16(a_f * v[8 * q4], a_f * v[8 * q4 + 1]),
                                         pack_bf16(a_f * v[8 * q4 + 2], a_f * v[8 * q4 + 3]), pack_bf16(a_f * v[8 * q4 + 4], a_f * v[8 * q4 + 5]),
                                         pack_bf16(a_f * v[8 * q4 + 6], a_f * v[8 * q4 + 7]));
                    } else {
#pragma unroll
                        for (int q4 = 0; q4 < 8; ++q4)
                            st_shared_v4(stgN + m * 256 + (uint32_t)((((cc - HW / 32) * 8 + q4) ^ (m & 7)) << 4), __float_as_uint(v[4 * q4]),
                                         __float_as_uint(v[4 * q4 + 1]), __float_as_uint(v[4 * q4 + 2]), __float_as_uint(v[4 * q4 + 3]));
                    }
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            __nv_bfloat16* gbase = p.Gw + (long long)bhf * D * D + j * HW;
            float* nbase = p.Nw + (long long)bhf * D * D + j * HW;
#pragma unroll 4
            for (int idx = tid; idx < R * 8; idx += 128) {
                const int row = idx >> 3, c = idx & 7;
                const uint4 u = ld_shared_v4(stgG + row * 128 + (uint32_t)((c ^ (row & 7)) << 4));
                st_global_v4(gbase + (long long)row * D + c * 8, u.x, u.y, u.z, u.w);
            }
#pragma unroll 4
            for (int idx = tid; idx < R * 16; idx += 128) {
                const int row = idx >> 4, c = idx & 15;
                const uint4 u = ld_shared_v4(stgN + row * 256 + (uint32_t)((c ^ (row & 7)) << 4));
                st_global_v4(nbase + (long long)row * D + c * 4, u.x, u.y, u.z, u.w);
            }
            if (tid == 0 && j == 0) p.gam[bhf] = a_f;
        }
    } else {
        // partial [Gram | A] of this split -> workspace (fp32, full-width rows [D][2D]; this CTA owns its columns).  Staged in
        // shared memory like the unsplit epilogue above (row-per-thread global stores touch 32 lines per instruction) and
        // copied out as whole 512-byte row segments, one per warp and instruction.
        if (warp < 4) {
            if (ntiles > 0) {
                mbar_wait(bar_done, 0);
                tc_fence_after();
            }
            constexpr uint32_t ROWB = NW * 4;           // bytes of a staged row: [Gram block | A block] fp32
            constexpr int CH = NW / 4;                  // 16-byte chunks per row
            const uint32_t stg = smem_u32(smem);
#pragma unroll 1
            for (int cc = 0; cc < NW / 32; ++cc) {
                float v[32];
                if (ntiles > 0) {
                    tmem_ld32(tmem_addr(tmem, warp * 32, cc * 32), v);
                } else {
#pragma unroll
                    for (int e = 0; e < 32; ++e) v[e] = 0.f;
                }
                if (m_ok) {
#pragma unroll
                    for (int q4 = 0; q4 < 8; ++q4)
                        st_shared_v4(stg + (uint32_t)m * ROWB + (uint32_t)(((cc * 8 + q4) ^ (m & 7)) << 4), __float_as_uint(v[4 * q4]),
                                     __float_as_uint(v[4 * q4 + 1]), __float_as_uint(v[4 * q4 + 2]), __float_as_uint(v[4 * q4 + 3]));
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            float* pbase = p.part + ((long long)bhf * p.NSPLIT + split) * D * (2 * D) + j * HW;
#pragma unroll 4
            for (int idx = tid; idx < D * CH; idx += 128) {
                const int row = idx / CH, c = idx % CH;
                const uint4 u = ld_shared_v4(stg + (uint32_t)row * ROWB + (uint32_t)((c ^ (row & 7)) << 4));
                const int col = c * 4;
                st_global_v4(pbase + (long long)row * (2 * D) + (col < HW ? col : D + (col - HW)), u.x, u.y, u.z, u.w);
            }
        }
        // the last CTA of the frame to get here reduces all partials in split order
        __threadfence();
        __syncthreads();
        if (tid == 0) {
            const unsigned int prev = atomicAdd(p.counters + bhf, 1u);
            const bool last = prev == (unsigned int)(p.NSPLIT * NC) - 1u;
            if (last) p.counters[bhf] = 0u;          // ready for the next call (stream order)
            *last_flag = last ? 1u : 0u;
        }
        __syncthreads();
        if (*last_flag) {
            __threadfence();
            const float4* src = reinterpret_cast<const float4*>(p.part + (long long)bhf * p.NSPLIT * D * 2 * D);
            constexpr int ROW4 = 2 * D / 4;             // float4 per summary row
            constexpr int TOT4 = D * ROW4;
            constexpr int UN = 4;                       // independent float4 columns per thread per pass ...
            constexpr int SG = 4;                       // ... times splits per group: UN * SG loads in flight per thread
            for (int e0 = tid; e0 < TOT4; e0 += UN * kSumThreads) {
                float4 acc[UN];
#pragma unroll
                for (int u = 0; u < UN; ++u) {
                    const int e = e0 + u * kSumThreads;
                    acc[u] = (e < TOT4) ? __ldcg(src + e) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
                for (int s0 = 1; s0 < p.NSPLIT; s0 += SG) {             // fixed split order; an absent split adds 0
                    float4 v[SG][UN];
#pragma unroll
                    for (int g = 0; g < SG; ++g)
#pragma unroll
                        for (int u = 0; u < UN; ++u) {
                            const int e = e0 + u * kSumThreads;
                            v[g][u] = (s0 + g < p.NSPLIT && e < TOT4) ? __ldcg(src + (long long)(s0 + g) * TOT4 + e) : make_float4(0.f, 0.f, 0.f, 0.f);
                        }
#pragma unroll
                    for (int g = 0; g < SG; ++g)
#pragma unroll
                        for (int u = 0; u < UN; ++u) { acc[u].x += v[g][u].x; acc[u].y += v[g][u].y; acc[u].z += v[g][u].z; acc[u].w += v[g][u].w; }
                }
#pragma unroll
                for (int u = 0; u < UN; ++u) {
                    const int e = e0 + u * kSumThreads;
                    if (e >= TOT4) continue;
                    const int mm = e / ROW4, c4 = e % ROW4;
                    if (c4 < D / 4) {
                        __nv_bfloat16* g = p.Gw + ((long long)bhf * D + mm) * D + c4 * 4;
                        uint2 uu;
                        uu.x = pack_bf16(a_f * acc[u].x, a_f * acc[u].y);
                        uu.y = pack_bf16(a_f * acc[u].z, a_f * acc[u].w);
                        *reinterpret_cast<uint2*>(g) = uu;
                    } else {
                        float* n = p.Nw + ((long long)bhf * D + mm) * D + (c4 - D / 4) * 4;
                        *reinterpret_cast<float4*>(n) = acc[u];
                    }
                }
            }
            if (tid == 0) p.gam[bhf] = a_f;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, NW);
}

// ---------------------------------------------------------------------------------------------------
// Phase A of BOTH passes of the normalised frame path in one launch (d = 128, no token split): CTA (b,h,f,j) streams
// 64-token tiles of K, V block j and K_raw once and keeps two accumulators,
//     [Gram | A](:, block j)       = (diag(beta) K)^T     [K block j     | V block j]       (matrix pass, Eq. 4-5)
//     [Gram_raw | b](:, block j)   = (diag(beta) K_raw)^T [K_raw block j | 1-column block]  (z pass, Eq. 20-21: b = K_raw^T beta)
// Launched one after the other, the two passes' Phase A grids (120 CTAs of 230 KB each at the paper's chunk) cannot be
// resident together and the second waits for SMs; here the second pass costs one more tile load and copy per tile.  The
// constant block is a 16-token slice addressed by every MMA of the tile through its own LBO (any distance is a legal LBO).
// ---------------------------------------------------------------------------------------------------
constexpr uint32_t kHBlk = 8192;       // one [64 tokens][64 features] bf16 block

template <int D>
struct DualSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t KT = NB * kHBlk;                        // [64 tokens][D] bf16
    static constexpr uint32_t STAGE = KT + kHBlk + KT;                // K | V block j | K_raw
    static constexpr int STAGES = 4;                                  // the ring is latency-bound: (load + copies + MMAs) / stages per tile
    static constexpr int SCB = 2;                                     // diag(beta) K copies
    static constexpr int SCR = 1;                                     // diag(beta) K_raw copies (one: what a fourth stage leaves room for)
    static constexpr uint32_t OFF_SCK = STAGES * STAGE;
    static constexpr uint32_t OFF_SCR = OFF_SCK + SCB * KT;
    static constexpr uint32_t OFF_ONE = OFF_SCR + SCR * KT;           // [16 tokens][64]: column 0 = 1 (block j = 0 only)
    static constexpr uint32_t OFF_BAR = OFF_ONE + 2048;
    static constexpr uint32_t TOTAL = OFF_BAR + 512 + 1024;
};

template <int D>
__global__ void __launch_bounds__(kSumThreads, 1)
gdn_frm_summaries_dual(const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV,
                       const __grid_constant__ CUtensorMap tmKr, const FrmParams p, const FrmParams pz) {
    static_assert(D == 128, "dual Phase A: d = 128 (two column CTAs per frame)");
    using L = DualSmem<D>;
    constexpr int NB = L::NB, NC = 2, STAGES = L::STAGES, SCB = L::SCB, SCR = L::SCR;
    constexpr int NW = 2 * D / NC;                // accumulator columns per pass: [Gram cols | A cols]
    constexpr int HW = D / NC;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* bar_full = bars;                    // [STAGES]
    uint64_t* bar_empty = bar_full + STAGES;      // [STAGES]
    uint64_t* bar_scK = bar_empty + STAGES;       // [SCB] diag(beta) K written (4 warps)
    uint64_t* bar_frK = bar_scK + SCB;            // [SCB] the MMAs that read it have completed
    uint64_t* bar_scR = bar_frK + SCB;            // [SCR] the same for K_raw
    uint64_t* bar_frR = bar_scR + SCR;
    uint64_t* bar_done = bar_frR + SCR;
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(bar_done + 1);

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int j = blockIdx.x % NC;
    const int bhf = blockIdx.x / NC;
    const int f = bhf % p.F, bh = bhf / p.F;
    const int b = bh / p.H, h = bh % p.H;
    const int ntiles = (p.G + 63) / 64;           // 64-token tiles of the frame

    if (tid == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(&bar_full[s], 1); mbar_init(&bar_empty[s], 1); }
        for (int s = 0; s < SCB; ++s) { mbar_init(&bar_scK[s], 4); mbar_init(&bar_frK[s], 1); }
        for (int s = 0; s < SCR; ++s) { mbar_init(&bar_scR[s], 4); mbar_init(&bar_frR[s], 1); }
        mbar_init(bar_done, 1);
        mbar_fence_init();
    }
    if (tid == 160) { tma_prefetch_desc(&tmK); tma_prefetch_desc(&tmV); tma_prefetch_desc(&tmKr); }
    if (warp == 0) tmem_alloc(tmem_slot, 2 * NW);
    if (tid < 16) {
        const uint32_t one = smem_u32(smem + L::OFF_ONE);
#pragma unroll
        for (int c = 0; c < 8; ++c) st_shared_v4(one + swz_chunk_off(tid, c, 0), (c == 0 && j == 0) ? 0x00003F80u : 0u, 0u, 0u, 0u);
        fence_proxy_async();
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_wait();                                    // (the front-end kernel of gdn_forward_chunk_full precedes)
    pdl_launch_dependents();

    if (warp == 5) {
        // ===== TMA producer =====
        if (elect_one()) {
            constexpr int kPF = 4;                 // L2 prefetch distance (64-token tiles) ahead of the ring
            const uint64_t pol = l2_policy_evict_first();
            auto prefetch = [&](int i) {
                const int n0 = i * 64;
                if (j == 0) {
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) { tma_prefetch_5d(&tmK, nb * 64, h, n0, f, b); tma_prefetch_5d(&tmKr, nb * 64, h, n0, f, b); }
                }
                tma_prefetch_5d(&tmV, j * 64, h, n0, f, b);
            };
            for (int i = STAGES; i < min(ntiles, STAGES + kPF); ++i) prefetch(i);
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES;
                if (i >= STAGES) mbar_wait(&bar_empty[st], (uint32_t)((i / STAGES) - 1) & 1u);
                if (i + kPF < ntiles && i >= STAGES) prefetch(i + kPF);
                uint8_t* base = smem + st * L::STAGE;
                mbar_expect_tx(&bar_full[st], L::STAGE);
                const int n0 = i * 64;
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(base + nb * kHBlk, &tmK, &bar_full[st], nb * 64, h, n0, f, b, pol);
                tma_load_5d_hint(base + L::KT, &tmV, &bar_full[st], j * 64, h, n0, f, b, pol);
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(base + L::KT + kHBlk + nb * kHBlk, &tmKr, &bar_full[st], nb * 64, h, n0, f, b, pol);
            }
        }
    }
    else if (warp == 4) {
        // ===== MMA issuer: four 16-token steps per pass and tile =====
        if (elect_one()) {
            const uint32_t id = umma_idesc(D, NW, true, true);
            const uint32_t one = smem_u32(smem + L::OFF_ONE);
            for (int i = 0; i < ntiles; ++i) {
                const int st = i % STAGES, sb = i % SCB, sr = i % SCR;
                mbar_wait(&bar_full[st], (uint32_t)(i / STAGES) & 1u);
                const uint32_t base = smem_u32(smem + st * L::STAGE);
                mbar_wait(&bar_scK[sb], (uint32_t)(i / SCB) & 1u);
                tc_fence_after();
                {   // matrix pass: B = [K block j | V block j]
                    const uint32_t a = smem_u32(smem + L::OFF_SCK + sb * L::KT), bq = base + (uint32_t)j * kHBlk;
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        umma_bf16(tmem, desc_mnmajor(a + s * 2048, kHBlk), desc_mnmajor(bq + s * 2048, (uint32_t)(NB - j) * kHBlk), id,
                                  (i > 0 || s > 0) ? 1u : 0u);
                    umma_commit(&bar_frK[sb]);
                }
                mbar_wait(&bar_scR[sr], (uint32_t)(i / SCR) & 1u);
                tc_fence_after();
                {   // z pass: B = [K_raw block j | the constant slice, the same 16 rows for every step]
                    const uint32_t a = smem_u32(smem + L::OFF_SCR + sr * L::KT), br = base + L::KT + kHBlk + (uint32_t)j * kHBlk;
#pragma unroll
                    for (int s = 0; s < 4; ++s)
                        umma_bf16(tmem + NW, desc_mnmajor(a + s * 2048, kHBlk), desc_mnmajor(br + s * 2048, one - (br + s * 2048)), id,
                                  (i > 0 || s > 0) ? 1u : 0u);
                    umma_commit(&bar_frR[sr]);
                }
                umma_commit(&bar_empty[st]);
            }
            umma_commit(bar_done);
        }
    } else {
        // ===== diag(beta) copies of K and K_raw: thread t -> token row t % 64 of feature block t / 64 =====
        const int r = tid & 63, blk = tid >> 6;
        const float* beta_f = p.beta + (long long)bh * p.T + (long long)f * p.G;
        auto load_beta = [&](int i) { const int n = i * 64 + r; return (i < ntiles && n < p.G) ? __ldg(beta_f + n) : 0.f; };
        auto scaled_copy = [&](uint32_t src, uint32_t dst, const Bf16Scale& bs) {
            uint4 x[8];
#pragma unroll
            for (int c = 0; c < 8; ++c) x[c] = ld_shared_v4(src + (uint32_t)(((c + r) & 7) << 4));
#pragma unroll
            for (int c = 0; c < 8; ++c)
                st_shared_v4(dst + (uint32_t)(((c + r) & 7) << 4), bf16x2_scale(x[c].x, bs), bf16x2_scale(x[c].y, bs),
                             bf16x2_scale(x[c].z, bs), bf16x2_scale(x[c].w, bs));
            fence_proxy_async();
            __syncwarp();
        };
        float b_next = load_beta(0);
        for (int i = 0; i < ntiles; ++i) {
            const int st = i % STAGES, sb = i % SCB, sr = i % SCR;
            const Bf16Scale bs = bf16_scale(b_next);
            b_next = load_beta(i + 1);
            const uint32_t stage = smem_u32(smem + st * L::STAGE), off = (uint32_t)blk * kHBlk + (uint32_t)r * 128u;
            if (i >= SCB) mbar_wait(&bar_frK[sb], (uint32_t)((i / SCB) - 1) & 1u);
            mbar_wait(&bar_full[st], (uint32_t)(i / STAGES) & 1u);
            scaled_copy(stage + off, smem_u32(smem + L::OFF_SCK + sb * L::KT) + off, bs);
            if (lane == 0) mbar_arrive(&bar_scK[sb]);
            if (i >= SCR) mbar_wait(&bar_frR[sr], (uint32_t)((i / SCR) - 1) & 1u);
            scaled_copy(stage + L::KT + kHBlk + off, smem_u32(smem + L::OFF_SCR + sr * L::KT) + off, bs);
            if (lane == 0) mbar_arrive(&bar_scR[sr]);
        }
    }

    // ---- epilogue (warps 0-3; thread = summary row m): G_f = alpha_f Gram (bf16), N_f = A (fp32) of both passes, staged in the
    //      idle ring and copied out in whole row segments (see gdn_frm_summaries) ----
    if (warp < 4) {
        const int m = tid;
        float a_f = p.alpha[bhf];
        if (p.log_alpha) a_f = expf(a_f);
        mbar_wait(bar_done, 0);
        tc_fence_after();
#pragma unroll 1
        for (int pass = 0; pass < 2; ++pass) {
            const FrmParams& q = pass ? pz : p;
            if (q.zero_sc) {                       // (see FrmParams::zero_sc)
                __nv_bfloat16* zb = q.zero_sc + (((long long)bh * q.NSc + f + 1) * D) * D + j * HW;
                for (int idx = tid; idx < D * (HW / 8); idx += 128) st_global_v4(zb + (long long)(idx / (HW / 8)) * D + (idx % (HW / 8)) * 8, 0u, 0u, 0u, 0u);
            }
            const uint32_t stgG = smem_u32(smem) + (uint32_t)pass * (D * 128 + D * 256), stgN = stgG + D * 128;
#pragma unroll 1
            for (int cc = 0; cc < NW / 32; ++cc) {
                float v[32];
                tmem_ld32(tmem_addr(tmem + pass * NW, warp * 32, cc * 32), v);
                if (cc < HW / 32) {
#pragma unroll
                    for (int q4 = 0; q4 < 4; ++q4)
                        st_shared_v4(stgG + m * 128 + (uint32_t)(((cc * 4 + q4) ^ (m & 7)) << 4), pack_bf16(a_f * v[8 * q4], a_f * v[8 * q4 + 1]),
                                     pack_bf16(a_f * v[8 * q4 + 2], a_f * v[8 * q4 + 3]), pack_bf16(a_f * v[8 * q4 + 4], a_f * v[8 * q4 + 5]),
                                     pack_bf16(a_f * v[8 * q4 + 6], a_f * v[8 * q4 + 7]));
                } else {
#pragma unroll
                    for (int q4 = 0; q4 < 8; ++q4)
                        st_shared_v4(stgN + m * 256 + (uint32_t)((((cc - HW / 32) * 8 + q4) ^ (m & 7)) << 4), __float_as_uint(v[4 * q4]),
                                     __float_as_uint(v[4 * q4 + 1]), __float_as_uint(v[4 * q4 + 2]), __float_as_uint(v[4 * q4 + 3]));
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            __nv_bfloat16* gbase = q.Gw + (long long)bhf * D * D + j * HW;
            float* nbase = q.Nw + (long long)bhf * D * D + j * HW;
#pragma unroll 4
            for (int idx = tid; idx < D * 8; idx += 128) {
                const int row = idx >> 3, c = idx & 7;
                const uint4 u = ld_shared_v4(stgG + row * 128 + (uint32_t)((c ^ (row & 7)) << 4));
                st_global_v4(gbase + (long long)row * D + c * 8, u.x, u.y, u.z, u.w);
            }
#pragma unroll 4
            for (int idx = tid; idx < D * 16; idx += 128) {
                const int row = idx >> 4, c = idx & 15;
                const uint4 u = ld_shared_v4(stgN + row * 256 + (uint32_t)((c ^ (row & 7)) << 4));
                st_global_v4(nbase + (long long)row * D + c * 4, u.x, u.y, u.z, u.w);
            }
            if (tid == 0 && j == 0) q.gam[bhf] = a_f;
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 2 * NW);
}

// ---------------------------------------------------------------------------------------------------
// Phase C.  grid = min(#SM, tiles), block = 192.   O = scale * Q_f S_f   (S_f = snapshot slot f + 1)
//   CTA c runs the contiguous tile range [c n / grid, (c+1) n / grid) of the (b,h,f,tile) order.
// ---------------------------------------------------------------------------------------------------
constexpr int kReadThreads = 192;      // warps 0-3: epilogue (thread = token row); warp 4: MMA issuer; warp 5: TMA producer

template <int D>
struct ReadSmem {
    static constexpr int NB = D / 64;
    static constexpr uint32_t Q_BYTES = NB * kBlk;                    // [128][D] bf16
    static constexpr uint32_t S_BYTES = (uint32_t)D * D * 2;          // NB blocks of [D][64] bf16
    static constexpr int QST = (D == 128) ? 3 : 4;
    static constexpr uint32_t OFF_S = QST * Q_BYTES;
    static constexpr uint32_t OFF_O = OFF_S + 2 * S_BYTES;            // 2 x out staging [128][D] bf16
    static constexpr uint32_t OFF_BAR = OFF_O + 2 * Q_BYTES;
    static constexpr uint32_t OFF_Z = OFF_BAR + 512;                  // fp32 z_f [D] (normalised readout)
    static constexpr uint32_t TOTAL = OFF_Z + 512 + 1024;
};

template <int D>
__global__ void __launch_bounds__(kReadThreads, 1)
gdn_frm_readout(const __grid_constant__ CUtensorMap tmQ, const __grid_constant__ CUtensorMap tmSc,
                const __grid_constant__ CUtensorMap tmO, const __grid_constant__ CUtensorMap tmGt,
                const __grid_constant__ CUtensorMap tmQr, const FrmParams p) {
    using L = ReadSmem<D>;
    constexpr int NB = L::NB, QST = L::QST;
    // normalised readout: the last ring slot holds the q_raw tile of the tile being finished, the Q ring is one slot shorter
    const bool norm = p.den_mode == 1;
    const int qst = norm ? QST - 1 : QST;
    uint8_t* sQr = nullptr;
    extern __shared__ uint8_t smem_raw[];
    uint8_t* smem = reinterpret_cast<uint8_t*>((reinterpret_cast<uintptr_t>(smem_raw) + 1023) & ~uintptr_t(1023));
    uint8_t* sS = smem + L::OFF_S;
    uint8_t* sO = smem + L::OFF_O;
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem + L::OFF_BAR);
    uint64_t* q_full = bars;                  // [QST]
    uint64_t* q_empty = q_full + QST;         // [QST] the MMAs that read the Q tile have completed
    uint64_t* s_full = q_empty + QST;         // [2]
    uint64_t* s_empty = s_full + 2;           // [2]   the last MMA that reads this state has completed
    uint64_t* acc_full = s_empty + 2;         // [2]
    uint64_t* acc_empty = acc_full + 2;       // [2]   drained by the 4 epilogue warps
    uint64_t* g_full = acc_empty + 2;         // [2]   output-gate tile landed in the staging buffer
    uint64_t* qr_full = g_full + 2;           // q_raw tile landed
    uint64_t* qr_empty = qr_full + 1;         // ... and has been read by the 4 epilogue warps
    uint32_t* tmem_slot = reinterpret_cast<uint32_t*>(qr_empty + 1);
    sQr = smem + (QST - 1) * L::Q_BYTES;

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long nt = p.total_tiles;
    const int t_lo = (int)(nt * blockIdx.x / gridDim.x), t_hi = (int)(nt * (blockIdx.x + 1) / gridDim.x);
    if (tid == 0) {
        for (int s = 0; s < QST; ++s) { mbar_init(&q_full[s], 1); mbar_init(&q_empty[s], 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(&s_full[s], 1); mbar_init(&s_empty[s], 1); mbar_init(&acc_full[s], 1); mbar_init(&acc_empty[s], 4); mbar_init(&g_full[s], 1); }
        mbar_init(qr_full, 1); mbar_init(qr_empty, 4);
        mbar_fence_init();
    }
    if (tid == 160) { tma_prefetch_desc(&tmQ); tma_prefetch_desc(&tmSc); tma_prefetch_desc(&tmO); }
    if (warp == 0) tmem_alloc(tmem_slot, 2 * D);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem = *tmem_slot;
    pdl_launch_dependents();                       // the next kernel in the stream (Phase A of the next call) may set itself up
    if (warp != 5) pdl_wait();                     // the chain's state snapshots are complete

    if (warp == 5) {
        // ===== TMA producer: Q tiles through the ring, S_f whenever the frame changes.  Q does not come from the previous
        //       kernel: the ring is filled before waiting for it =====
        if (elect_one()) {
            auto load_q = [&](int t, int i) {
                const int bhf = t / p.TPF, tile = t % p.TPF;
                const int f = bhf % p.F, bh = bhf / p.F;
                const int st = i % qst;
                mbar_expect_tx(&q_full[st], L::Q_BYTES);
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(smem + st * L::Q_BYTES + nb * kBlk, &tmQ, &q_full[st], nb * 64, bh % p.H, tile * 128, f, bh / p.H, l2_policy_evict_first());
            };
            auto load_qr = [&](int t) {
                const int bhf = t / p.TPF, tile = t % p.TPF;
                const int f = bhf % p.F, bh = bhf / p.F;
                mbar_expect_tx(qr_full, L::Q_BYTES);
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(sQr + nb * kBlk, &tmQr, qr_full, nb * 64, bh % p.H, tile * 128, f, bh / p.H, l2_policy_evict_first());
            };
            for (int i = 0; i < qst && t_lo + i < t_hi; ++i) load_q(t_lo + i, i);
            if (norm && t_lo < t_hi) load_qr(t_lo);
            pdl_wait();
            int cur = -1, ns = 0;
            for (int t = t_lo, i = 0; t < t_hi; ++t, ++i) {
                const int bhf = t / p.TPF;
                const int f = bhf % p.F, bh = bhf / p.F;
                if (bhf != cur) {
                    const int sb = ns & 1;
                    if (ns >= 2) mbar_wait(&s_empty[sb], (uint32_t)((ns >> 1) - 1) & 1u);
                    mbar_expect_tx(&s_full[sb], L::S_BYTES);
#pragma unroll
                    for (int nb = 0; nb < NB; ++nb) tma_load_3d(sS + sb * L::S_BYTES + nb * (D * 128), &tmSc, &s_full[sb], nb * 64, 0, bh * p.NSc + f + 1);
                    cur = bhf; ++ns;
                }
                if (i >= qst) {
                    mbar_wait(&q_empty[i % qst], (uint32_t)((i / qst) - 1) & 1u);
                    load_q(t, i);
                }
                if (norm && i >= 1) {
                    mbar_wait(qr_empty, (uint32_t)(i - 1) & 1u);             // the epilogue has formed den of the previous tile
                    load_qr(t);
                }
            }
        }
    } else if (warp == 4) {
        // ===== MMA issuer: acc[i & 1] = Q tile (A, K-major) * S_f (B, MN-major) =====
        if (elect_one()) {
            const uint32_t id = umma_idesc(128, D, false, true);
            int cur = -1, ns = 0;
            for (int t = t_lo, i = 0; t < t_hi; ++t, ++i) {
                const int bhf = t / p.TPF;
                if (bhf != cur) {
                    if (cur >= 0) umma_commit(&s_empty[(ns - 1) & 1]);       // every MMA on the previous state has been issued
                    mbar_wait(&s_full[ns & 1], (uint32_t)(ns >> 1) & 1u);
                    cur = bhf; ++ns;
                }
                const int st = i % qst, a = i & 1;
                mbar_wait(&q_full[st], (uint32_t)(i / qst) & 1u);
                if (i >= 2) mbar_wait(&acc_empty[a], (uint32_t)((i >> 1) - 1) & 1u);
                tc_fence_after();
                const uint32_t aQ = smem_u32(smem + st * L::Q_BYTES), aS = smem_u32(sS + ((ns - 1) & 1) * L::S_BYTES);
#pragma unroll
                for (int s = 0; s < D / 16; ++s)
                    umma_bf16(tmem + a * D, desc_kmajor(aQ + (s >> 2) * kBlk + (s & 3) * 32), desc_mnmajor(aS + s * 2048, D * 128), id, s > 0);
                umma_commit(&acc_full[a]);
                umma_commit(&q_empty[st]);
            }
        }
    } else {
        // ===== epilogue: TMEM -> registers -> scale (/ normaliser) -> bf16 -> swizzled staging -> TMA store =====
        const int row = tid;
        int z_cur = -1, z_nxt_bhf = -1;
        unsigned short z_nxt = 0;
        // Output gate (Eq. 23): the gate tile of a token tile has the layout of the output tile, so it is brought by TMA INTO
        // the staging buffer the output tile is about to be written to; each thread reads a 16-byte piece of the gate, scales
        // its accumulator piece and writes the result over it.  (One global load per piece and thread, issued when needed,
        // put a full memory latency on every tile: +6 us on the paper's chunk.)  The tile after the next is requested as soon
        // as the store that last used its buffer has read it.
        const bool gated = p.gate != nullptr;
        auto load_gate = [&](int t, int i) {
            const int bhf = t / p.TPF, tile = t % p.TPF;
            const int f = bhf % p.F, bh = bhf / p.F;
            mbar_expect_tx(&g_full[i & 1], L::Q_BYTES);
#pragma unroll
            for (int nb = 0; nb < NB; ++nb) tma_load_5d_hint(sO + (i & 1) * L::Q_BYTES + nb * kBlk, &tmGt, &g_full[i & 1], nb * 64, bh % p.H, tile * 128, f, bh / p.H, l2_policy_evict_first());
        };
        if (gated && tid == 0 && t_lo < t_hi) load_gate(t_lo, 0);
        for (int t = t_lo, i = 0; t < t_hi; ++t, ++i) {
            const int bhf = t / p.TPF, tile = t % p.TPF;
            const int f = bhf % p.F, bh = bhf / p.F;
            const int a = i & 1;
            const int n = tile * 128 + row;                      // token inside the frame
            float mul = p.scale;
            if (norm) {
                // Eq. 20-22: den = q_raw . z_f (fp32 accumulation; eps after the dot product, no clamp).  z_f: column 0 of the z
                // pass's snapshot, fetched when the frame changes; q_raw row: this thread's row of the staged tile.
                const uint32_t zb = smem_u32(smem + L::OFF_Z);
                auto z_of = [&](int bhf_) {                      // element `row` of z of frame-head bhf_ (bf16 bits)
                    const int f_ = bhf_ % p.F, bh_ = bhf_ / p.F;
                    return (row < D) ? __ldcg(reinterpret_cast<const unsigned short*>(p.z_sc) + (((long long)bh_ * p.NSc + f_ + 1) * D + row) * D) : (unsigned short)0;
                };
                if (bhf != z_cur) {                              // uniform over the 128 epilogue threads
                    if (z_nxt_bhf != bhf) z_nxt = z_of(bhf);     // (first tile of the CTA: nothing was requested ahead)
                    asm volatile("bar.sync 1, 128;" ::: "memory");
                    if (row < D) sts_f32(zb + row * 4, __uint_as_float((uint32_t)z_nxt << 16));
                    asm volatile("bar.sync 1, 128;" ::: "memory");
                    z_cur = bhf;
                }
                if (t + 1 < t_hi && (t + 1) / p.TPF != bhf) {    // the next tile is in another frame: its z is requested a tile ahead
                    z_nxt_bhf = (t + 1) / p.TPF;
                    z_nxt = z_of(z_nxt_bhf);
                }
                mbar_wait(qr_full, (uint32_t)i & 1u);
                const uint32_t qr = smem_u32(sQr);
                uint4 qv[D / 8];
#pragma unroll
                for (int c = 0; c < D / 8; ++c) qv[c] = ld_shared_v4(qr + swz_chunk_off(row, c, kBlk));
                float den = 0.f;
#pragma unroll
                for (int c = 0; c < D / 8; ++c) {
                    float x[8];
                    unpack8(qv[c], x);
                    const float4 z0 = lds_f4(zb + c * 32), z1 = lds_f4(zb + c * 32 + 16);
                    den = fmaf(x[0], z0.x, den); den = fmaf(x[1], z0.y, den); den = fmaf(x[2], z0.z, den); den = fmaf(x[3], z0.w, den);
                    den = fmaf(x[4], z1.x, den); den = fmaf(x[5], z1.y, den); den = fmaf(x[6], z1.z, den); den = fmaf(x[7], z1.w, den);
                }
                // The slot is released only now, behind the arithmetic that consumed the loaded registers: an arrive issued
                // right after the loads overtook them (measured: the next tile's q_raw landed in rows still being read).
                __syncwarp();
                if (lane == 0) mbar_arrive(qr_empty);
                if (n < p.G) mul = p.scale / (den + p.eps);
            }
            // the store that read staging buffer `a` two tiles ago must have finished reading it
            if (tid == 0) {
                if (gated) {
                    tma_store_wait_read();           // ... and the previous tile's store its own: that buffer takes the next gate tile
                    if (t + 1 < t_hi) load_gate(t + 1, i + 1);
                } else {
                    tma_store_wait_read_but1();
                }
            }
            mbar_wait(&acc_full[a], (uint32_t)(i >> 1) & 1u);
            tc_fence_after();
            if (p.drop_q && n < p.G) {                           // the MMAs have read the Q tile (and the dot product above the q_raw tile)
                const long long roff = ((((long long)(bh / p.H) * p.T + (long long)f * p.G + n) * p.H) + bh % p.H) * D;
#pragma unroll
                for (int l = 0; l < D * 2 / 128; ++l) {
                    asm volatile("discard.global.L2 [%0], 128;" ::"l"(p.drop_q + roff + l * 64) : "memory");
                    if (p.drop_qr) asm volatile("discard.global.L2 [%0], 128;" ::"l"(p.drop_qr + roff + l * 64) : "memory");
                }
            }
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (gated) mbar_wait(&g_full[a], (uint32_t)(i >> 1) & 1u);
            const uint32_t stg = smem_u32(sO + a * L::Q_BYTES);
#pragma unroll
            for (int cc = 0; cc < D / 32; ++cc) {
                float v[32];
                tmem_ld32(tmem_addr(tmem + a * D, warp * 32, cc * 32), v);
                if (cc == D / 32 - 1) {
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&acc_empty[a]);
                }
#pragma unroll
                for (int q4 = 0; q4 < 4; ++q4) {
                    float m[8];
#pragma unroll
                    for (int e = 0; e < 8; ++e) m[e] = mul;
                    if (gated) {
                        float gv[8];
                        unpack8(ld_shared_v4(stg + swz_chunk_off(row, cc * 4 + q4, kBlk)), gv);
#pragma unroll
                        for (int e = 0; e < 8; ++e) m[e] *= gv[e];
                    }
                    st_shared_v4(stg + swz_chunk_off(row, cc * 4 + q4, kBlk),
                                 pack_bf16(m[0] * v[8 * q4], m[1] * v[8 * q4 + 1]), pack_bf16(m[2] * v[8 * q4 + 2], m[3] * v[8 * q4 + 3]),
                                 pack_bf16(m[4] * v[8 * q4 + 4], m[5] * v[8 * q4 + 5]), pack_bf16(m[6] * v[8 * q4 + 6], m[7] * v[8 * q4 + 7]));
                }
            }
            fence_proxy_async();
            asm volatile("bar.sync 1, 128;" ::: "memory");
            if (tid == 0) {
#pragma unroll
                for (int nb = 0; nb < NB; ++nb) tma_store_5d_hint(&tmO, sO + a * L::Q_BYTES + nb * kBlk, nb * 64, bh % p.H, tile * 128, f, bh / p.H, l2_policy_evict_first());
                tma_store_commit();
            }
        }
        if (tid == 0) tma_store_wait_all();
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 0) tmem_dealloc(tmem, 2 * D);
}

}  // namespace frm
}  // namespace gdn
