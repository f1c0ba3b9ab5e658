// gdn_tc.cuh -- host side of the tcgen05 tensor-core paths: support matrix, workspace carving, tensor
// maps, launches.  Token-wise path: prepass -> chain -> output (gdn_tc_token.cuh).
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <cstdlib>
#include <new>
#include <string>
#include <utility>
#include <vector>

#include "../../include/gdn.h"
#include "gdn_profile.cuh"
#include "gdn_tc_token.cuh"
#include "gdn_tc_frame.cuh"
#include "gdn_tc_fused.cuh"
#include "gdn_tc_tile64.cuh"
#include "gdn_tc_fused64.cuh"
#include "tc_tmap.cuh"

namespace gdn {

struct TcPlan {
    bool ready = false;
    unsigned attr_mask = 0;                    // which launchers have raised their kernels' dynamic shared-memory limit on this plan's device
    int sm_count = 0;
    int mode = 0;                              // GDN_PATH_TC_TOKEN or GDN_PATH_TC_FRAME
    int D = 0, C = 0, NT = 0, NC = 0, BH = 0;
    int G = 1, F = 0, TPF = 0, NSPLIT = 1, NSc = 0;   // frame-wise: frames, 128-token tiles per frame, token splits
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    // token path workspace
    __nv_bfloat16 *Gw = nullptr, *Qt = nullptr, *Ol = nullptr, *Sc = nullptr;
    float *Nw = nullptr, *gam = nullptr, *part = nullptr;
    CUtensorMap tmG, tmN, tmQt, tmOl, tmSc, tmScS;   // static (workspace) maps; tmScS: [D][64] store box of the chain
    CUtensorMap tmQt64, tmOl64;                      // the same rows with a 64-row box (light 64-token tile workers, d = 64)
    bool tile64 = false;                             // d = 64, C = 64: summaries by gdn_tok_tile64 (activation boxes of 64 tokens)
    // d = 64, C = 64, single persistent kernel with the two-level scan (gdn_tc_fused64.cuh)
    bool fused64 = false;
    F64Params f64{};                                 // workspace pointers / offsets; per-call fields filled at launch
    CUtensorMap tmM3, tmR2;
    // per-call activation maps, cached on the pointers they were built for
    const void *cq = nullptr, *ck = nullptr, *cv = nullptr, *co = nullptr;
    CUtensorMap tmQ, tmK, tmV, tmO;
    CUtensorMap tmGt;                                // output gate (Eq. 23), same tiling as tmO
    const void* cgate = nullptr;
    CUtensorMap tmK64, tmV64, tmKr64;                // 64-token boxes of k, v, k_raw: the dual Phase A of the normalised frame path
    const void *ck64 = nullptr, *cv64 = nullptr, *ckr64 = nullptr;
    // fused single-kernel token path (C = 128): per-tile ready flags and the call epoch
    bool fused = false;
    unsigned int* flags = nullptr;
    unsigned int epoch = 0;
    int HPR = 0, NWC = 0, grid = 0;
    // normaliser on the frame path: z as column 0 of the chain kernel's state, den = q_raw . z per token
    TcPlan* zplan = nullptr;                   // the z pass runs concurrently on its own workspace, stream and events
    cudaStream_t zs = nullptr;
    cudaEvent_t zev0 = nullptr, zev1 = nullptr;
    // bidirectional in-chunk scan: reverse-scan snapshots S<_f, bf16 [BH][F][D][D]
    bool bidir = false;
    const void *cqr = nullptr, *ckr = nullptr;
    CUtensorMap tmQr, tmKr;
};

struct NormArgs {                                  // the extra operands of gdn_forward_chunk_norm / gdn_forward_chunk_full
    const void *q_raw, *k_raw;
    const float* z_in;
    float* z_out;
    const void* gate = nullptr;                    // output gate G_f (Eq. 23) or NULL
    long long g_ts = 0;
    // gdn_forward_chunk_full: the four feature tensors are the plan's own dense buffers, whatever strides the plan's
    // config gives for the caller's q / k
    bool dense_qk = false;
};

inline int tc_default_chunk(const gdn_config_t& c) { return c.chunk ? c.chunk : 128; }

// Does a tensor-core path exist for this config? Fills the resolved path / compute tile / launch count.
inline bool tc_supported(const gdn_config_t& c, gdn_path_t* path, int* chunk, int* launches) {
    if (c.io_dtype != GDN_BF16) return false;
    // head dim 112 (the paper's, PAPER.md L316 / Alg. 1 l.1) is computed as 128: the tensor maps zero-fill features 112..127
    // on load and clip them on store, and zero features leave their rows / columns of every summary and state zero
    if (c.d_k != c.d_v || !(c.d_k == 64 || c.d_k == 112 || c.d_k == 128)) return false;
    if (c.d_k == 112 && c.group == 1 && (c.chunk == 64 || (c.flags & GDN_FLAG_UNFUSED))) return false;   // fused token kernel only
    if (c.group != 1) {                                               // frame-wise (the paper's variant)
        *path = GDN_PATH_TC_FRAME;
        *chunk = 0;
        *launches = 3;
        return true;
    }
    *path = GDN_PATH_TC_TOKEN;
    *chunk = tc_default_chunk(c);
    *launches = ((*chunk == 128 || c.d_k == 64) && !(c.flags & GDN_FLAG_UNFUSED)) ? 1 : 3;
    return true;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// token splits per frame for Phase A.  A split CTA streams `per` tiles and then pays for its partial (write, and
// a share of the last CTA's fixed-order reduction): about two tile times each.  Minimise waves x that.
inline int frame_splits(int units, int tpf, int sms) {
    int best = 1;
    double best_cost = 1e30;
    for (int ns = 1; ns <= tpf; ++ns) {
        const int per = (tpf + ns - 1) / ns;
        if ((ns - 1) * per >= tpf) continue;                   // would leave an empty split
        const long long ctas = (long long)units * ns;
        const double epi = ns > 1 ? 2.0 + 0.5 * ns : 1.0;
        const double cost = (double)((ctas + sms - 1) / sms) * (per + epi);
        if (cost < best_cost - 1e-9) { best_cost = cost; best = ns; }
    }
    return best;
}

inline gdn_status_t tc_plan_init_frame(TcPlan& tp, const gdn_config_t& c, int sm_count, std::string* err) {
    tp.mode = GDN_PATH_TC_FRAME;
    tp.sm_count = sm_count;
    tp.D = c.d_k == 112 ? 128 : c.d_k; tp.C = 0; tp.BH = c.B * c.H;
    tp.G = c.group; tp.F = c.T / c.group; tp.TPF = (c.group + 127) / 128;
    tp.NC = tp.F; tp.NSc = tp.F + 1; tp.NT = tp.F * tp.TPF;
    tp.NSPLIT = frame_splits(tp.BH * tp.F * (tp.D == 128 ? 2 : 1), tp.TPF, sm_count > 0 ? sm_count : 148);
    const size_t D = tp.D, BH = tp.BH, F = tp.F, NS = tp.NSPLIT;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 1024); return o; };
    const size_t oP = carve(NS > 1 ? BH * F * NS * D * 2 * D * 4 : 16), oG = carve(BH * F * D * D * 2), oN = carve(BH * F * D * D * 4);
    const size_t oGam = carve(BH * F * 4), oSc = carve(BH * (F + 1) * D * D * 2), oCnt = carve(BH * F * 4);
    const bool norm = (c.flags & GDN_FLAG_NORMALIZER) != 0;
    tp.bidir = (c.flags & GDN_FLAG_BIDIR) != 0;
    if (cudaMalloc(&tp.workspace, off) != cudaSuccess) {
        cudaGetLastError();
        if (err) *err = "workspace allocation of " + std::to_string(off) + " bytes failed";
        return GDN_ERR_NOMEM;
    }
    tp.workspace_bytes = off;
    uint8_t* w = static_cast<uint8_t*>(tp.workspace);
    tp.part = reinterpret_cast<float*>(w + oP);
    tp.Gw = reinterpret_cast<__nv_bfloat16*>(w + oG);
    tp.Nw = reinterpret_cast<float*>(w + oN);
    tp.gam = reinterpret_cast<float*>(w + oGam);
    tp.Sc = reinterpret_cast<__nv_bfloat16*>(w + oSc);
    tp.flags = reinterpret_cast<unsigned int*>(w + oCnt);          // per-frame split counters (self-resetting)
    if (cudaMemset(tp.flags, 0, BH * F * 4) != cudaSuccess) {
        cudaGetLastError(); cudaFree(tp.workspace); tp.workspace = nullptr;
        if (err) *err = "counter initialisation failed";
        return GDN_ERR_CUDA;
    }
    bool ok = true;
    {
        const uint64_t dims[3] = {D, D, BH * F}, str[3] = {2, D * 2, D * D * 2};
        const uint32_t box[3] = {64, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmG, tp.Gw, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        const uint64_t dimsS[3] = {D, D, BH * (F + 1)};
        ok = ok && tc::make_tmap(&tp.tmSc, tp.Sc, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dimsS, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        ok = ok && tc::make_tmap(&tp.tmScS, tp.Sc, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dimsS, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    {
        const uint64_t dims[3] = {D, D, BH * F}, str[3] = {4, D * 4, D * D * 4};
        const uint32_t box[3] = {32, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmN, tp.Nw, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    if (!ok) { cudaFree(tp.workspace); tp.workspace = nullptr; return GDN_ERR_CUDA; }
    if (norm) {
        tp.zplan = new (std::nothrow) TcPlan();
        gdn_config_t zc = c;
        zc.flags &= ~(uint32_t)GDN_FLAG_NORMALIZER;
        gdn_status_t zs = tp.zplan ? tc_plan_init_frame(*tp.zplan, zc, sm_count, err) : GDN_ERR_NOMEM;
        if (zs == GDN_OK && (cudaStreamCreateWithFlags(&tp.zs, cudaStreamNonBlocking) != cudaSuccess ||
                             cudaEventCreateWithFlags(&tp.zev0, cudaEventDisableTiming) != cudaSuccess ||
                             cudaEventCreateWithFlags(&tp.zev1, cudaEventDisableTiming) != cudaSuccess)) {
            cudaGetLastError();
            if (err) *err = "normaliser stream / event creation failed";
            zs = GDN_ERR_CUDA;
        }
        if (zs != GDN_OK) { cudaFree(tp.workspace); tp.workspace = nullptr; return zs; }
        tp.workspace_bytes += tp.zplan->workspace_bytes;
    }
    tp.ready = true;
    return GDN_OK;
}


// d = 64, C = 64 token path as one persistent kernel: workspace, flags, the two workspace tensor maps, role split.
inline gdn_status_t tc_plan_init_fused64(TcPlan& tp, const gdn_config_t& c, int sm_count, std::string* err) {
    const int sms = sm_count > 0 ? sm_count : 148;
    const int BH = tp.BH, NC = (c.T + 63) / 64;
    tp.NC = NC; tp.NSc = NC; tp.fused64 = true; tp.tile64 = true;
    // segments: chain CTAs (2 NS - 1 per stream) may take up to a quarter of the 4-per-SM CTA slots
    int NS = 1;
    while (NS < 4 && (NS + 1) * 2 <= NC && BH * (2 * (NS + 1) - 1) <= sms) ++NS;
    // segment 0 (scanned by the CTA that also runs level 2) is about three chunks longer than the others
    int L1 = NS > 1 ? (NC - 3 + NS - 1) / NS : NC;
    if (L1 < 1) L1 = 1;
    int L0 = NS > 1 ? NC - (NS - 1) * L1 : NC;
    if (L0 < L1) { L1 = (NC + NS - 1) / NS; L0 = L1; NS = (NC + L1 - 1) / L1; }
    F64Params& f = tp.f64;
    f.NS = NS; f.L0 = L0; f.L1 = L1; f.NCH = BH * (1 + 2 * (NS - 1));
    const size_t nchunk = (size_t)BH * NC, nseg = (size_t)BH * NS;
    f.zG = 0; f.zN = (int)nchunk; f.zSc = (int)(2 * nchunk); f.zGA = (int)(3 * nchunk);
    f.zGs = (int)(4 * nchunk); f.zBs = (int)(4 * nchunk + nseg); f.zSk = (int)(4 * nchunk + 2 * nseg);
    const size_t slots = 4 * nchunk + 3 * nseg, rows = 2 * nchunk * 64;
    f.rQt = 0; f.rOl = (long long)(nchunk * 64);
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 1024); return o; };
    const size_t nflag = 3 * nchunk + 3 * nseg;
    const size_t oM3 = carve(slots * 8192), oR2 = carve(rows * 128), oFl = carve(nflag * 8 + 64);
    if (cudaMalloc(&tp.workspace, off) != cudaSuccess) {
        cudaGetLastError();
        if (err) *err = "workspace allocation of " + std::to_string(off) + " bytes failed";
        return GDN_ERR_NOMEM;
    }
    tp.workspace_bytes = off;
    uint8_t* w = static_cast<uint8_t*>(tp.workspace);
    unsigned long long* fl = reinterpret_cast<unsigned long long*>(w + oFl);
    f.f_tile = fl; f.f_snap = fl + nchunk; f.f_snapA = fl + 2 * nchunk;
    f.f_segA = fl + 3 * nchunk; f.f_segB = f.f_segA + nseg; f.f_segS = f.f_segB + nseg;
    if (cudaMemset(fl, 0, nflag * 8 + 64) != cudaSuccess) {
        cudaGetLastError(); cudaFree(tp.workspace); tp.workspace = nullptr;
        if (err) *err = "flag initialisation failed";
        return GDN_ERR_CUDA;
    }
    f.n_tile_tasks = L0 * NS * BH; f.n_out_tasks = L0 * NS * BH;
    long long grid = (long long)f.NCH + f.n_tile_tasks;
    if (grid > 4LL * sms) grid = 4LL * sms;
    if (grid < f.NCH + 1) grid = f.NCH + 1;
    tp.grid = (int)grid;
    bool ok = true;
    {
        const uint64_t dims[3] = {64, 64, slots}, str[3] = {2, 128, 8192};
        const uint32_t box[3] = {64, 64, 1};
        ok = ok && tc::make_tmap(&tp.tmM3, w + oM3, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        const uint64_t dims2[2] = {64, rows}, str2[2] = {2, 128};
        const uint32_t box2[2] = {64, 64};
        ok = ok && tc::make_tmap(&tp.tmR2, w + oR2, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims2, str2, box2, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    if (!ok) { cudaFree(tp.workspace); tp.workspace = nullptr; return GDN_ERR_CUDA; }
    tp.ready = true;
    return GDN_OK;
}

inline gdn_status_t tc_plan_init(TcPlan& tp, const gdn_config_t& c, int sm_count, std::string* err) {
    if (c.group != 1) return tc_plan_init_frame(tp, c, sm_count, err);
    tp.mode = GDN_PATH_TC_TOKEN;
    tp.sm_count = sm_count;
    tp.D = c.d_k == 112 ? 128 : c.d_k;
    tp.C = tc_default_chunk(c);
    tp.BH = c.B * c.H;
    tp.NT = (c.T + 127) / 128;
    tp.NC = tp.C == 128 ? tp.NT : 2 * tp.NT;
    tp.NSc = tp.NC;
    if (tp.D == 64 && tp.C == 64 && c.d_k == 64 && !(c.flags & GDN_FLAG_UNFUSED)) return tc_plan_init_fused64(tp, c, sm_count, err);
    const size_t D = tp.D, BH = tp.BH, NT = tp.NT, NC = tp.NC;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 1024); return o; };
    const bool fused_plan = tc_default_chunk(c) == 128 && !(c.flags & GDN_FLAG_UNFUSED);
    const size_t oG = carve(BH * NC * D * D * 2), oN = carve(BH * NC * D * D * (fused_plan ? 2 : 4)), oGam = carve(BH * NC * 4);
    const size_t oQt = carve(BH * NT * 128 * D * 2), oOl = carve(BH * NT * 128 * D * 2);
    tp.fused = tp.C == 128 && !(c.flags & GDN_FLAG_UNFUSED);
    const size_t oSc = tp.fused ? 0 : carve(BH * NC * D * D * 2);
    const size_t oFl = tp.fused ? carve(BH * NT * 4) : 0;
    if (tp.fused) {
        // role split: chain workers own (head, 64-column tile) units; heads are processed in groups of HPR.
        // HPR minimises a two-term estimate: the prepass workers (all SMs but the chain workers) need
        // ceil(tiles / workers) tile times, the chain workers need groups * NT serial steps.
        const int sms = sm_count > 0 ? sm_count : 148, nct = tp.D / 64;
        const double t_tile = tp.D == 128 ? 14.0 : 10.0, t_step = tp.D == 128 ? 2.2 : 1.3;     // microseconds per prepass tile / chain step: constants of the split model, measured on B200 in round 1 (2026-11); only their ratio matters
        int hpr = 1;
        double best = 1e30;
        for (int h = 1; h <= tp.BH && h * nct < sms; ++h) {
            const int nwp = sms - h * nct, groups = (tp.BH + h - 1) / h;
            const double t_pre = (double)(((long long)BH * NT + nwp - 1) / nwp) * t_tile;
            const double t_chain = (double)groups * NT * t_step;
            const double est = (t_pre > t_chain ? t_pre : t_chain) + 0.02 * groups;
            if (est < best - 1e-9) { best = est; hpr = h; }
        }
        if (hpr < 1) hpr = 1;
        if (hpr > tp.BH) hpr = tp.BH;
        if (hpr * nct > sms - 1) hpr = (sms - 1) / nct > 0 ? (sms - 1) / nct : 1;
        tp.HPR = hpr;
        tp.NWC = hpr * nct;
        long long nwp = (long long)sms - tp.NWC;
        if (nwp > (long long)(BH * NT)) nwp = (long long)(BH * NT);
        if (nwp < 1) nwp = 1;
        tp.grid = tp.NWC + (int)nwp;
    }
    if (cudaMalloc(&tp.workspace, off) != cudaSuccess) {
        cudaGetLastError();
        if (err) *err = "workspace allocation of " + std::to_string(off) + " bytes failed";
        return GDN_ERR_NOMEM;
    }
    tp.workspace_bytes = off;
    uint8_t* w = static_cast<uint8_t*>(tp.workspace);
    tp.Gw = reinterpret_cast<__nv_bfloat16*>(w + oG);
    tp.Nw = reinterpret_cast<float*>(w + oN);
    tp.gam = reinterpret_cast<float*>(w + oGam);
    tp.Qt = reinterpret_cast<__nv_bfloat16*>(w + oQt);
    tp.Ol = reinterpret_cast<__nv_bfloat16*>(w + oOl);
    tp.Sc = reinterpret_cast<__nv_bfloat16*>(w + oSc);
    if (tp.fused) {
        tp.flags = reinterpret_cast<unsigned int*>(w + oFl);
        if (cudaMemset(tp.flags, 0, BH * NT * 4) != cudaSuccess) {
            cudaGetLastError(); cudaFree(tp.workspace); tp.workspace = nullptr;
            if (err) *err = "flag initialisation failed";
            return GDN_ERR_CUDA;
        }
    }
    bool ok = true;
    {   // G_c: bf16 (D, D, BH*NC), box {64, D, 1}
        const uint64_t dims[3] = {D, D, BH * NC}, str[3] = {2, D * 2, D * D * 2};
        const uint32_t box[3] = {64, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmG, tp.Gw, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        ok = ok && tc::make_tmap(&tp.tmSc, tp.Sc, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    {   // S_c snapshots written by the chain: one column tile [D rows][64 cols] per TMA store
        const uint64_t dims[3] = {D, D, BH * NC}, str[3] = {2, D * 2, D * D * 2};
        const uint32_t box[3] = {64, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmScS, tp.Sc, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    if (tp.fused) {   // N_c of the fused kernel: bf16 (D, D, BH*NC), box {64, D, 1} 
        const uint64_t dims[3] = {D, D, BH * NC}, str[3] = {2, D * 2, D * D * 2};
        const uint32_t box[3] = {64, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmN, tp.Nw, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    } else {          // N_c: fp32 (D, D, BH*NC), box {32, D, 1}
        const uint64_t dims[3] = {D, D, BH * NC}, str[3] = {4, D * 4, D * D * 4};
        const uint32_t box[3] = {32, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmN, tp.Nw, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    {   // Qt: bf16 (D, BH*NT*128), box {64, 128}
        const uint64_t dims[2] = {D, BH * NT * 128}, str[2] = {2, D * 2};
        const uint32_t box[2] = {64, 128};
        ok = ok && tc::make_tmap(&tp.tmQt, tp.Qt, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        ok = ok && tc::make_tmap(&tp.tmOl, tp.Ol, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
        const uint32_t box64[2] = {64, 64};
        ok = ok && tc::make_tmap(&tp.tmQt64, tp.Qt, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims, str, box64, CU_TENSOR_MAP_SWIZZLE_128B, err);
        ok = ok && tc::make_tmap(&tp.tmOl64, tp.Ol, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims, str, box64, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    tp.tile64 = tp.D == 64 && tp.C == 64;
    if (!ok) { cudaFree(tp.workspace); tp.workspace = nullptr; return GDN_ERR_CUDA; }
    tp.ready = true;
    return GDN_OK;
}

inline void tc_plan_free(TcPlan& tp) {
    if (tp.zplan) { tc_plan_free(*tp.zplan); delete tp.zplan; tp.zplan = nullptr; }
    if (tp.zs) cudaStreamDestroy(tp.zs);
    if (tp.zev0) cudaEventDestroy(tp.zev0);
    if (tp.zev1) cudaEventDestroy(tp.zev1);
    tp.zs = nullptr; tp.zev0 = tp.zev1 = nullptr;
    if (tp.workspace) cudaFree(tp.workspace);
    tp.workspace = nullptr;
    tp.ready = false;
}

// Launch `kern` as a programmatic dependent of the previous kernel in the stream (see tc::pdl_wait).
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid; cfg.blockDim = block; cfg.dynamicSmemBytes = smem; cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr; cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, std::forward<Args>(args)...);
}

template <typename Kern>
inline cudaError_t set_smem(Kern kern, size_t bytes) {
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <int D, int C>
inline cudaError_t tc_launch_token(TcPlan& tp, const TokParams& p, cudaStream_t st, Profiler* prof) {
    using namespace tok;
    constexpr int NB = D / 64;
    const size_t smem1 = prepass_smem_bytes<D>() + 1024;
    const size_t smem2 = ChainSmem<D>::TOTAL;
    const size_t smem3 = NB * kBlk + (C == 128 ? 1 : 2) * D * D * 2 + 256 + 1024;
    if (!(tp.attr_mask & 1u)) {
        cudaError_t e = set_smem(gdn_tok_prepass<D, C>, smem1);
        if (e == cudaSuccess) e = set_smem(gdn_tok_chain<D>, smem2);
        if (e == cudaSuccess) e = set_smem(gdn_tok_output<D, C>, smem3);
        if (e != cudaSuccess) return e;
        tp.attr_mask |= 1u;
    }
    if (prof) prof->begin(st);
    if (D == 64 && C == 64) {
        if (!(tp.attr_mask & 2u)) {
            cudaError_t e = set_smem(t64::gdn_tok_tile64, t64::SMEM_BYTES);
            if (e != cudaSuccess) return e;
            tp.attr_mask |= 2u;
        }
        t64::gdn_tok_tile64<<<tp.BH * tp.NC, t64::kThreads, t64::SMEM_BYTES, st>>>(tp.tmQ, tp.tmK, tp.tmV, tp.tmG, tp.tmN, tp.tmQt64, tp.tmOl64, p);
        if (prof) prof->mark(st, "gdn_tok_tile64");
    } else {
        gdn_tok_prepass<D, C><<<tp.BH * tp.NT, kPrepassThreads, smem1, st>>>(tp.tmQ, tp.tmK, tp.tmV, tp.tmG, tp.tmN, tp.tmQt, tp.tmOl, p);
        if (prof) prof->mark(st, "gdn_tok_prepass");
    }
    cudaError_t le = launch_pdl(gdn_tok_chain<D>, dim3(tp.BH * (D / 64)), dim3(kChainThreads), smem2, st, tp.tmG, tp.tmN, tp.tmScS, p);
    if (le != cudaSuccess) return le;
    if (prof) prof->mark(st, "gdn_tok_chain");
    le = launch_pdl(gdn_tok_output<D, C>, dim3(tp.BH * tp.NT), dim3(128), smem3, st, tp.tmQt, tp.tmSc, p);
    if (le != cudaSuccess) return le;
    if (prof) prof->mark(st, "gdn_tok_output");
    return cudaGetLastError();
}

template <int D>
inline cudaError_t tc_launch_fused(TcPlan& tp, const TokParams& p, cudaStream_t st, Profiler* prof) {
    const size_t smem = fused::fused_smem_bytes<D>();
    if (!(tp.attr_mask & 4u)) {
        cudaError_t e = set_smem(fused::gdn_tok_fused<D>, smem);
        if (e != cudaSuccess) return e;
        tp.attr_mask |= 4u;
    }
    FusedParams fp{};
    fp.t = p;
    fp.flags = tp.flags;
    fp.epoch = ++tp.epoch;
    fp.NWC = tp.NWC; fp.HPR = tp.HPR; fp.total_tiles = tp.BH * tp.NT;
    if (prof) prof->begin(st);
    cudaError_t le = launch_pdl(fused::gdn_tok_fused<D>, dim3(tp.grid), dim3(fused::kThreads), smem, st, tp.tmQ, tp.tmK, tp.tmV, tp.tmG, tp.tmN, tp.tmQt,
                                tp.tmO, fp);
    if (le != cudaSuccess) return le;
    if (prof) prof->mark(st, "gdn_tok_fused");
    return cudaGetLastError();
}


inline cudaError_t tc_launch_fused64(TcPlan& tp, const TokParams& p, cudaStream_t st, Profiler* prof) {
    if (!(tp.attr_mask & 8u)) {
        cudaError_t e = set_smem(f64::gdn_tok_fused64, t64::SMEM_BYTES);
        if (e != cudaSuccess) return e;
        tp.attr_mask |= 8u;
    }
    F64Params fp = tp.f64;
    fp.t = p;
    fp.epoch = ++tp.epoch;
    if (prof) prof->begin(st);
    f64::gdn_tok_fused64<<<tp.grid, t64::kThreads, t64::SMEM_BYTES, st>>>(tp.tmQ, tp.tmK, tp.tmV, tp.tmO, tp.tmM3, tp.tmR2, fp);
    if (prof) prof->mark(st, "gdn_tok_fused64");
    return cudaGetLastError();
}

template <int D>
inline cudaError_t tc_launch_frame(TcPlan& tp, const CUtensorMap& tmK, const CUtensorMap& tmV, const CUtensorMap& tmQ,
                                   const FrmParams& fp, const TokParams& cp, cudaStream_t st, Profiler* prof,
                                   cudaEvent_t before_readout = nullptr, bool readout = true, const CUtensorMap* tmQr = nullptr,
                                   bool phase_a = true, TcPlan* zt = nullptr, const TokParams* zc = nullptr) {
    using namespace frm;
    const size_t smem1 = SumSmem<D>::TOTAL;
    const size_t smem2 = tok::ChainSmem<D>::TOTAL;
    const size_t smem3 = ReadSmem<D>::TOTAL;
    if (!(tp.attr_mask & 16u)) {
        cudaError_t e = set_smem(gdn_frm_summaries<D>, smem1);
        if (e == cudaSuccess) e = set_smem(tok::gdn_tok_chain<D>, smem2);
        if (e == cudaSuccess) e = set_smem(tok::gdn_tok_chain_bidir<D>, smem2);
        if (e == cudaSuccess) e = set_smem(tok::gdn_tok_chain_multi<D>, smem2);
        if (e == cudaSuccess) e = set_smem(gdn_frm_readout<D>, smem3);
        if (e != cudaSuccess) return e;
        tp.attr_mask |= 16u;
    }
    const int sms = tp.sm_count > 0 ? tp.sm_count : 148;
    const int grid3 = fp.total_tiles < sms ? fp.total_tiles : sms;
    cudaError_t le;
    if (phase_a) {
        if (prof) prof->begin(st);
        // Launched as a programmatic dependent of whatever precedes it in the stream (the front-end kernel, the readout of the
        // previous call): the kernel waits for that grid before its first global access, only its prologue overlaps.
        le = launch_pdl(gdn_frm_summaries<D>, dim3(tp.BH * tp.F * tp.NSPLIT * sum_nc<D>()), dim3(kSumThreads), smem1, st, tmK, tmV, fp);
        if (le != cudaSuccess) return le;
    }
    if (prof && phase_a) prof->mark(st, "gdn_frm_summaries");
    const int nchain = tp.BH * (cp.col_tiles ? cp.col_tiles : D / 64);
    const bool both = tp.bidir && tp.F > 1;
    // Alg. 1 l.9-21: forward scan and, in the same launch, the reverse scan over the frames F-1 .. 1 from a zero state; both ADD
    // their snapshots into the forward snapshot slots (zeroed by Phase A): S^hist = S> + S< with no pass of its own
    auto scan_pair = [&](TcPlan& t, const TokParams& base, TokParams& fwd, TokParams& rev) {
        fwd = base;
        rev = base;
        rev.rev = 1; rev.NCa = t.F; rev.NC = t.F - 1; rev.NSc = t.F; rev.S_in = nullptr; rev.S_out = nullptr;
        rev.z_vec_in = nullptr; rev.z_vec_out = nullptr;            // z< starts from zero as well and is not carried
        fwd.snap_add = rev.snap_add = 1;                            // both add into the forward snapshots (zeroed by Phase A)
        rev.snap_off = 1; rev.snap_stride = t.NSc;
    };
    if (zt && zc) {
        // normalised path with the dual Phase A: the scans of both passes in one launch
        tok::ChainSets cs{};
        const int nz = tp.BH * (zc->col_tiles ? zc->col_tiles : D / 64);
        if (both) {
            scan_pair(tp, cp, cs.p[0], cs.p[1]);
            scan_pair(*zt, *zc, cs.p[2], cs.p[3]);
            cs.n[0] = cs.n[1] = nchain; cs.n[2] = cs.n[3] = nz;
        } else {
            cs.p[0] = cp; cs.p[2] = *zc;
            cs.n[0] = nchain; cs.n[1] = 0; cs.n[2] = nz; cs.n[3] = 0;
        }
        const int total = cs.n[0] + cs.n[1] + cs.n[2] + cs.n[3];
        le = launch_pdl(tok::gdn_tok_chain_multi<D>, dim3(total), dim3(tok::kChainThreads), smem2, st, tp.tmG, tp.tmN, tp.tmScS,
                        tp.tmScS, zt->tmG, zt->tmN, zt->tmScS, zt->tmScS, cs);
        if (le != cudaSuccess) return le;
        if (prof) prof->mark(st, "gdn_tok_chain_multi");
    } else if (both) {
        TokParams fwd, rp;
        scan_pair(tp, cp, fwd, rp);
        le = launch_pdl(tok::gdn_tok_chain_bidir<D>, dim3(2 * nchain), dim3(tok::kChainThreads), smem2, st, tp.tmG, tp.tmN, tp.tmScS, tp.tmScS, fwd, rp, nchain);
        if (le != cudaSuccess) return le;
        if (prof) prof->mark(st, "gdn_tok_chain_bidir");
    } else {
        le = launch_pdl(tok::gdn_tok_chain<D>, dim3(nchain), dim3(tok::kChainThreads), smem2, st, tp.tmG, tp.tmN, tp.tmScS, cp);
        if (le != cudaSuccess) return le;
        if (prof) prof->mark(st, "gdn_tok_chain");
    }
    if (!readout) return cudaGetLastError();       // the z pass ends with its scan: the matrix pass's readout takes z_f from its snapshots
    if (before_readout) { le = cudaStreamWaitEvent(st, before_readout, 0); if (le != cudaSuccess) return le; }   // the z pass's scan
    le = launch_pdl(gdn_frm_readout<D>, dim3(grid3), dim3(kReadThreads), smem3, st, tmQ, tp.tmSc, tp.tmO, fp.gate ? tp.tmGt : tp.tmO,
                    tmQr ? *tmQr : tmQ, fp);
    if (le != cudaSuccess) return le;
    if (prof) prof->mark(st, "gdn_frm_readout");
    return cudaGetLastError();
}

inline gdn_status_t tc_forward(TcPlan& tp, const gdn_config_t& c, const void* q, const void* k, const void* v,
                               const float* alpha, const float* beta, const float* S_in, void* out, float* S_out,
                               cudaStream_t st, Profiler* prof, std::string* err, const NormArgs* na = nullptr) {
    if (!tp.ready) { if (err) *err = "tensor-core plan was not initialised (no sm_100 device at plan time)"; return GDN_ERR_ARCH; }
    auto ts = [&](long long s, int d) { return s ? s : (long long)c.H * d; };
    if (q != tp.cq || k != tp.ck || v != tp.cv) {
        const int Gm = (tp.mode == GDN_PATH_TC_FRAME) ? c.group : c.T;      // token-wise: one "frame" of T tokens
        const int rows = tp.tile64 ? 64 : 128;
        const bool dense = na && na->dense_qk;         // the plan's own feature buffers (gdn_forward_chunk_full)
        bool ok = tc::make_act_tmap(&tp.tmQ, q, c.B, c.T, c.H, c.d_k, Gm, ts(dense ? 0 : c.q_token_stride, c.d_k), rows, err) &&
                  tc::make_act_tmap(&tp.tmK, k, c.B, c.T, c.H, c.d_k, Gm, ts(dense ? 0 : c.k_token_stride, c.d_k), rows, err) &&
                  tc::make_act_tmap(&tp.tmV, v, c.B, c.T, c.H, c.d_v, Gm, ts(c.v_token_stride, c.d_v), rows, err);
        if (!ok) { tp.cq = tp.ck = tp.cv = nullptr; return GDN_ERR_CUDA; }
        tp.cq = q; tp.ck = k; tp.cv = v;
    }
    if ((tp.fused || tp.fused64 || tp.mode == GDN_PATH_TC_FRAME) && out != tp.co) {
        const int Gm = (tp.mode == GDN_PATH_TC_FRAME) ? c.group : c.T;
        if (!tc::make_act_tmap(&tp.tmO, out, c.B, c.T, c.H, c.d_v, Gm, ts(c.o_token_stride, c.d_v), tp.fused64 ? 64 : 128, err)) { tp.co = nullptr; return GDN_ERR_CUDA; }
        tp.co = out;
    }
    if (tp.mode == GDN_PATH_TC_FRAME) {
        FrmParams fp{};
        fp.alpha = alpha; fp.beta = beta; fp.out = out; fp.part = tp.part; fp.counters = tp.flags; fp.Gw = tp.Gw; fp.Nw = tp.Nw; fp.gam = tp.gam;
        fp.total_tiles = tp.BH * tp.F * tp.TPF;
        fp.B = c.B; fp.H = c.H; fp.T = c.T; fp.G = tp.G; fp.F = tp.F; fp.NSPLIT = tp.NSPLIT; fp.TPF = tp.TPF; fp.NSc = tp.NSc;
        fp.o_ts = ts(c.o_token_stride, c.d_v);
        fp.scale = c.scale;
        fp.log_alpha = (c.flags & GDN_FLAG_LOG_ALPHA) ? 1 : 0;
        fp.zero_sc = (tp.bidir && tp.F > 1) ? tp.Sc : nullptr;
        TokParams cp{};
        cp.S_in = S_in; cp.S_out = S_out; cp.Gw = tp.Gw; cp.Nw = tp.Nw; cp.gam = tp.gam; cp.Sc = tp.Sc;
        cp.B = c.B; cp.H = c.H; cp.T = c.T; cp.NT = tp.NT; cp.NC = tp.NC; cp.NCa = tp.NC; cp.NSc = tp.NSc; cp.dr = c.d_k;
        cudaError_t e = cudaSuccess;
        cudaEvent_t den_ready = nullptr;
        bool dual = false;
        TokParams zscan{};
        if (na) {
            // z pass (Eq. 20-21 through the same Phase A and scan kernels): K_raw summaries with the constant block as V, the
            // scan on a [D][D] state whose column 0 is z (first 64-column tile only).  It shares nothing with the matrix pass
            // until the division in Phase C, so it runs beside it on its own stream and workspace; Phase C of the matrix pass
            // takes z_f from its snapshots and forms q_raw . z_f itself.
            TcPlan& zt = *tp.zplan;
            if (na->q_raw != tp.cqr || na->k_raw != tp.ckr) {
                bool ok = tc::make_act_tmap(&tp.tmQr, na->q_raw, c.B, c.T, c.H, c.d_k, c.group, ts(na->dense_qk ? 0 : c.q_token_stride, c.d_k), 128, err) &&
                          tc::make_act_tmap(&tp.tmKr, na->k_raw, c.B, c.T, c.H, c.d_k, c.group, ts(na->dense_qk ? 0 : c.k_token_stride, c.d_k), 128, err);
                if (!ok) { tp.cqr = tp.ckr = nullptr; return GDN_ERR_CUDA; }
                tp.cqr = na->q_raw; tp.ckr = na->k_raw;
            }
            FrmParams zf = fp;
            zf.part = zt.part; zf.counters = zt.flags; zf.Gw = zt.Gw; zf.Nw = zt.Nw; zf.gam = zt.gam;
            zf.zpass = 1; zf.scale = 1.f;
            zf.zero_sc = (tp.bidir && tp.F > 1) ? zt.Sc : nullptr;
            TokParams zc = cp;
            zc.Gw = zt.Gw; zc.Nw = zt.Nw; zc.gam = zt.gam; zc.Sc = zt.Sc;
            zc.S_in = nullptr; zc.S_out = nullptr;
            zc.zvec = 1; zc.z_vec_in = na->z_in; zc.z_vec_out = na->z_out;      // z <-> column 0 of the state, in the chain kernel
            zc.col_tiles = 1;                        // ... so only the first 64-column tile is run (the readout uses column 0 only)
            // d = 128 without a token split: Phase A of both passes in ONE launch (gdn_frm_summaries_dual), then the z scan
            // beside the matrix scan
            dual = tp.D == 128 && tp.NSPLIT == 1 && zt.NSPLIT == 1;
            if (dual) {
                if (k != tp.ck64 || v != tp.cv64 || na->k_raw != tp.ckr64) {
                    const bool dense = na->dense_qk;
                    bool ok = tc::make_act_tmap(&tp.tmK64, k, c.B, c.T, c.H, c.d_k, c.group, ts(dense ? 0 : c.k_token_stride, c.d_k), 64, err) &&
                              tc::make_act_tmap(&tp.tmV64, v, c.B, c.T, c.H, c.d_v, c.group, ts(c.v_token_stride, c.d_v), 64, err) &&
                              tc::make_act_tmap(&tp.tmKr64, na->k_raw, c.B, c.T, c.H, c.d_k, c.group, ts(dense ? 0 : c.k_token_stride, c.d_k), 64, err);
                    if (!ok) { tp.ck64 = tp.cv64 = tp.ckr64 = nullptr; return GDN_ERR_CUDA; }
                    tp.ck64 = k; tp.cv64 = v; tp.ckr64 = na->k_raw;
                }
                const size_t smemD = frm::DualSmem<128>::TOTAL;
                if (!(tp.attr_mask & 32u)) {
                    e = set_smem(frm::gdn_frm_summaries_dual<128>, smemD);
                    if (e != cudaSuccess) { if (err) *err = std::string("dual Phase A attribute: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
                    tp.attr_mask |= 32u;
                }
                if (prof) prof->begin(st);
                e = launch_pdl(frm::gdn_frm_summaries_dual<128>, dim3(tp.BH * tp.F * 2), dim3(frm::kSumThreads), smemD, st, tp.tmK64, tp.tmV64,
                               tp.tmKr64, fp, zf);
                if (e != cudaSuccess) { if (err) *err = std::string("dual Phase A launch: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
                if (prof) prof->mark(st, "gdn_frm_summaries_dual");
            }
            if (!dual) {
                e = cudaEventRecord(tp.zev0, st);     // after everything queued on the caller's stream so far
                if (e == cudaSuccess) e = cudaStreamWaitEvent(tp.zs, tp.zev0, 0);
                if (e != cudaSuccess) { if (err) *err = std::string("z pass fork: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
                e = (tp.D == 64) ? tc_launch_frame<64>(zt, tp.tmKr, tp.tmKr, tp.tmKr, zf, zc, tp.zs, nullptr, nullptr, false)
                                 : tc_launch_frame<128>(zt, tp.tmKr, tp.tmKr, tp.tmKr, zf, zc, tp.zs, nullptr, nullptr, false);
                if (e == cudaSuccess) e = cudaEventRecord(tp.zev1, tp.zs);
                if (e != cudaSuccess) { if (err) *err = std::string("normaliser pass: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
                den_ready = tp.zev1;
            } else {
                zscan = zc;                          // the z scan rides in the matrix pass's scan launch (tc_launch_frame below)
            }
            fp.den_mode = 1; fp.eps = c.eps; fp.z_sc = zt.Sc;
            if (na->dense_qk && c.d_k == 128) { fp.drop_q = static_cast<const __nv_bfloat16*>(q); fp.drop_qr = static_cast<const __nv_bfloat16*>(na->q_raw); }
            fp.gate = static_cast<const __nv_bfloat16*>(na->gate); fp.g_ts = na->g_ts ? na->g_ts : (long long)c.H * c.d_v; fp.dr = c.d_v;
            if (na->gate && na->gate != tp.cgate) {
                if (!tc::make_act_tmap(&tp.tmGt, na->gate, c.B, c.T, c.H, c.d_v, c.group, fp.g_ts, 128, err)) { tp.cgate = nullptr; return GDN_ERR_CUDA; }
                tp.cgate = na->gate;
            }
        }
        e = (tp.D == 64) ? tc_launch_frame<64>(tp, tp.tmK, tp.tmV, tp.tmQ, fp, cp, st, prof, den_ready, true, na ? &tp.tmQr : nullptr, !dual)
                         : tc_launch_frame<128>(tp, tp.tmK, tp.tmV, tp.tmQ, fp, cp, st, prof, den_ready, true, na ? &tp.tmQr : nullptr, !dual,
                                                dual ? tp.zplan : nullptr, dual ? &zscan : nullptr);
        if (e != cudaSuccess) { if (err) *err = std::string("frame tensor-core launch: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
        return GDN_OK;
    }
    TokParams p{};
    p.alpha = alpha; p.beta = beta; p.S_in = S_in; p.S_out = S_out; p.out = out;
    p.Gw = tp.Gw; p.Nw = tp.Nw; p.gam = tp.gam; p.Qt = tp.Qt; p.Ol = tp.Ol; p.Sc = tp.Sc;
    p.B = c.B; p.H = c.H; p.T = c.T; p.NT = tp.NT; p.NC = tp.NC; p.NCa = tp.NC; p.NSc = tp.NSc; p.dr = c.d_k;
    p.o_ts = ts(c.o_token_stride, c.d_v);
    p.scale = c.scale;
    p.log_alpha = (c.flags & GDN_FLAG_LOG_ALPHA) ? 1 : 0;
    cudaError_t e;
    if (tp.fused64) e = tc_launch_fused64(tp, p, st, prof);
    else if (tp.fused) e = (tp.D == 64) ? tc_launch_fused<64>(tp, p, st, prof) : tc_launch_fused<128>(tp, p, st, prof);
    else if (tp.D == 64) e = (tp.C == 128) ? tc_launch_token<64, 128>(tp, p, st, prof) : tc_launch_token<64, 64>(tp, p, st, prof);
    else            e = (tp.C == 128) ? tc_launch_token<128, 128>(tp, p, st, prof) : tc_launch_token<128, 64>(tp, p, st, prof);
    if (e != cudaSuccess) { if (err) *err = std::string("token tensor-core launch: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
    return GDN_OK;
}

}  // namespace gdn
