// gdn_tc.cuh -- host side of the tcgen05 tensor-core paths: support matrix, workspace carving, tensor
// maps, launches.  Token-wise path: prepass -> chain -> output (gdn_tc_token.cuh).
#pragma once
#include <cuda_runtime.h>

#include <cstdio>
#include <string>

#include "../../include/gdn.h"
#include "gdn_profile.cuh"
#include "gdn_tc_token.cuh"
#include "tc_tmap.cuh"

namespace gdn {

struct TcPlan {
    bool ready = false;
    int sm_count = 0;
    int D = 0, C = 0, NT = 0, NC = 0, BH = 0;
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    // token path workspace
    __nv_bfloat16 *Gw = nullptr, *Qt = nullptr, *Ol = nullptr, *Sc = nullptr;
    float *Nw = nullptr, *gam = nullptr;
    CUtensorMap tmG, tmN, tmQt, tmSc, tmScS;   // static (workspace) maps; tmScS: [D][64] store box of the chain
    // per-call activation maps, cached on the pointers they were built for
    const void *cq = nullptr, *ck = nullptr, *cv = nullptr;
    CUtensorMap tmQ, tmK, tmV;
};

inline int tc_default_chunk(const gdn_config_t& c) { return c.chunk ? c.chunk : 128; }

// Does a tensor-core path exist for this config? Fills the resolved path / compute tile / launch count.
inline bool tc_supported(const gdn_config_t& c, gdn_path_t* path, int* chunk, int* launches) {
    if (c.io_dtype != GDN_BF16) return false;
    if (c.d_k != c.d_v || !(c.d_k == 64 || c.d_k == 128)) return false;
    if (c.group != 1) return false;                                   // frame-wise tensor-core path: not yet
    *path = GDN_PATH_TC_TOKEN;
    *chunk = tc_default_chunk(c);
    *launches = 3;
    return true;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

inline gdn_status_t tc_plan_init(TcPlan& tp, const gdn_config_t& c, int sm_count, std::string* err) {
    tp.sm_count = sm_count;
    tp.D = c.d_k;
    tp.C = tc_default_chunk(c);
    tp.BH = c.B * c.H;
    tp.NT = (c.T + 127) / 128;
    tp.NC = tp.C == 128 ? tp.NT : 2 * tp.NT;
    const size_t D = tp.D, BH = tp.BH, NT = tp.NT, NC = tp.NC;
    size_t off = 0;
    auto carve = [&](size_t bytes) { size_t o = off; off = align_up(off + bytes, 1024); return o; };
    const size_t oG = carve(BH * NC * D * D * 2), oN = carve(BH * NC * D * D * 4), oGam = carve(BH * NC * 4);
    const size_t oQt = carve(BH * NT * 128 * D * 2), oOl = carve(BH * NT * 128 * D * 2), oSc = carve(BH * NC * D * D * 2);
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
    {   // N_c: fp32 (D, D, BH*NC), box {32, D, 1}
        const uint64_t dims[3] = {D, D, BH * NC}, str[3] = {4, D * 4, D * D * 4};
        const uint32_t box[3] = {32, (uint32_t)D, 1};
        ok = ok && tc::make_tmap(&tp.tmN, tp.Nw, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 3, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    {   // Qt: bf16 (D, BH*NT*128), box {64, 128}
        const uint64_t dims[2] = {D, BH * NT * 128}, str[2] = {2, D * 2};
        const uint32_t box[2] = {64, 128};
        ok = ok && tc::make_tmap(&tp.tmQt, tp.Qt, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
    }
    if (!ok) { cudaFree(tp.workspace); tp.workspace = nullptr; return GDN_ERR_CUDA; }
    tp.ready = true;
    return GDN_OK;
}

inline void tc_plan_free(TcPlan& tp) {
    if (tp.workspace) cudaFree(tp.workspace);
    tp.workspace = nullptr;
    tp.ready = false;
}

template <typename Kern>
inline cudaError_t set_smem(Kern kern, size_t bytes) {
    return cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
}

template <int D, int C>
inline cudaError_t tc_launch_token(TcPlan& tp, const TokParams& p, cudaStream_t st, Profiler* prof) {
    using namespace tok;
    constexpr int NB = D / 64;
    const size_t smem1 = 3 * NB * kBlk + 6 * kBlk + 4096 + 1024;   // + 18 KB static (sL)
    const size_t smem2 = ChainSmem<D>::TOTAL;
    const size_t smem3 = NB * kBlk + (C == 128 ? 1 : 2) * D * D * 2 + 256 + 1024;
    static bool attr_done = false;
    if (!attr_done) {
        cudaError_t e = set_smem(gdn_tok_prepass<D, C>, smem1);
        if (e == cudaSuccess) e = set_smem(gdn_tok_chain<D>, smem2);
        if (e == cudaSuccess) e = set_smem(gdn_tok_output<D, C>, smem3);
        if (e != cudaSuccess) return e;
        attr_done = true;
    }
    if (prof) prof->begin(st);
    gdn_tok_prepass<D, C><<<tp.BH * tp.NT, kPrepassThreads, smem1, st>>>(tp.tmQ, tp.tmK, tp.tmV, p);
    if (prof) prof->mark(st, "gdn_tok_prepass");
    gdn_tok_chain<D><<<tp.BH * (D / 64), kChainThreads, smem2, st>>>(tp.tmG, tp.tmN, tp.tmScS, p);
    if (prof) prof->mark(st, "gdn_tok_chain");
    gdn_tok_output<D, C><<<tp.BH * tp.NT, 128, smem3, st>>>(tp.tmQt, tp.tmSc, p);
    if (prof) prof->mark(st, "gdn_tok_output");
    return cudaGetLastError();
}

inline gdn_status_t tc_forward(TcPlan& tp, const gdn_config_t& c, const void* q, const void* k, const void* v,
                               const float* alpha, const float* beta, const float* S_in, void* out, float* S_out,
                               cudaStream_t st, Profiler* prof, std::string* err) {
    if (!tp.ready) { if (err) *err = "tensor-core plan was not initialised (no sm_100 device at plan time)"; return GDN_ERR_ARCH; }
    auto ts = [&](long long s, int d) { return s ? s : (long long)c.H * d; };
    if (q != tp.cq || k != tp.ck || v != tp.cv) {
        bool ok = tc::make_act_tmap(&tp.tmQ, q, c.B, c.T, c.H, c.d_k, c.T, ts(c.q_token_stride, c.d_k), 128, err) &&
                  tc::make_act_tmap(&tp.tmK, k, c.B, c.T, c.H, c.d_k, c.T, ts(c.k_token_stride, c.d_k), 128, err) &&
                  tc::make_act_tmap(&tp.tmV, v, c.B, c.T, c.H, c.d_v, c.T, ts(c.v_token_stride, c.d_v), 128, err);
        if (!ok) { tp.cq = tp.ck = tp.cv = nullptr; return GDN_ERR_CUDA; }
        tp.cq = q; tp.ck = k; tp.cv = v;
    }
    TokParams p{};
    p.alpha = alpha; p.beta = beta; p.S_in = S_in; p.S_out = S_out; p.out = out;
    p.Gw = tp.Gw; p.Nw = tp.Nw; p.gam = tp.gam; p.Qt = tp.Qt; p.Ol = tp.Ol; p.Sc = tp.Sc;
    p.B = c.B; p.H = c.H; p.T = c.T; p.NT = tp.NT; p.NC = tp.NC;
    p.o_ts = ts(c.o_token_stride, c.d_v);
    p.scale = c.scale;
    p.log_alpha = (c.flags & GDN_FLAG_LOG_ALPHA) ? 1 : 0;
    p.dbg = nullptr;
#ifdef GDN_PHASE_TIMING
    static long long* dbg_dev = nullptr;
    if (!dbg_dev) { cudaMalloc(&dbg_dev, 64 * sizeof(long long)); cudaMemset(dbg_dev, 0, 64 * sizeof(long long)); }
    p.dbg = dbg_dev;
#endif
    cudaError_t e;
    if (tp.D == 64) e = (tp.C == 128) ? tc_launch_token<64, 128>(tp, p, st, prof) : tc_launch_token<64, 64>(tp, p, st, prof);
    else            e = (tp.C == 128) ? tc_launch_token<128, 128>(tp, p, st, prof) : tc_launch_token<128, 64>(tp, p, st, prof);
    if (e != cudaSuccess) { if (err) *err = std::string("token tensor-core launch: ") + cudaGetErrorString(e); return GDN_ERR_CUDA; }
#ifdef GDN_PHASE_TIMING
    {
        long long hst[64];
        cudaStreamSynchronize(st);
        cudaMemcpy(hst, p.dbg, sizeof(hst), cudaMemcpyDeviceToHost);
        fprintf(stderr, "[gdn phase cycles]");
        for (int i = 1; i < 16; ++i) fprintf(stderr, " %d:%lld", i, hst[i] - hst[i - 1]);
        fprintf(stderr, " [5->19:%lld 19->20:%lld 20->21:%lld 21->16:%lld 16->18:%lld 18->17:%lld 17->6:%lld]", hst[19] - hst[5], hst[20] - hst[19], hst[21] - hst[20], hst[16] - hst[21], hst[18] - hst[16], hst[17] - hst[18], hst[6] - hst[17]);
        fprintf(stderr, " total:%lld\n", hst[15] - hst[0]);
        fprintf(stderr, "[gdn chain step cycles] snapshot:%lld premath:%lld wait_mma:%lld ld+sub:%lld publish:%lld fence+sync:%lld total:%lld\n",
                hst[33] - hst[32], hst[34] - hst[33], hst[35] - hst[34], hst[36] - hst[35], hst[37] - hst[36], hst[38] - hst[37], hst[38] - hst[32]);
    }
#endif
    return GDN_OK;
}

}  // namespace gdn
