// gdn_tc.cuh -- host-side interface of the tcgen05 tensor-core paths (token-wise and frame-wise).
#pragma once
#include <cuda_runtime.h>

#include <string>

#include "../../include/gdn.h"
#include "gdn_profile.cuh"

namespace gdn {

struct TcPlan {
    void* workspace = nullptr;
    size_t workspace_bytes = 0;
    int sm_count = 0;
};

// Does a tensor-core path exist for this config? Fills the resolved path / compute tile / launch count.
inline bool tc_supported(const gdn_config_t& c, gdn_path_t* path, int* chunk, int* launches) {
    (void)c; (void)path; (void)chunk; (void)launches;
    return false;
}

inline gdn_status_t tc_plan_init(TcPlan& tp, const gdn_config_t& c, int sm_count, std::string* err) {
    (void)tp; (void)c; (void)sm_count; (void)err;
    return GDN_OK;
}

inline void tc_plan_free(TcPlan& tp) {
    if (tp.workspace) cudaFree(tp.workspace);
    tp.workspace = nullptr;
}

inline gdn_status_t tc_forward(TcPlan& tp, const gdn_config_t& c, const void* q, const void* k, const void* v,
                               const float* alpha, const float* beta, const float* S_in, void* out, float* S_out,
                               cudaStream_t st, Profiler* prof, std::string* err) {
    (void)prof;
    (void)tp; (void)c; (void)q; (void)k; (void)v; (void)alpha; (void)beta; (void)S_in; (void)out; (void)S_out; (void)st;
    if (err) *err = "tensor-core path not built";
    return GDN_ERR_UNSUPPORTED;
}

}  // namespace gdn
