// tc_tmap.cuh -- host side: build CUtensorMap descriptors (TMA) without linking libcuda: the driver's
// cuTensorMapEncodeTiled is fetched through cudaGetDriverEntryPoint at first use.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include <string>

namespace gdn {
namespace tc {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = reinterpret_cast<EncodeTiledFn>(p);
    }
    return fn;
}

// Generic tiled map. dims/strides innermost first; strides in BYTES for dims 1..rank-1 (stride of dim 0 is
// the element size). box in elements. OOB elements read as zero and are clipped on store.
inline bool make_tmap(CUtensorMap* out, const void* base, CUtensorMapDataType dt, int rank, const uint64_t* dims,
                      const uint64_t* strides_bytes, const uint32_t* box, CUtensorMapSwizzle swz, std::string* err) {
    EncodeTiledFn fn = encode_fn();
    if (!fn) { if (err) *err = "cuTensorMapEncodeTiled entry point not available"; return false; }
    cuuint64_t gdim[5], gstr[4];
    cuuint32_t bx[5], es[5];
    for (int i = 0; i < rank; ++i) { gdim[i] = dims[i]; bx[i] = box[i]; es[i] = 1; }
    for (int i = 0; i + 1 < rank; ++i) gstr[i] = strides_bytes[i + 1];
    CUresult r = fn(out, dt, (cuuint32_t)rank, const_cast<void*>(base), gdim, gstr, bx, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                    swz, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { if (err) *err = "cuTensorMapEncodeTiled failed with CUresult " + std::to_string((int)r); return false; }
    return true;
}

// [B, T = F*G, H, d] bf16 activation tensor viewed as 5-D (d, H, G, F, B); box = [rows tokens][64 features].
// Token tiles never straddle a group (frame) because the G dimension clips/zero-fills at G.
inline bool make_act_tmap(CUtensorMap* out, const void* base, int B, int T, int H, int d, int G, long long token_stride,
                          int box_rows, std::string* err) {
    const uint64_t dims[5] = {(uint64_t)d, (uint64_t)H, (uint64_t)G, (uint64_t)(T / G), (uint64_t)B};
    const uint64_t ts = (uint64_t)token_stride * 2;
    const uint64_t str[5] = {2, (uint64_t)d * 2, ts, ts * G, ts * T};
    const uint32_t box[5] = {64, 1, (uint32_t)box_rows, 1, 1};
    return make_tmap(out, base, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 5, dims, str, box, CU_TENSOR_MAP_SWIZZLE_128B, err);
}

}  // namespace tc
}  // namespace gdn
