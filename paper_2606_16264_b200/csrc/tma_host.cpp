// tma_host.cpp -- host-side TMA tensor-map encoding.  cuTensorMapEncodeTiled is a driver entry
// point; it is resolved at run time through the runtime so the library links without libcuda.
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

#include "tma_host.h"

namespace tropical {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn resolve_encode() {
    static EncodeTiledFn fn = nullptr;
    static bool tried = false;
    if (!tried) {
        tried = true;
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres) == cudaSuccess &&
            qres == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

// Pool viewed as a 2-D bf16 matrix [rows = num_pages*Hkv*16][cols = D]; box = 64 cols x 16 rows
// (one half of a (page, head) block at D = 128), SWIZZLE_128B.  Out-of-range rows read as zeros.  box_rows = 1: single
// slots (the page that holds both prior context and this step's rows in the fused step).
bool encode_pool_map(CUtensorMap* map, const void* base, long long rows, int D, int box_rows) {
    EncodeTiledFn enc = resolve_encode();
    if (!enc) return false;
    cuuint64_t dims[2] = {(cuuint64_t)D, (cuuint64_t)rows};
    cuuint64_t strides[1] = {(cuuint64_t)D * 2};
    cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    cuuint32_t estr[2] = {1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// q viewed as 3-D bf16 [T][Hq][D]; box = 64 cols x box_heads x box_tokens, SWIZZLE_128B:
// (1 head x 128 tokens) = a prefill Q tile half; the same view of k_new / v_new [T][Hkv][D] with 16- and 1-token
// boxes feeds this step's rows to the fused step.
bool encode_q_map(CUtensorMap* map, const void* base, int T, int Hq, int D, int box_heads, int box_tokens) {
    EncodeTiledFn enc = resolve_encode();
    if (!enc) return false;
    cuuint64_t dims[3] = {(cuuint64_t)D, (cuuint64_t)Hq, (cuuint64_t)T};
    cuuint64_t strides[2] = {(cuuint64_t)D * 2, (cuuint64_t)Hq * D * 2};
    cuuint32_t box[3] = {64, (cuuint32_t)box_heads, (cuuint32_t)box_tokens};
    cuuint32_t estr[3] = {1, 1, 1};
    return enc(map, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 3, const_cast<void*>(base), dims, strides, box, estr,
               CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
               CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tropical
