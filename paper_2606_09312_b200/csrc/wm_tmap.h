// Host helper shared by the TMA-fed kernels (wm_tcp.cu, wm_tc2.cu, wm_tcg.cu, wm_tsc.cu): a CUtensorMap over a row-major
// 2-D array of 16-bit values.  The driver entry point is looked up at run time (the library links no libcuda).
#pragma once

#include <cuda.h>

#include "wm_internal.h"

namespace wm {

// `cols` x `rows` elements of 16 bits, rows `row_bytes` apart; one box = box_cols x box_rows.  swizzle128: the box lands in
// shared memory in the 128-byte-swizzled K-major operand layout (box_cols = 64); otherwise as it is in memory (the pre-swizzled
// weight images).  Rows past `rows` read as zero.  Returns WM_OK or WM_ERR_CUDA (message set, prefixed with `who`).
inline int encode_tmap_2d(CUtensorMap* out, CUtensorMapDataType dtype, void* base, uint64_t cols, uint64_t rows,
                          uint64_t row_bytes, uint32_t box_cols, uint32_t box_rows, bool swizzle128, const char* who) {
    typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                      const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    void* fn = nullptr;
    cudaDriverEntryPointQueryResult qr;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr) != cudaSuccess || !fn ||
        qr != cudaDriverEntryPointSuccess) {
        set_error("%s: cuTensorMapEncodeTiled is not available from this driver", who);
        return WM_ERR_CUDA;
    }
    const cuuint64_t dims[2] = {cols, rows};
    const cuuint64_t strides[1] = {row_bytes};
    const cuuint32_t box[2] = {box_cols, box_rows}, es[2] = {1, 1};
    const CUresult r = ((EncodeTiledFn)fn)(out, dtype, 2, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                                           swizzle128 ? CU_TENSOR_MAP_SWIZZLE_128B : CU_TENSOR_MAP_SWIZZLE_NONE,
                                           CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) {
        set_error("%s: cuTensorMapEncodeTiled failed (%d)", who, (int)r);
        return WM_ERR_CUDA;
    }
    return WM_OK;
}

}  // namespace wm
