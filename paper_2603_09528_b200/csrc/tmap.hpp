// tmap.hpp — host-side construction of TMA tensor maps (cuTensorMapEncodeTiled), resolved through the runtime's driver
// entry point so that libcuda is not linked directly.  Encoding is a pure host computation (no driver call reaches
// the device), cheap enough to run inside every launch wrapper — the field pointers belong to the caller and may
// change from solve to solve.
#pragma once

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>

namespace tpt {

using EncodeTiledFn = CUresult (*)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *, const cuuint64_t *,
                                   const cuuint64_t *, const cuuint32_t *, const cuuint32_t *, CUtensorMapInterleave,
                                   CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_tiled_fn() {
    // function-local static with an initialiser: thread-safe since C++11; the entry point is process-wide, not per device
    static const EncodeTiledFn fn = [] {
        void *ptr = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &ptr, cudaEnableDefault, &q) == cudaSuccess &&
            q == cudaDriverEntryPointSuccess)
            return reinterpret_cast<EncodeTiledFn>(ptr);
        return static_cast<EncodeTiledFn>(nullptr);
    }();
    return fn;
}

// FP64 tensor of rank 2 to 4.  dims[] in elements (dim 0 contiguous), strides_bytes[] for dims 1.. (multiples of 16),
// box[] in elements.  Returns false if the driver entry point is missing or the encoding is rejected.
inline bool make_f64_map(CUtensorMap *map, const void *base, int rank, const uint64_t *dims,
                         const uint64_t *strides_bytes, const uint32_t *box, CUtensorMapSwizzle swizzle) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn || rank < 2 || rank > 4) return false;
    cuuint64_t d[4], s[3];
    cuuint32_t b[4], e[4] = {1, 1, 1, 1};
    for (int q = 0; q < rank; ++q) { d[q] = dims[q]; b[q] = box[q]; }
    for (int q = 0; q + 1 < rank; ++q) s[q] = strides_bytes[q];
    return fn(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, const_cast<void *>(base), d, s, b, e,
              CU_TENSOR_MAP_INTERLEAVE_NONE, swizzle, CU_TENSOR_MAP_L2_PROMOTION_L2_128B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tpt
