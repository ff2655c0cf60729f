// tensor_maps.h -- host side: CUtensorMap descriptors for the TMA tile loads of the persistent kernels.
// cuTensorMapEncodeTiled is a pure host function of the driver; it is fetched through the runtime
// (cudaGetDriverEntryPoint), so libtdh.so does not link against libcuda.  Descriptors are encoded per launch (the
// state blocks are caller-owned pointers) and passed to the kernels as __grid_constant__ parameters.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>

namespace tdh {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*,
                                  const cuuint64_t*, const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave,
                                  CUtensorMapSwizzle, CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

inline EncodeTiledFn encode_tiled_fn() {
    static EncodeTiledFn fn = []() -> EncodeTiledFn {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) != cudaSuccess) return nullptr;
        if (q != cudaDriverEntryPointSuccess) return nullptr;
        return reinterpret_cast<EncodeTiledFn>(p);
    }();
    return fn;
}

// Block [nplanes][NY][NZ] complex128 as seen by the tile kernels (tile_kernels.cuh): 128-byte lines of 8 values,
//   dim0 = 16 doubles of a line, dim1 = line inside a group of S rows (S*NZ/8), dim2 = row group (NY/S), dim3 = plane;
//   box {16, NZ/8, NY/S, ppc} at coordinates {0, r*NZ/8, 0, plane}, 128-byte swizzle.
inline bool encode_tile_map(CUtensorMap* m, const void* base, size_t nplanes, int ny, int nz, int s, int ppc) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {16, (cuuint64_t)(s * nz / 8), (cuuint64_t)(ny / s), (cuuint64_t)nplanes};
    const cuuint64_t strides[3] = {128, (cuuint64_t)s * nz * 16, (cuuint64_t)ny * nz * 16};
    const cuuint32_t box[4] = {16, (cuuint32_t)(nz / 8), (cuuint32_t)(ny / s), (cuuint32_t)ppc};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

// The same block as seen by the x-pencil kernel (xpencil_kernel.cuh): 256-byte chunks of 16 values,
//   dim0 = 32 doubles of a chunk, dim1 = chunk inside a row (NZ/16), dim2 = row (NY), dim3 = plane;
//   box {32, 1, 2, NX} at coordinates {0, chunk, 2*rho2, state*NX}, no swizzle.
inline bool encode_line_map(CUtensorMap* m, const void* base, size_t nplanes, int nx, int ny, int nz) {
    EncodeTiledFn fn = encode_tiled_fn();
    if (!fn) return false;
    const cuuint64_t dims[4] = {32, (cuuint64_t)(nz / 16), (cuuint64_t)ny, (cuuint64_t)nplanes};
    const cuuint64_t strides[3] = {256, (cuuint64_t)nz * 16, (cuuint64_t)ny * nz * 16};
    const cuuint32_t box[4] = {32, 1, 2, (cuuint32_t)nx};
    const cuuint32_t es[4] = {1, 1, 1, 1};
    return fn(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, const_cast<void*>(base), dims, strides, box, es,
              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE) == CUDA_SUCCESS;
}

}  // namespace tdh
