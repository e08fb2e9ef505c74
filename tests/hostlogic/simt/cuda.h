// tests/hostlogic/simt/cuda.h -- TEST INFRASTRUCTURE: stands in for <cuda.h> in the SIMT-emulation
// build (see cuda_runtime.h in this directory).  Only the tensor-map types the launch code uses.
#pragma once
#include <stdint.h>
#include <string.h>
#include <cuda_runtime.h>

typedef uint64_t cuuint64_t;
typedef uint32_t cuuint32_t;
typedef int CUresult;
enum { CUDA_SUCCESS = 0, CUDA_ERROR_INVALID_VALUE = 1 };
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_L2_128B = 2 };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };

// 128 opaque bytes, 64-byte aligned, as the driver's; the emulation stores a SimTensorMap in it
struct alignas(64) CUtensorMap { uint64_t opaque[16]; };

namespace simt {
struct SimTensorMap {
    uint64_t magic;
    const void* base;
    uint32_t rank;
    uint32_t dims[3];       // elements
    uint64_t strides[2];    // bytes, dims 1..2
    uint32_t box[3];
};
static_assert(sizeof(SimTensorMap) <= sizeof(CUtensorMap), "SimTensorMap must fit the opaque map");
constexpr uint64_t TMAP_MAGIC = 0x544D4150454D554Cull;
}  // namespace simt

// cuTensorMapEncodeTiled as the launch code reaches it (through cudaGetDriverEntryPoint)
inline CUresult simt_cuTensorMapEncodeTiled(CUtensorMap* map, CUtensorMapDataType dt, cuuint32_t rank, void* base,
                                            const cuuint64_t* dims, const cuuint64_t* strides, const cuuint32_t* box,
                                            const cuuint32_t* estr, CUtensorMapInterleave, CUtensorMapSwizzle,
                                            CUtensorMapL2promotion, CUtensorMapFloatOOBfill) {
    if (dt != CU_TENSOR_MAP_DATA_TYPE_FLOAT32 || rank != 3) return CUDA_ERROR_INVALID_VALUE;
    if ((uintptr_t)base & 15) return CUDA_ERROR_INVALID_VALUE;
    simt::SimTensorMap m{};
    m.magic = simt::TMAP_MAGIC;
    m.base = base;
    m.rank = rank;
    for (int d = 0; d < 3; ++d) {
        if (dims[d] == 0 || dims[d] > (1ull << 32) || box[d] == 0 || box[d] > 256 || estr[d] != 1)
            return CUDA_ERROR_INVALID_VALUE;
        m.dims[d] = (uint32_t)dims[d];
        m.box[d] = box[d];
    }
    if ((box[0] * 4u) % 16u) return CUDA_ERROR_INVALID_VALUE;
    for (int d = 0; d < 2; ++d) {
        if (strides[d] % 16 || strides[d] >= (1ull << 40)) return CUDA_ERROR_INVALID_VALUE;
        m.strides[d] = strides[d];
    }
    memset(map, 0, sizeof(*map));
    memcpy(map, &m, sizeof(m));
    return CUDA_SUCCESS;
}
inline cudaError_t cudaGetDriverEntryPoint(const char* name, void** fn, int, cudaDriverEntryPointQueryResult* qr) {
    *fn = strcmp(name, "cuTensorMapEncodeTiled") == 0 ? (void*)&simt_cuTensorMapEncodeTiled : nullptr;
    *qr = cudaDriverEntryPointSuccess;
    return *fn ? cudaSuccess : 1;
}
