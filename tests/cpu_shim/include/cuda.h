// tests/cpu_shim/include/cuda.h -- TEST INFRASTRUCTURE, not product code.
// Stand-in for the CUDA driver header when the kernel sources are compiled for the host by tests/cpu_shim
// (see tests/cpu_shim/README.md): the tensor-map types the library passes to cuTensorMapEncodeTiled.
#pragma once
#include <stdint.h>

typedef uint64_t cuuint64_t;
typedef uint32_t cuuint32_t;
typedef int CUresult;
enum { CUDA_SUCCESS = 0, CUDA_ERROR_INVALID_VALUE = 1 };

typedef enum { CU_TENSOR_MAP_DATA_TYPE_INT32 = 4, CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7 } CUtensorMapDataType;
typedef enum { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 } CUtensorMapInterleave;
typedef enum { CU_TENSOR_MAP_SWIZZLE_NONE = 0 } CUtensorMapSwizzle;
typedef enum { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0, CU_TENSOR_MAP_L2_PROMOTION_L2_128B = 2 } CUtensorMapL2promotion;
typedef enum { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 } CUtensorMapFloatOOBfill;

// 128 opaque bytes, 64-byte aligned, like the real one; the shim keeps its own record inside
struct alignas(64) CUtensorMap { uint64_t opaque[16]; };
