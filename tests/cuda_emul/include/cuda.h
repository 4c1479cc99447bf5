// TEST INFRASTRUCTURE ONLY -- host-side stand-in for the driver API types the product uses (tensor maps).
// See cuda_runtime.h in this directory.
#pragma once
#include "cuda_runtime.h"

typedef int CUresult;
enum { CUDA_SUCCESS = 0, CUDA_ERROR_INVALID_VALUE = 1 };
typedef unsigned long long cuuint64_t;
typedef unsigned int cuuint32_t;
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0, CU_TENSOR_MAP_L2_PROMOTION_L2_128B = 2 };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };

// The emulated descriptor: what cuTensorMapEncodeTiled was told (rank <= 3, fp32).
struct __attribute__((aligned(64))) CUtensorMap_st {
    void *base;
    unsigned long long dim[3];
    unsigned long long stride_bytes[2];
    unsigned int box[3];
    unsigned int rank;
    unsigned long long pad[6];
};
typedef CUtensorMap_st CUtensorMap;
