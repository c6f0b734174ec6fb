// cuda.h -- TEST INFRASTRUCTURE (tests/emu/README.md): the driver-API types synim_api.cu names, for the host emulation
#pragma once
#include <stdint.h>
typedef int CUresult;
enum { CUDA_SUCCESS = 0 };
typedef uint64_t cuuint64_t;
typedef uint32_t cuuint32_t;
struct alignas(64) CUtensorMap { uint64_t opaque[16]; };
struct EmuTensorMap { const float *base; uint64_t dims[3]; uint64_t strides[2]; uint32_t box[3]; };
static_assert(sizeof(EmuTensorMap) <= sizeof(CUtensorMap), "");
enum CUtensorMapDataType { CU_TENSOR_MAP_DATA_TYPE_FLOAT32 = 7 };
enum CUtensorMapInterleave { CU_TENSOR_MAP_INTERLEAVE_NONE = 0 };
enum CUtensorMapSwizzle { CU_TENSOR_MAP_SWIZZLE_NONE = 0 };
enum CUtensorMapL2promotion { CU_TENSOR_MAP_L2_PROMOTION_NONE = 0 };
enum CUtensorMapFloatOOBfill { CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE = 0 };
