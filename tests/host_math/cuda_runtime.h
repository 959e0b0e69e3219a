// Host stand-in for <cuda_runtime.h>, used only by tests/test_device_math_on_host.py to compile
// paper_1204_6192_b200/csrc/hsg_math.cuh with g++ (-ffp-contract=off): the CUDA function qualifiers become nothing and the
// individually rounded intrinsics become the IEEE operations they are defined as.
#pragma once
#include <cmath>
#include <cstdint>
#include <cstring>

#define __device__
#define __host__
#define __forceinline__ inline

static inline uint32_t __umulhi(uint32_t a, uint32_t b) { return (uint32_t)(((uint64_t)a * (uint64_t)b) >> 32); }
static inline float __fmaf_rn(float a, float b, float c) { return std::fma(a, b, c); }
static inline float __fmul_rn(float a, float b) { return a * b; }
static inline float __fadd_rn(float a, float b) { return a + b; }
static inline float __fsub_rn(float a, float b) { return a - b; }
static inline float __uint_as_float(uint32_t w) { float f; std::memcpy(&f, &w, 4); return f; }
static inline uint32_t __float_as_uint(float f) { uint32_t w; std::memcpy(&w, &f, 4); return w; }

// kernel qualifiers and the handful of runtime types the kernel headers mention (tests/test_zmarch_on_host.py)
#define __global__
#define __launch_bounds__(...)
typedef int cudaError_t;
typedef void* cudaStream_t;
enum { cudaSuccess = 0, cudaErrorNotSupported = 801 };
