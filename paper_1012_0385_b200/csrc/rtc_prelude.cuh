// rtc_prelude.cuh — fixed-width integer names for sources compiled at run time by NVRTC (which has no <cstdint>).
// Under nvcc the standard headers provide them.
#pragma once
#ifdef __CUDACC_RTC__
typedef unsigned int uint32_t;
typedef int int32_t;
typedef unsigned long long uint64_t;
typedef long long int64_t;
#else
#include <cstdint>
#include <cuda_runtime.h>
#endif
