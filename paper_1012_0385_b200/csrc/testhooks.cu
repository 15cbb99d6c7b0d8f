// testhooks.cu — TEST-ONLY library (libkpz_b200_testhooks.so), not linked into the product.
// K0: dumps Philox4x32-10 words computed by the product's device function and by cuRAND's own
// curand_Philox4x32_10 device routine for the same counters, so that tests can pin the device generator
// against an implementation that is neither ours nor the oracle's (SURVEY §8(c) "Philox4x32-10" pin (ii)).
#include <cstdint>
#include <cuda_runtime.h>
#include <curand_philox4x32_x.h>

#include "philox.cuh"
#include "common.cuh"

#define HOOK_API extern "C" __attribute__((visibility("default")))

namespace {

__global__ void k0_philox_dump(const __grid_constant__ kpz::PhiloxKeys K, const uint32_t* ctr, int n, uint32_t* ours,
                               uint32_t* curand_out) {
  const int i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i >= n) return;
  const uint32_t c0 = ctr[4 * i], c1 = ctr[4 * i + 1], c2 = ctr[4 * i + 2], c3 = ctr[4 * i + 3];
  const uint4 a = kpz::philox4x32_10(c0, c1, c2, c3, K);
  ours[4 * i] = a.x; ours[4 * i + 1] = a.y; ours[4 * i + 2] = a.z; ours[4 * i + 3] = a.w;
  const uint4 b = curand_Philox4x32_10(make_uint4(c0, c1, c2, c3), make_uint2(K.k0[0], K.k1[0]));
  curand_out[4 * i] = b.x; curand_out[4 * i + 1] = b.y; curand_out[4 * i + 2] = b.z; curand_out[4 * i + 3] = b.w;
}

// Bernoulli mask of supergroups via the product's lazy comparator (device function bernoulli128).
__global__ void k0_bernoulli(const __grid_constant__ kpz::PhiloxKeys K, uint32_t tag, kpz::Thresh T, uint32_t sample,
                             long long timekey, int ngroups, uint32_t* out) {
  const int G = blockIdx.x * blockDim.x + threadIdx.x;
  if (G >= ngroups) return;
  const uint4 m = kpz::bernoulli128(K, tag, sample, (uint32_t)timekey, (uint32_t)((unsigned long long)timekey >> 32),
                                    (uint32_t)G, T);
  out[4 * G] = m.x; out[4 * G + 1] = m.y; out[4 * G + 2] = m.z; out[4 * G + 3] = m.w;
}

}  // namespace

// d_ctr: n*4 counter words (device); d_ours / d_curand: n*4 output words (device).  Returns 0 or a cudaError_t.
HOOK_API int kpz_test_philox_dump(uint64_t seed, const uint32_t* d_ctr, int n, uint32_t* d_ours, uint32_t* d_curand,
                                  void* stream) {
  const kpz::PhiloxKeys K = kpz::make_keys(seed);
  k0_philox_dump<<<(n + 127) / 128, 128, 0, (cudaStream_t)stream>>>(K, d_ctr, n, d_ours, d_curand);
  return (int)cudaGetLastError();
}

HOOK_API int kpz_test_bernoulli(uint64_t seed, uint32_t tag, double prob, uint32_t sample, long long timekey, int ngroups,
                                uint32_t* d_out, void* stream) {
  const kpz::PhiloxKeys K = kpz::make_keys(seed);
  k0_bernoulli<<<(ngroups + 127) / 128, 128, 0, (cudaStream_t)stream>>>(K, tag, kpz::make_thresh(prob), sample, timekey,
                                                                       ngroups, d_out);
  return (int)cudaGetLastError();
}
