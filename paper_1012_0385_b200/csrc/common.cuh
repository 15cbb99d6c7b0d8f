// common.cuh — shared host/device helpers of the CUDA path (error reporting, thresholds, bit layout helpers).
#pragma once
#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

#include "../../include/kpz_b200.h"
#include "sweep_types.cuh"

namespace kpz {

// ---- error reporting -------------------------------------------------------------------------------------
void set_error(const char* fmt, ...);
int fail(int code, const char* fmt, ...);
void count_launch(int n = 1);

#define KPZ_CUDA_CHECK(expr)                                                                       \
  do {                                                                                             \
    cudaError_t _e = (expr);                                                                       \
    if (_e != cudaSuccess) return kpz::fail(KPZ_ECUDA, "%s: %s", #expr, cudaGetErrorString(_e));   \
  } while (0)

#define KPZ_LAUNCH_CHECK(name)                                                                     \
  do {                                                                                             \
    cudaError_t _e = cudaGetLastError();                                                           \
    if (_e != cudaSuccess) return kpz::fail(KPZ_ECUDA, "launch %s: %s", name, cudaGetErrorString(_e)); \
    kpz::count_launch();                                                                           \
  } while (0)

// ---- thresholds -----------------------------------------------------------------------------
// T(x) = floor(x * 2^32) in [0, 2^32]; acceptance of a 32-bit uniform U is (uint64)U < T.
inline bool valid_prob(double x) { return x >= 0.0 && x <= 1.0; }
inline uint64_t threshold(double x) { return (uint64_t)std::floor(x * 4294967296.0); }

inline Thresh make_thresh(double x) {
  uint64_t T = threshold(x);
  Thresh t;
  t.always = (T >> 32) ? 1u : 0u;
  t.value = (uint32_t)T;
  return t;
}
// Number of leading bit-planes that can influence U < T: 0 for T in {0, 2^32}, else 32 - ctz(T).
inline int planes_needed(const Thresh& t) {
  if (t.always || t.value == 0) return 0;
  int z = 0;
  while (!((t.value >> z) & 1u)) ++z;
  return 32 - z;
}

inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

// ---- bit layout helpers ----------------------------------------------------------------------------------
// Natural layout: bit (i&31) of word (i>>5) = site i.  De-interleaved ("EO") layout of a 64-site group g:
// word E[g] bit k = site 64g+2k (even sites), word O[g] bit k = site 64g+2k+1 (odd sites).

// Gather the even-position bits of x into the low 16 bits.
__host__ __device__ __forceinline__ uint32_t compress_even(uint32_t x) {
  x &= 0x55555555u;
  x = (x | (x >> 1)) & 0x33333333u;
  x = (x | (x >> 2)) & 0x0F0F0F0Fu;
  x = (x | (x >> 4)) & 0x00FF00FFu;
  x = (x | (x >> 8)) & 0x0000FFFFu;
  return x;
}
// Scatter the low 16 bits of x to the even bit positions.
__host__ __device__ __forceinline__ uint32_t spread_even(uint32_t x) {
  x &= 0x0000FFFFu;
  x = (x | (x << 8)) & 0x00FF00FFu;
  x = (x | (x << 4)) & 0x0F0F0F0Fu;
  x = (x | (x << 2)) & 0x33333333u;
  x = (x | (x << 1)) & 0x55555555u;
  return x;
}
__host__ __device__ __forceinline__ void nat_to_eo(uint32_t w0, uint32_t w1, uint32_t& E, uint32_t& O) {
  E = compress_even(w0) | (compress_even(w1) << 16);
  O = compress_even(w0 >> 1) | (compress_even(w1 >> 1) << 16);
}
__host__ __device__ __forceinline__ void eo_to_nat(uint32_t E, uint32_t O, uint32_t& w0, uint32_t& w1) {
  w0 = spread_even(E) | (spread_even(O) << 1);
  w1 = spread_even(E >> 16) | (spread_even(O >> 16) << 1);
}

#ifdef __CUDACC__
// Bernoulli mask of one 128-element supergroup: bit k of word w = [ U(tag, time key, pass 0, 128 G + 32 w + k) < T ].
// MSB-first lazy comparison: plane b carries bit 31-b of the 128 uniforms.
__device__ __forceinline__ uint4 bernoulli128(const PhiloxKeys& K, uint32_t tag, uint32_t gsample, uint32_t time_lo,
                                              uint32_t time_hi, uint32_t G, Thresh T) {
  if (T.always) return make_uint4(~0u, ~0u, ~0u, ~0u);
  uint4 lt = make_uint4(0, 0, 0, 0);
  if (T.value == 0) return lt;
  uint4 eq = make_uint4(~0u, ~0u, ~0u, ~0u);
  const int last = 31 - (__ffs(T.value) - 1);  // last plane whose threshold bit is 1
  for (int b = 0; b <= last; ++b) {
    if ((eq.x | eq.y | eq.z | eq.w) == 0) break;
    const uint4 R = philox4x32_10(G, gsample, time_lo, ctr3(tag, 0, (uint32_t)b, time_hi), K);
    if ((T.value >> (31 - b)) & 1u) {
      lt.x |= eq.x & ~R.x; lt.y |= eq.y & ~R.y; lt.z |= eq.z & ~R.z; lt.w |= eq.w & ~R.w;
      eq.x &= R.x; eq.y &= R.y; eq.z &= R.z; eq.w &= R.w;
    } else {
      eq.x &= ~R.x; eq.y &= ~R.y; eq.z &= ~R.z; eq.w &= ~R.w;
    }
  }
  return lt;
}
#endif

}  // namespace kpz
