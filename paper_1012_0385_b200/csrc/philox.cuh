// philox.cuh — device/host Philox4x32-10 and the method's counter packing (§R4).
// Product code (CUDA path).  Shares nothing with oracle/.
#pragma once
#include "rtc_prelude.cuh"

namespace kpz {

constexpr uint32_t kPhiloxM0 = 0xD2511F53u;
constexpr uint32_t kPhiloxM1 = 0xCD9E8D57u;
constexpr uint32_t kPhiloxW0 = 0x9E3779B9u;
constexpr uint32_t kPhiloxW1 = 0xBB67AE85u;

// Stream tags (counter field c3[31:28]).
enum : uint32_t {
  TAG_PAIR = 0,
  TAG_OFFSET = 1,
  TAG_SLOW_P = 2,
  TAG_SLOW_Q = 3,
  TAG_INIT_A = 4,
  TAG_INIT_B = 5,
  TAG_PAIR_B = 6,
  TAG_TURN = 7,
  TAG_SWITCH_AB = 8,
  TAG_SWITCH_BA = 9,
  TAG_TURN_V = 11  // flags v_i of the B->A crossings when independent of u_i; 10 is oracle-only
};

// The ten round keys, precomputed on the host from the seed (the key schedule is a Weyl sequence, so the
// kernels never spend instructions on it; the values sit in the constant bank as kernel parameters).
struct PhiloxKeys {
  uint32_t k0[10];
  uint32_t k1[10];
};

#ifndef __CUDACC_RTC__
inline PhiloxKeys make_keys(uint64_t seed) {
  PhiloxKeys K;
  uint32_t a = (uint32_t)(seed & 0xFFFFFFFFull), b = (uint32_t)(seed >> 32);
  for (int r = 0; r < 10; ++r) {
    K.k0[r] = a;
    K.k1[r] = b;
    a += kPhiloxW0;
    b += kPhiloxW1;
  }
  return K;
}
#endif

// c3 = tag<<28 | pass<<27 | plane<<22 | time_hi(22 bits)
__host__ __device__ __forceinline__ uint32_t ctr3(uint32_t tag, uint32_t pass, uint32_t plane, uint32_t time_hi) {
  return (tag << 28) | (pass << 27) | (plane << 22) | time_hi;
}

// One Philox4x32-10 call.  Per round: 2 IMAD.WIDE (fma pipe) + 2 LOP3 (alu pipe).
__host__ __device__ __forceinline__ uint4 philox4x32_10(uint32_t c0, uint32_t c1, uint32_t c2, uint32_t c3,
                                                        const PhiloxKeys& K) {
#pragma unroll
  for (int r = 0; r < 10; ++r) {
    const unsigned long long p0 = (unsigned long long)kPhiloxM0 * c0;
    const unsigned long long p1 = (unsigned long long)kPhiloxM1 * c2;
    const uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ K.k0[r];
    const uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ K.k1[r];
    c1 = (uint32_t)p1;
    c3 = (uint32_t)p0;
    c0 = n0;
    c2 = n2;
  }
  return make_uint4(c0, c1, c2, c3);
}

}  // namespace kpz
