// height_lut.cuh — heights of 8 sites at a time, shared by the fused K2 of the on-chip
// sweep (k1_sweep_jit.cuh) and the multi-CTA reduction of the streamed paths (kpz_k3.cuh).  No host headers: also
// compiled by NVRTC.
//
// A 256-entry table in shared memory, index = 4 even-site bits | 4 odd-site bits << 4 (site order e0,o0,e1,o1,...),
// entry = (r8+8) | (s1+36)<<5 | s2<<12 with r_k the height after k sites relative to the height before the byte,
// s1 = sum r_k, s2 = sum r_k^2.
#pragma once
#include "rtc_prelude.cuh"

namespace kpz {

__device__ __forceinline__ uint32_t height_lut_entry(int idx) {
  int r = 0, s1 = 0, s2 = 0;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    r += 2 * ((idx >> k) & 1) - 1;
    s1 += r;
    s2 += r * r;
    r += 2 * ((idx >> (4 + k)) & 1) - 1;
    s1 += r;
    s2 += r * r;
  }
  return (uint32_t)(r + 8) | ((uint32_t)(s1 + 36) << 5) | ((uint32_t)s2 << 12);
}

// Sums over the 64*nw sites of one unit (even-site words P, odd-site words Q, frame 0) of the heights relative to the
// site before the unit: r = total slope, s1 = sum, s2 = sum of squares (|r| <= 256, s2 <= 2^24: int32 is exact).
// (N = 4 words per thread, or 8 when a thread of the on-chip sweep holds two units: |r| <= 512, s2 <= 2^27.)
template <int N>
__device__ __forceinline__ void unit_relative_sums_lut(const uint32_t (&P)[N], const uint32_t (&Q)[N], int nw,
                                                       const uint32_t* lut, int& r_out, int& s1_out, int& s2_out) {
  int r = 0, s1 = 0, s2 = 0;
#pragma unroll
  for (int w = 0; w < N; ++w) {
    if (w < nw) {
#pragma unroll
      for (int k = 0; k < 8; ++k) {
        const uint32_t idx = ((P[w] >> (4 * k)) & 15u) | (((Q[w] >> (4 * k)) & 15u) << 4);
        const uint32_t v = lut[idx];
        const int d = (int)(v & 31u) - 8, a1 = (int)((v >> 5) & 127u) - 36, a2 = (int)(v >> 12);
        s1 += 8 * r + a1;
        s2 += 8 * r * r + 2 * r * a1 + a2;
        r += d;
      }
    }
  }
  r_out = r;
  s1_out = s1;
  s2_out = s2;
}

}  // namespace kpz
