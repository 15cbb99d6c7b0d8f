// kpz_k1.cuh — K1: persistent on-chip sweep, one CTA per sample (north_star (1),(3)).
//
// Layout on chip.  A thread owns one "unit" = 128 pairs = 256 sites = one Philox supergroup, held in
// registers for the whole run as 4 even-site words P[4] and 4 odd-site words Q[4] (de-interleaved, so that a
// pass whose offset equals the current "frame" is pure lane-local bitwise logic):
//   frame 0:  P[w] bit k = site 64(4u+w)+2k      Q[w] bit k = site 64(4u+w)+2k+1     pairs (P,Q)  = (2j, 2j+1)
//   frame 1:  P[w] bit k = site 64(4u+w)+2k+2    (P shifted by one even site)         pairs (Q,P)  = (2j+1, 2j+2)
// Changing frame is a 1-bit funnel shift through the unit plus ONE neighbour word (warp __shfl when the sample
// is one warp, a shared-memory halo slot + barrier when it spans several warps).  The ring closure (L-1,0) is the
// wrap-around of that neighbour index (PAPER.md:95 "close the ring"; :128 "pass first and last elements").
//
// Randomness.  U<T is evaluated MSB-first from bit-planes (one Philox call = one bit of 128 pairs' uniforms) and
// stops as soon as no pair of the unit is still undecided; offsets are drawn 32 passes at a time (one Philox call
// per lane, ballot).  Records: heights prefix + exact int64 sums, fused (K2).
#pragma once
#include "common.cuh"

namespace kpz {

// -------------------------------------------------------------------------------------------------------
// One sub-lattice pass on a unit held in the right frame: a = departure side of a forward hop, b = the other.
// (1,0) -> (0,1) iff U < T(p or p_slow at a);  (0,1) -> (1,0) iff U < T(q or q_slow at b)   (§R3).
// DIS: 0 no disorder, 1 slow-p tags only, 2 slow-p and slow-q tags.  NPS >= 0: exactly NPS planes, unrolled;
// NPS < 0: up to D.nplanes planes with early exit.
// -------------------------------------------------------------------------------------------------------
template <int DIS, int NPS>
__device__ __forceinline__ void pass_update(uint32_t (&a)[4], uint32_t (&b)[4], const uint32_t (&spa)[4],
                                            const uint32_t (&sqb)[4], const KpzDev& D, uint32_t G, uint32_t gs,
                                            uint32_t tlo, uint32_t c3) {
  uint32_t mp[4], mps[4], mq[4], mqs[4], lt[4], eq[4];
  const uint32_t AL0 = D.thr[0].always ? ~0u : 0u, AL1 = D.thr[1].always ? ~0u : 0u;
  const uint32_t AL2 = D.thr[2].always ? ~0u : 0u, AL3 = D.thr[3].always ? ~0u : 0u;
  const uint32_t PA0 = (!D.thr[0].always && D.thr[0].value) ? ~0u : 0u;
  const uint32_t PA1 = (!D.thr[1].always && D.thr[1].value) ? ~0u : 0u;
  const uint32_t PA2 = (!D.thr[2].always && D.thr[2].value) ? ~0u : 0u;
  const uint32_t PA3 = (!D.thr[3].always && D.thr[3].value) ? ~0u : 0u;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint32_t x = a[w] ^ b[w];
    mp[w] = x & a[w];
    mq[w] = x & b[w];
    mps[w] = 0;
    mqs[w] = 0;
    if (DIS >= 1) {
      mps[w] = mp[w] & spa[w];
      mp[w] &= ~spa[w];
    }
    if (DIS >= 2) {
      mqs[w] = mq[w] & sqb[w];
      mq[w] &= ~sqb[w];
    }
    lt[w] = (mp[w] & AL0) | (mq[w] & AL2);
    eq[w] = (mp[w] & PA0) | (mq[w] & PA2);
    if (DIS >= 1) {
      lt[w] |= mps[w] & AL1;
      eq[w] |= mps[w] & PA1;
    }
    if (DIS >= 2) {
      lt[w] |= mqs[w] & AL3;
      eq[w] |= mqs[w] & PA3;
    }
  }
  auto plane_step = [&](int pl) {
    const uint4 R4 = philox4x32_10(G, gs, tlo, c3 | ((uint32_t)pl << 22), D.keys);
    const uint32_t R[4] = {R4.x, R4.y, R4.z, R4.w};
    const uint32_t TB0 = 0u - ((D.thr[0].value >> (31 - pl)) & 1u);
    const uint32_t TB1 = 0u - ((D.thr[1].value >> (31 - pl)) & 1u);
    const uint32_t TB2 = 0u - ((D.thr[2].value >> (31 - pl)) & 1u);
    const uint32_t TB3 = 0u - ((D.thr[3].value >> (31 - pl)) & 1u);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      uint32_t tb = (mp[w] & TB0) | (mq[w] & TB2);
      if (DIS >= 1) tb |= mps[w] & TB1;
      if (DIS >= 2) tb |= mqs[w] & TB3;
      lt[w] |= eq[w] & tb & ~R[w];   // U bit 0, T bit 1 on a still-equal prefix: U < T decided
      eq[w] &= ~(R[w] ^ tb);         // prefix stays equal only where the bits agree
    }
  };
  if constexpr (NPS >= 0) {
#pragma unroll
    for (int pl = 0; pl < NPS; ++pl) plane_step(pl);
  } else {
    const int np = D.nplanes;
#pragma unroll 1
    for (int pl = 0; pl < np; ++pl) {
      if ((eq[0] | eq[1] | eq[2] | eq[3]) == 0) break;
      plane_step(pl);
    }
  }
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    a[w] ^= lt[w];
    b[w] ^= lt[w];
  }
}

// -------------------------------------------------------------------------------------------------------
// Neighbour exchange: value held by unit `src` of this sample.
// -------------------------------------------------------------------------------------------------------
template <bool SINGLE_WARP>
__device__ __forceinline__ uint32_t unit_exchange(uint32_t mine, int src, uint32_t* halo, int& parity) {
  if (SINGLE_WARP) {
    return __shfl_sync(0xFFFFFFFFu, mine, src);
  } else {
    uint32_t* slot = halo + parity * 1024;
    slot[threadIdx.x] = mine;
    __syncthreads();
    const uint32_t v = slot[src];
    parity ^= 1;
    return v;
  }
}

// frame 0 -> 1: P'[w] = P[w] >> 1 | next << 31, next = P[w+1] or h = the first word of the next unit.
template <bool PARTIAL>
__device__ __forceinline__ void shift_up(uint32_t (&P)[4], int nw, uint32_t h) {
  if (!PARTIAL) {
    P[0] = __funnelshift_r(P[0], P[1], 1);
    P[1] = __funnelshift_r(P[1], P[2], 1);
    P[2] = __funnelshift_r(P[2], P[3], 1);
    P[3] = __funnelshift_r(P[3], h, 1);
  } else {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t next = (w + 1 < nw) ? P[w + 1 < 4 ? w + 1 : 3] : h;
      P[w] = (w < nw) ? __funnelshift_r(P[w], next, 1) : 0u;
    }
  }
}
// frame 1 -> 0: P[w] = P'[w] << 1 | prev >> 31, prev = P'[w-1] or h = the last valid word of the previous unit.
template <bool PARTIAL>
__device__ __forceinline__ void shift_down(uint32_t (&P)[4], int nw, uint32_t h) {
  if (!PARTIAL) {
    P[3] = __funnelshift_l(P[2], P[3], 1);
    P[2] = __funnelshift_l(P[1], P[2], 1);
    P[1] = __funnelshift_l(P[0], P[1], 1);
    P[0] = __funnelshift_l(h, P[0], 1);
  } else {
#pragma unroll
    for (int w = 3; w >= 0; --w) {
      const uint32_t prev = (w > 0) ? P[w > 0 ? w - 1 : 0] : h;
      P[w] = (w < nw) ? __funnelshift_l(prev, P[w], 1) : 0u;
    }
  }
}
template <bool PARTIAL>
__device__ __forceinline__ uint32_t last_valid_word(const uint32_t (&P)[4], int nw) {
  if (!PARTIAL) return P[3];
  return nw >= 4 ? P[3] : nw == 3 ? P[2] : nw == 2 ? P[1] : P[0];
}

template <bool SINGLE_WARP, bool PARTIAL>
__device__ __forceinline__ void reframe_up(uint32_t (&P)[4], int nw, int nxt, uint32_t* halo, int& parity) {
  const uint32_t h = unit_exchange<SINGLE_WARP>(P[0], nxt, halo, parity);
  shift_up<PARTIAL>(P, nw, h);
}
template <bool SINGLE_WARP, bool PARTIAL>
__device__ __forceinline__ void reframe_down(uint32_t (&P)[4], int nw, int prv, uint32_t* halo, int& parity) {
  const uint32_t h = unit_exchange<SINGLE_WARP>(last_valid_word<PARTIAL>(P, nw), prv, halo, parity);
  shift_down<PARTIAL>(P, nw, h);
}

// -------------------------------------------------------------------------------------------------------
// K2 fused: heights h_x = inclusive prefix of (2n-1) and exact sums for one sample.
// A unit computes its sums relative to its first site in int32 (|r| <= 256, sum r^2 <= 2^24), then lifts them
// with its base height (exclusive scan over units) in int64.
// -------------------------------------------------------------------------------------------------------
// Heights of one unit relative to the site before it: r = total slope, s1 = sum of relative heights,
// s2 = sum of their squares (frame 0 words).
__device__ __forceinline__ void unit_relative_sums(const uint32_t (&P)[4], const uint32_t (&Q)[4], int nw, int& r_out,
                                                   int& s1_out, int& s2_out) {
  int r = 0, s1 = 0, s2 = 0;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    if (w < nw) {
      uint32_t e = P[w], o = Q[w];
#pragma unroll 8
      for (int k = 0; k < 32; ++k) {
        r += 2 * (int)(e & 1u) - 1;
        s1 += r;
        s2 += r * r;
        r += 2 * (int)(o & 1u) - 1;
        s1 += r;
        s2 += r * r;
        e >>= 1;
        o >>= 1;
      }
    }
  }
  r_out = r;
  s1_out = s1;
  s2_out = s2;
}

template <bool SINGLE_WARP>
__device__ __forceinline__ void record_sums(const uint32_t (&P)[4], const uint32_t (&Q)[4], int nw, int U,
                                            long long* scratch /* smem, >= 3*32 */, long long* out_h,
                                            long long* out_h2) {
  int r, s1, s2;
  unit_relative_sums(P, Q, nw, r, s1, s2);
  const int lane = threadIdx.x & 31;
  // inclusive scan of unit totals inside the warp
  int incl = r;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += v;
  }
  long long base = (long long)(incl - r);
  if (!SINGLE_WARP) {
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    int* wtot = reinterpret_cast<int*>(scratch + 64);
    __syncthreads();  // scratch reuse
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    int add = 0;
    for (int k = 0; k < warp; ++k) add += wtot[k];
    base += add;
    (void)nwarps;
  }
  const long long n = 64LL * nw;
  long long H = n * base + (long long)s1;
  long long H2 = n * base * base + 2LL * base * (long long)s1 + (long long)s2;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    H += __shfl_down_sync(0xFFFFFFFFu, H, d);
    H2 += __shfl_down_sync(0xFFFFFFFFu, H2, d);
  }
  if (SINGLE_WARP) {
    if (lane == 0) {
      *out_h = H;
      *out_h2 = H2;
    }
  } else {
    const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
    if (lane == 0) {
      scratch[warp] = H;
      scratch[32 + warp] = H2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      long long a = 0, b = 0;
      for (int k = 0; k < nwarps; ++k) {
        a += scratch[k];
        b += scratch[32 + k];
      }
      *out_h = a;
      *out_h2 = b;
    }
  }
  (void)U;
}

// -------------------------------------------------------------------------------------------------------
// The kernel.  grid = S samples, block = 32 * ceil(U/32) threads, thread u = unit u (idle when u >= U, but it
// still takes part in every barrier / shuffle).
// -------------------------------------------------------------------------------------------------------
template <bool SINGLE_WARP, bool PARTIAL, int DIS, int NPS>
__global__ void kpz_k1_kernel(const __grid_constant__ KpzDev D, const __grid_constant__ KpzRunArgs A) {
  __shared__ uint32_t halo[SINGLE_WARP ? 1 : 2048];
  __shared__ long long scratch[SINGLE_WARP ? 1 : 96];
  const int s = blockIdx.x;
  const int u = threadIdx.x;
  const int U = D.U;
  const bool active = u < U;
  const int nw = !active ? 0 : (PARTIAL ? min(4, D.PW - 4 * u) : 4);
  const int nxt = (u + 1 >= U) ? 0 : u + 1;
  const int prv = (u == 0) ? U - 1 : u - 1;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const size_t row = (size_t)s * D.PWp + 4 * (size_t)(active ? u : 0);
  int parity = 0;

  uint32_t P[4] = {0, 0, 0, 0}, Q[4] = {0, 0, 0, 0};
  uint32_t spa0[4] = {0, 0, 0, 0}, spa1[4] = {0, 0, 0, 0}, sqb0[4] = {0, 0, 0, 0}, sqb1[4] = {0, 0, 0, 0};
  if (active) {
    const uint4 e = *reinterpret_cast<const uint4*>(D.E + row);
    const uint4 o = *reinterpret_cast<const uint4*>(D.O + row);
    P[0] = e.x; P[1] = e.y; P[2] = e.z; P[3] = e.w;
    Q[0] = o.x; Q[1] = o.y; Q[2] = o.z; Q[3] = o.w;
    if (DIS >= 1) {
      const uint4 x = *reinterpret_cast<const uint4*>(D.SPE + row);
      const uint4 y = *reinterpret_cast<const uint4*>(D.SPO + row);
      spa0[0] = x.x; spa0[1] = x.y; spa0[2] = x.z; spa0[3] = x.w;   // frame 0: a = even site
      spa1[0] = y.x; spa1[1] = y.y; spa1[2] = y.z; spa1[3] = y.w;   // frame 1: a = odd site
    }
    if (DIS >= 2) {
      const uint4 x = *reinterpret_cast<const uint4*>(D.SQO + row);
      const uint4 y = *reinterpret_cast<const uint4*>(D.SQE + row);
      sqb0[0] = x.x; sqb0[1] = x.y; sqb0[2] = x.z; sqb0[3] = x.w;   // frame 0: b = odd site
      sqb1[0] = y.x; sqb1[1] = y.y; sqb1[2] = y.z; sqb1[3] = y.w;   // frame 1: b = next even site (shifted below)
    }
  }
  if (DIS >= 2) reframe_up<SINGLE_WARP, PARTIAL>(sqb1, nw, nxt, halo, parity);

  int frame = 0;
  int ri = A.rec_begin;
  long long next_rec = ri < A.nt ? A.rec_t[ri] : -1;
  uint32_t offbits = 0;
  const long long t_end = A.t0 + A.n_mcs;
  const int lane = threadIdx.x & 31;

  for (long long m = A.t0; m < t_end; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    if (D.offset_mode == 0 && (m == A.t0 || (m & 15) == 0)) {
      // offsets of the 32 passes of MCS (m & ~15) .. +15: lane l draws (mcs = base + l/2, pass = l & 1)
      const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
      const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), D.keys);
      offbits = __ballot_sync(0xFFFFFFFFu, w.x & 1u);
    }
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      const int o = D.offset_mode ? pass : (int)((offbits >> (2 * ((int)m & 15) + pass)) & 1u);
      if (o != frame) {
        if (o) reframe_up<SINGLE_WARP, PARTIAL>(P, nw, nxt, halo, parity);
        else reframe_down<SINGLE_WARP, PARTIAL>(P, nw, prv, halo, parity);
        frame = o;
      }
      const uint32_t c3 = ctr3(TAG_PAIR, (uint32_t)pass, 0, thi);
      if (o == 0) pass_update<DIS, NPS>(P, Q, spa0, sqb0, D, (uint32_t)u, gs, tlo, c3);
      else pass_update<DIS, NPS>(Q, P, spa1, sqb1, D, (uint32_t)u, gs, tlo, c3);
    }
    if (m + 1 == next_rec) {
      if (frame) {
        reframe_down<SINGLE_WARP, PARTIAL>(P, nw, prv, halo, parity);
        frame = 0;
      }
      record_sums<SINGLE_WARP>(P, Q, nw, U, scratch, A.rec_sum_h + (size_t)ri * D.S + s,
                               A.rec_sum_h2 + (size_t)ri * D.S + s);
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
  }
  if (frame) reframe_down<SINGLE_WARP, PARTIAL>(P, nw, prv, halo, parity);
  if (active) {
    *reinterpret_cast<uint4*>(D.E + row) = make_uint4(P[0], P[1], P[2], P[3]);
    *reinterpret_cast<uint4*>(D.O + row) = make_uint4(Q[0], Q[1], Q[2], Q[3]);
  }
}

}  // namespace kpz
