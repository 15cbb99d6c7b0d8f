// lanes_k4.cuh — K4: two-lane opposite-direction lattice gas with turning points (north_star (4);
// PAPER.md:253-275).  One CTA per sample, persistent over the whole run.
//
// Layout on chip: NATURAL bit order (bit i&31 of word i>>5 = site i), because the dominant random streams of
// this model are per SITE (lane changes, turning points): one Philox call is one bit-plane of 128 consecutive
// sites = 4 natural words, usable without any bit shuffling.  A thread owns one unit = 256 sites = 8 words of
// lane A, lane B and the turning-point mask, in registers.  In-lane hops are bitwise on the words: offset 0 pairs
// are (bit 2k, bit 2k+1) of a word; offset 1 pairs are (bit 2k+1, bit 2k+2), which needs bit 0 of the next word
// (next unit: warp __shfl / shared-memory halo) and sends one carry bit back — the ring closure (L-1,0) is the
// wrap-around of that exchange.  In-lane uniforms are per PAIR: their accept mask is built in
// pair order and spread to site order only when p < 1 (config 5 has p = 1: no in-lane Philox call at all).
#pragma once
#include "kpz_k1.cuh"

namespace kpz {

// Initial occupations / turning points in natural layout: thread = one supergroup of 128 sites.
__global__ void k_site_mask_nat(const __grid_constant__ PhiloxKeys K, uint32_t tag, Thresh T, long long timekey,
                                int first_sample, int S, int W, int Wp, uint32_t* M) {
  const int ng = (W + 3) / 4;
  const size_t n = (size_t)S * ng;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int s = (int)(i / ng), G = (int)(i % ng);
    const uint4 m = bernoulli128(K, tag, (uint32_t)(first_sample + s), (uint32_t)timekey,
                                 (uint32_t)((unsigned long long)timekey >> 32), (uint32_t)G, T);
    const uint32_t v[4] = {m.x, m.y, m.z, m.w};
    for (int k = 0; k < 4; ++k)
      if (4 * G + k < W) M[(size_t)s * Wp + 4 * G + k] = v[k];
  }
}

__global__ void k_copy_rows(const uint32_t* src, int S, int W, int src_stride, int dst_stride, uint32_t* dst) {
  const size_t n = (size_t)S * W;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t s = i / W, w = i % W;
    dst[s * dst_stride + w] = src[s * src_stride + w];
  }
}

// Lazy U < T over the live elements of one 128-element supergroup (pair stream or site stream).
__device__ __forceinline__ void lazy_less(uint32_t (&lt)[4], const uint32_t (&live)[4], const PhiloxKeys& K, uint32_t G,
                                          uint32_t gs, uint32_t tlo, uint32_t c3, Thresh T, int np) {
  if (T.always) {
#pragma unroll
    for (int w = 0; w < 4; ++w) lt[w] = live[w];
    return;
  }
  uint32_t eq[4];
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    lt[w] = 0;
    eq[w] = T.value ? live[w] : 0u;
  }
#pragma unroll 1
  for (int pl = 0; pl < np; ++pl) {
    if ((eq[0] | eq[1] | eq[2] | eq[3]) == 0) break;
    const uint4 R4 = philox4x32_10(G, gs, tlo, c3 | ((uint32_t)pl << 22), K);
    const uint32_t R[4] = {R4.x, R4.y, R4.z, R4.w};
    const uint32_t tb = 0u - ((T.value >> (31 - pl)) & 1u);
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      lt[w] |= eq[w] & tb & ~R[w];
      eq[w] &= ~(R[w] ^ tb);
    }
  }
}

// In-lane pass of one lane held in natural words.  RIGHT: (1,0)->(0,1) at pairs (a, a+1); else (0,1)->(1,0).
// next0 = word 0 of the next unit (old value).  Returns the carry bit for the next unit's bit 0 (offset 1 only).
template <bool PARTIAL, bool RIGHT>
__device__ __forceinline__ uint32_t lane_pass(uint32_t (&X)[8], int nwn, int o, uint32_t next0, const PhiloxKeys& K,
                                              uint32_t tag, uint32_t G, uint32_t gs, uint32_t tlo, uint32_t c3time,
                                              Thresh T, int np, unsigned long long& hops) {
  uint32_t hop[8];
  const uint32_t amask = o ? 0xAAAAAAAAu : 0x55555555u;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    uint32_t sh;
    if (o == 0) {
      sh = X[w] >> 1;
    } else {
      uint32_t nx = (w < 7) ? X[w < 7 ? w + 1 : 7] : next0;
      if (PARTIAL) nx = (w + 1 < nwn) ? nx : next0;
      sh = __funnelshift_r(X[w], nx, 1);
    }
    hop[w] = (RIGHT ? (X[w] & ~sh) : (~X[w] & sh)) & amask;
    if (PARTIAL) hop[w] = (w < nwn) ? hop[w] : 0u;
  }
  if (!T.always) {
    // candidates in pair order (bit j of word k = pair 32k+j of this unit), lazy compare, spread back
    uint32_t live[4], acc[4];
#pragma unroll
    for (int k = 0; k < 4; ++k)
      live[k] = compress_even(hop[2 * k] >> o) | (compress_even(hop[2 * k + 1] >> o) << 16);
    lazy_less(acc, live, K, G, gs, tlo, ctr3(tag, 0, 0, 0) | c3time, T, np);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      hop[2 * k] = spread_even(acc[k]) << o;
      hop[2 * k + 1] = spread_even(acc[k] >> 16) << o;
    }
  }
  uint32_t carry = 0, out = 0;
  unsigned cnt = 0;
#pragma unroll
  for (int w = 0; w < 8; ++w) {
    X[w] ^= hop[w] | (hop[w] << 1) | carry;
    carry = o ? (hop[w] >> 31) : 0u;
    cnt += __popc(hop[w]);
    if (PARTIAL && w + 1 == nwn) {  // the carry of the last valid word leaves the unit
      out = carry;
      carry = 0;
    }
  }
  if (!PARTIAL) out = carry;
  hops += cnt;
  return out;
}

template <bool SINGLE_WARP, bool PARTIAL>
__global__ void __launch_bounds__(1024) lanes_k4_kernel(const __grid_constant__ LanesDev D, const __grid_constant__ LanesRunArgs R) {
  __shared__ uint32_t halo[SINGLE_WARP ? 1 : 2048];
  __shared__ unsigned long long red[SINGLE_WARP ? 1 : 4 * 32];
  const int s = blockIdx.x;
  const int u = threadIdx.x;
  const int U = D.U;
  const bool active = u < U;
  const int nwn = !active ? 0 : (PARTIAL ? min(8, D.W - 8 * u) : 8);
  const int nxt = (u + 1 >= U) ? 0 : u + 1;
  const int prv = (u == 0) ? U - 1 : u - 1;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const size_t row = (size_t)s * D.Wp + 8 * (size_t)(active ? u : 0);
  const int lane = threadIdx.x & 31;
  int parity = 0;

  uint32_t A[8], B[8], T[8];
#pragma unroll
  for (int w = 0; w < 8; ++w) A[w] = B[w] = T[w] = 0;
  if (active) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      const uint4 a = *reinterpret_cast<const uint4*>(D.A + row + 4 * h);
      const uint4 b = *reinterpret_cast<const uint4*>(D.B + row + 4 * h);
      const uint4 t = *reinterpret_cast<const uint4*>(D.T + row + 4 * h);
      A[4 * h] = a.x; A[4 * h + 1] = a.y; A[4 * h + 2] = a.z; A[4 * h + 3] = a.w;
      B[4 * h] = b.x; B[4 * h + 1] = b.y; B[4 * h + 2] = b.z; B[4 * h + 3] = b.w;
      T[4 * h] = t.x; T[4 * h + 1] = t.y; T[4 * h + 2] = t.z; T[4 * h + 3] = t.w;
    }
  }
  unsigned long long jA = 0, jB = 0;
  int ri = R.rec_begin;
  long long next_rec = ri < R.nt ? R.rec_t[ri] : -1;
  uint32_t offbits = 0;
  const long long t_end = R.t0 + R.n_mcs;
  const int np_w = D.np_w;

  auto block_sum4 = [&](unsigned long long v0, unsigned long long v1, unsigned long long v2, unsigned long long v3,
                        unsigned long long (&out)[4]) {
    unsigned long long v[4] = {v0, v1, v2, v3};
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) v[k] += __shfl_down_sync(0xFFFFFFFFu, v[k], d);
    if (SINGLE_WARP) {
#pragma unroll
      for (int k = 0; k < 4; ++k) out[k] = v[k];  // valid in lane 0
    } else {
      const int warp = threadIdx.x >> 5, nwarps = blockDim.x >> 5;
      __syncthreads();
      if (lane == 0)
#pragma unroll
        for (int k = 0; k < 4; ++k) red[k * 32 + warp] = v[k];
      __syncthreads();
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        unsigned long long a = 0;
        for (int w = 0; w < nwarps; ++w) a += red[k * 32 + w];
        out[k] = a;
      }
    }
  };

  for (long long m = R.t0; m < t_end; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    if (D.offset_mode == 0 && (m == R.t0 || (m & 15) == 0)) {
      const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
      const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), D.keys);
      offbits = __ballot_sync(0xFFFFFFFFu, w.x & 1u);
    }
    // turning points redrawn at the start of every epoch (epoch 0 was drawn at create)
    if (D.period > 0 && m > 0 && (m % D.period) == 0) {
      const unsigned long long ep = (unsigned long long)(m / D.period);
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint4 t = bernoulli128(D.keys, TAG_TURN, gs, (uint32_t)ep, (uint32_t)(ep >> 32), (uint32_t)(2 * u + h), D.t_turn);
        T[4 * h] = t.x; T[4 * h + 1] = t.y; T[4 * h + 2] = t.z; T[4 * h + 3] = t.w;
      }
      if (PARTIAL || !active) {
#pragma unroll
        for (int w = 0; w < 8; ++w) T[w] = (w < nwn) ? T[w] : 0u;
      }
    }
#pragma unroll 1
    for (int pass = 0; pass < 2; ++pass) {
      const int o = D.offset_mode ? pass : (int)((offbits >> (2 * ((int)m & 15) + pass)) & 1u);
      // ---- in-lane hops of both lanes with the same offset ----
      uint32_t nA = 0, nB = 0;
      if (o) {
        nA = unit_exchange<SINGLE_WARP>(A[0], nxt, halo, parity);
        nB = unit_exchange<SINGLE_WARP>(B[0], nxt, halo, parity);
        if (!active) nA = nB = 0;  // idle threads hold all-zero words and must not see a neighbour bit
      }
      const uint32_t c3t = ((uint32_t)pass << 27) | thi;
      uint32_t cA, cB;
      if (o == 0) {
        cA = lane_pass<PARTIAL, true>(A, nwn, 0, nA, D.keys, TAG_PAIR, (uint32_t)u, gs, tlo, c3t, D.t_pa, D.np_a, jA);
        cB = lane_pass<PARTIAL, false>(B, nwn, 0, nB, D.keys, TAG_PAIR_B, (uint32_t)u, gs, tlo, c3t, D.t_pb, D.np_b, jB);
      } else {
        cA = lane_pass<PARTIAL, true>(A, nwn, 1, nA, D.keys, TAG_PAIR, (uint32_t)u, gs, tlo, c3t, D.t_pa, D.np_a, jA);
        cB = lane_pass<PARTIAL, false>(B, nwn, 1, nB, D.keys, TAG_PAIR_B, (uint32_t)u, gs, tlo, c3t, D.t_pb, D.np_b, jB);
        const uint32_t inA = unit_exchange<SINGLE_WARP>(cA, prv, halo, parity);
        const uint32_t inB = unit_exchange<SINGLE_WARP>(cB, prv, halo, parity);
        if (active) {
          A[0] ^= inA;
          B[0] ^= inB;
        }
      }
      // ---- lane changes at turning points: A->B after pass 0, B->A after pass 1 ----
      const uint32_t tag = pass == 0 ? TAG_SWITCH_AB : TAG_SWITCH_BA;
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        uint32_t live[4], mv[4];
#pragma unroll
        for (int w = 0; w < 4; ++w)
          live[w] = T[4 * h + w] & (pass == 0 ? (A[4 * h + w] & ~B[4 * h + w]) : (B[4 * h + w] & ~A[4 * h + w]));
        lazy_less(mv, live, D.keys, (uint32_t)(2 * u + h), gs, tlo, ctr3(tag, 0, 0, thi), D.t_omega, np_w);
#pragma unroll
        for (int w = 0; w < 4; ++w) {
          A[4 * h + w] ^= mv[w];
          B[4 * h + w] ^= mv[w];
        }
      }
    }
    const long long t = m + 1;
    // occupancy profile at epoch ends
    if (D.period > 0 && (t % D.period) == 0 && active) {
      uint32_t* oa = D.occA + (size_t)s * 32 * D.W + 256 * (size_t)u;
      uint32_t* ob = D.occB + (size_t)s * 32 * D.W + 256 * (size_t)u;
#pragma unroll 1
      for (int w = 0; w < nwn; ++w) {
        const uint32_t a = A[w], b = B[w];
#pragma unroll 4
        for (int k = 0; k < 32; ++k) {
          oa[32 * w + k] += (a >> k) & 1u;
          ob[32 * w + k] += (b >> k) & 1u;
        }
      }
    }
    if (t == next_rec) {
      unsigned long long na = 0, nb = 0;
#pragma unroll
      for (int w = 0; w < 8; ++w) {
        na += __popc(A[w]);
        nb += __popc(B[w]);
      }
      unsigned long long tot[4];
      block_sum4(jA, jB, na, nb, tot);
      if (threadIdx.x == 0) {
        const size_t cell = (size_t)ri * D.S + s, plane = (size_t)R.nt * D.S;
        R.rec[cell] = (long long)(D.JA[s] + tot[0]);
        R.rec[plane + cell] = (long long)(D.JB[s] + tot[1]);
        R.rec[2 * plane + cell] = (long long)tot[2];
        R.rec[3 * plane + cell] = (long long)tot[3];
      }
      ++ri;
      next_rec = ri < R.nt ? R.rec_t[ri] : -1;
    }
  }
  {
    unsigned long long tot[4];
    block_sum4(jA, jB, 0, 0, tot);
    if (threadIdx.x == 0) {
      D.JA[s] += tot[0];
      D.JB[s] += tot[1];
    }
  }
  if (active) {
#pragma unroll
    for (int h = 0; h < 2; ++h) {
      *reinterpret_cast<uint4*>(D.A + row + 4 * h) = make_uint4(A[4 * h], A[4 * h + 1], A[4 * h + 2], A[4 * h + 3]);
      *reinterpret_cast<uint4*>(D.B + row + 4 * h) = make_uint4(B[4 * h], B[4 * h + 1], B[4 * h + 2], B[4 * h + 3]);
      *reinterpret_cast<uint4*>(D.T + row + 4 * h) = make_uint4(T[4 * h], T[4 * h + 1], T[4 * h + 2], T[4 * h + 3]);
    }
  }
}

}  // namespace kpz
