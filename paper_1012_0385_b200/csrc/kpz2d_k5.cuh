// kpz2d_k5.cuh — K5: checkerboard sweep of the 2+1D generalisation ("two-sub-lattice
// updates, which can be generalized to checker-board lattice decomposition in two dimensions"): the dimer /
// octahedron move of ref. [7] - a site moves when its x-pair AND its y-pair of slopes are both (1,0) (forward, rate p) or
// both (0,1) (backward, rate q).  Product code (CUDA path); shares nothing with oracle/.
//
// Layout: slopes as bits, natural order: sx[s][y][x >> 5] bit (x & 31) = slope of bond ((x-1,y),(x,y)), sy likewise for
// bond ((x,y-1),(x,y)); RW = Lx / 32 words per row.
//
// One launch = one colour pass over all samples, IN PLACE.  Sites of one colour share no bond, so every bit is read and
// flipped by exactly one thread of the pass; what threads share are WORDS (the x+1 neighbour of a block's last site, and
// row y+1 of sy), so every flip is a `red.global.xor` on the word - commutative, no ownership, no scratch array, no
// second phase - and every read looks only at bits no other thread of the pass touches.
// Thread = one Philox supergroup = 128 consecutive elements of stream PAIR = 4 element-words = 4 x 64 sites (element j
// of row y is the site x = 2 j + ((y + o) & 1)); acceptance U < T MSB-first over bit-planes, both rate classes at once,
// lazily: planes are drawn only while a candidate of the warp is undecided.
#pragma once
#include "common.cuh"

namespace kpz {

struct Kpz2dDev {
  PhiloxKeys keys;
  Thresh t_p, t_q;
  int32_t offset_mode, first_sample, S;
  int32_t Lx, Ly, RW;        // RW = Lx / 32
  int32_t n_ew;              // element-words (64 sites) per sample = Lx * Ly / 64
  int32_t n_sg;              // supergroups per sample = ceil(n_ew / 4)
  uint32_t* sx;              // [S][Ly][RW]
  uint32_t* sy;
};

// flat start h = (x + y) & 1: sx = sy = (x + y) & 1
__global__ void k2d_init_flat(uint32_t* sx, uint32_t* sy, int S, int Ly, int RW) {
  const size_t n = (size_t)S * Ly * RW;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int y = (int)((i / RW) % Ly);
    const uint32_t w = (y & 1) ? 0x55555555u : 0xAAAAAAAAu;
    sx[i] = w;
    sy[i] = w;
  }
}

// offsets of np passes starting at global pass index p0 (pass = 2 m + ps): out[k * S + s]
__global__ void k2d_offsets(const __grid_constant__ PhiloxKeys K, int first_sample, int S, long long p0, int np, int offset_mode,
                            unsigned char* out) {
  const size_t n = (size_t)np * S;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int k = (int)(i / S), s = (int)(i % S);
    const unsigned long long gp = (unsigned long long)(p0 + k);
    const unsigned long long m = gp >> 1;
    const uint32_t ps = (uint32_t)(gp & 1ull);
    uint32_t o = ps;
    if (offset_mode == 0)
      o = philox4x32_10(0u, (uint32_t)(first_sample + s), (uint32_t)m, ctr3(TAG_OFFSET, ps, 0, (uint32_t)(m >> 32)), K).x & 1u;
    out[i] = (unsigned char)o;
  }
}

__device__ __forceinline__ uint32_t compress_even64(unsigned long long v) {  // even-position bits of 64 -> 32 bits
  return compress_even((uint32_t)v) | (compress_even((uint32_t)(v >> 32)) << 16);
}
__device__ __forceinline__ unsigned long long spread_even64(uint32_t v) {  // 32 bits -> even positions of 64
  return (unsigned long long)spread_even(v) | ((unsigned long long)spread_even(v >> 16) << 32);
}

// One colour pass (MCS m, pass ps) of every sample.  off[s] = colour offset o of this pass.
__global__ void __launch_bounds__(128) k2d_pass(const __grid_constant__ Kpz2dDev D, const unsigned char* __restrict__ off,
                                                long long m, int ps) {
  const long long gid = (long long)blockIdx.x * 128 + threadIdx.x;
  const bool live_thread = gid < (long long)D.S * D.n_sg;
  const int s = live_thread ? (int)(gid / D.n_sg) : 0;
  const int G = live_thread ? (int)(gid % D.n_sg) : 0;
  const uint32_t o = off[s];
  uint32_t* sx = D.sx + (size_t)s * D.Ly * D.RW;
  uint32_t* sy = D.sy + (size_t)s * D.Ly * D.RW;
  const int ewr = D.RW / 2;  // element-words per row

  // candidates of the 4 element-words, in element order: cf = forward-eligible, cb = backward-eligible
  uint32_t cf[4], cb[4];
  int ey[4], ek[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const int ew = 4 * G + k;
    cf[k] = cb[k] = 0u;
    ey[k] = ek[k] = 0;
    if (live_thread && ew < D.n_ew) {
      const int y = ew / ewr, kb = ew % ewr;
      ey[k] = y;
      ek[k] = kb;
      const uint32_t c = ((uint32_t)y + o) & 1u;  // active sites of this row: x = 2 j + c
      const uint32_t* rx = sx + (size_t)y * D.RW;
      const uint32_t* ra = sy + (size_t)y * D.RW;
      const uint32_t* rb = sy + (size_t)((y + 1) % D.Ly) * D.RW;
      const unsigned long long X = (unsigned long long)rx[2 * kb] | ((unsigned long long)rx[2 * kb + 1] << 32);
      const unsigned long long nx = rx[(2 * kb + 2) % D.RW] & 1u;  // slope of the bond right of the block's last site
      const unsigned long long Xn = (X >> 1) | (nx << 63);
      const unsigned long long Ya = (unsigned long long)ra[2 * kb] | ((unsigned long long)ra[2 * kb + 1] << 32);
      const unsigned long long Yb = (unsigned long long)rb[2 * kb] | ((unsigned long long)rb[2 * kb + 1] << 32);
      const unsigned long long f = X & ~Xn & Ya & ~Yb;  // both pairs (1,0)
      const unsigned long long b = ~X & Xn & ~Ya & Yb;  // both pairs (0,1)
      cf[k] = compress_even64(f >> c);
      cb[k] = compress_even64(b >> c);
    }
  }
  // U < T(p) on cf, U < T(q) on cb, MSB first, plane by plane while any lane of the warp is undecided
  uint32_t lt[4], eqf[4], eqb[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    lt[k] = (D.t_p.always ? cf[k] : 0u) | (D.t_q.always ? cb[k] : 0u);
    eqf[k] = (D.t_p.always || D.t_p.value == 0u) ? 0u : cf[k];
    eqb[k] = (D.t_q.always || D.t_q.value == 0u) ? 0u : cb[k];
  }
  const int lastf = D.t_p.value ? 31 - (__ffs(D.t_p.value) - 1) : -1;  // last plane whose threshold bit is 1
  const int lastb = D.t_q.value ? 31 - (__ffs(D.t_q.value) - 1) : -1;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
#pragma unroll 1
  for (int pl = 0; pl < 32; ++pl) {
    if (pl > lastf)
#pragma unroll
      for (int k = 0; k < 4; ++k) eqf[k] = 0u;  // an equal prefix can no longer become "less"
    if (pl > lastb)
#pragma unroll
      for (int k = 0; k < 4; ++k) eqb[k] = 0u;
    const uint32_t any = eqf[0] | eqf[1] | eqf[2] | eqf[3] | eqb[0] | eqb[1] | eqb[2] | eqb[3];
    if (!__any_sync(0xFFFFFFFFu, any != 0u)) break;
    const uint4 v = philox4x32_10((uint32_t)G, gs, tlo, ctr3(TAG_PAIR, (uint32_t)ps, (uint32_t)pl, thi), D.keys);
    const uint32_t R[4] = {v.x, v.y, v.z, v.w};
    const uint32_t tf = 0u - ((D.t_p.value >> (31 - pl)) & 1u), tb = 0u - ((D.t_q.value >> (31 - pl)) & 1u);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      lt[k] |= (eqf[k] & tf & ~R[k]) | (eqb[k] & tb & ~R[k]);
      eqf[k] &= ~(R[k] ^ tf);
      eqb[k] &= ~(R[k] ^ tb);
    }
  }
  // flips: site x flips sx[y][x], sx[y][x+1], sy[y][x], sy[y+1][x]
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    if (lt[k] == 0u) continue;
    const int y = ey[k], kb = ek[k];
    const uint32_t c = ((uint32_t)y + o) & 1u;
    const unsigned long long hop = spread_even64(lt[k]) << c;  // accepted moves at their site positions
    const unsigned long long fx = hop | (hop << 1);
    uint32_t* rx = sx + (size_t)y * D.RW;
    uint32_t* ra = sy + (size_t)y * D.RW;
    uint32_t* rb = sy + (size_t)((y + 1) % D.Ly) * D.RW;
    if ((uint32_t)fx) atomicXor(rx + 2 * kb, (uint32_t)fx);
    if ((uint32_t)(fx >> 32)) atomicXor(rx + 2 * kb + 1, (uint32_t)(fx >> 32));
    if (hop >> 63) atomicXor(rx + (2 * kb + 2) % D.RW, 1u);
    if ((uint32_t)hop) {
      atomicXor(ra + 2 * kb, (uint32_t)hop);
      atomicXor(rb + 2 * kb, (uint32_t)hop);
    }
    if ((uint32_t)(hop >> 32)) {
      atomicXor(ra + 2 * kb + 1, (uint32_t)(hop >> 32));
      atomicXor(rb + 2 * kb + 1, (uint32_t)(hop >> 32));
    }
  }
}

// Heights h(x,0) = sum_{i<=x} (2 sx[0][i] - 1), h(x,y) = h(x,y-1) + 2 sy[y][x] - 1: one thread per column.
// MODE 0: exact sums of h and h^2 over the sample (atomicAdd per block); MODE 1: write h[y][x] of one sample.
template <int MODE>
__global__ void __launch_bounds__(256) k2d_heights(const uint32_t* __restrict__ sx, const uint32_t* __restrict__ sy, int Lx,
                                                   int Ly, int RW, int nxb, unsigned long long* out_h,
                                                   unsigned long long* out_h2, int32_t* h_out) {
  const int s = blockIdx.x / nxb, x = (blockIdx.x % nxb) * 256 + threadIdx.x;
  const uint32_t* rx = sx + (size_t)s * Ly * RW;
  const uint32_t* ry = sy + (size_t)s * Ly * RW;
  long long s1 = 0, s2 = 0;
  if (x < Lx) {
    int cnt = 0;
    for (int w = 0; w < (x >> 5); ++w) cnt += __popc(rx[w]);
    cnt += __popc(rx[x >> 5] & (0xFFFFFFFFu >> (31 - (x & 31))));
    int h = 2 * cnt - (x + 1);
    for (int y = 0; y < Ly; ++y) {
      if (y > 0) h += 2 * (int)((ry[(size_t)y * RW + (x >> 5)] >> (x & 31)) & 1u) - 1;
      if (MODE == 1) h_out[(size_t)y * Lx + x] = h;
      s1 += h;
      s2 += (long long)h * h;
    }
  }
  if (MODE == 0) {
    __shared__ long long red[16];
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) {
      s1 += __shfl_down_sync(0xFFFFFFFFu, s1, d);
      s2 += __shfl_down_sync(0xFFFFFFFFu, s2, d);
    }
    const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    if (lane == 0) {
      red[warp] = s1;
      red[8 + warp] = s2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      long long a = 0, b = 0;
      for (int k = 0; k < 8; ++k) {
        a += red[k];
        b += red[8 + k];
      }
      atomicAdd(out_h + s, (unsigned long long)a);  // exact: two's-complement wrap-around addition
      atomicAdd(out_h2 + s, (unsigned long long)b);
    }
  }
}

}  // namespace kpz
