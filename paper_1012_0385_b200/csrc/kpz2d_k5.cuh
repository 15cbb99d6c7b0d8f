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

// ---- K5S: the same sweep with a whole sample ON CHIP ---------------------------------------------------------------
// One CTA per sample, persistent over the whole kpz2d_run: both slope fields live in shared memory (2 Lx Ly bits: 64 KiB
// for 512 x 512), global memory is touched at the start and at the end of the launch only (as in the 1+1D
// on-chip kernel).  On chip the slopes are DE-INTERLEAVED by the parity of x (as the 1+1D kernels do): word k
// of EX[y] holds sx[y][x] of the even sites x = 64 k + 2 j in bit j, OX[y] the odd sites, EY / OY the same for sy.  The
// active sites of a row of colour c = (y + o) & 1 are then exactly the bits of its parity-c words, in the element order of
// the random stream: no bit gather between site order and element order, all logic on 32-bit words:
//   c = 0: x-pair (EX[y][k], OX[y][k]), y-pair (EY[y][k], EY[y+1][k]);   c = 1: x-pair (OX[y][k], EX[y][k] >> 1 | next << 31),
//   y-pair (OY[y][k], OY[y+1][k]).
// In one pass a parity row of sy is touched by ONE row of sites only (rows of colour 0 use EY[y], EY[y+1]; their
// neighbours y +- 1 have colour 1 and use OY), so the sy flips are plain stores; so are the sx flips of a colour-0 row; a
// colour-1 row shifts its flips into EX[y][k] and EX[y][k+1], words it shares with the neighbouring element-word: those
// two are `atoms.xor`.  A pass ends with ONE __syncthreads.  Colour offsets are drawn in the kernel 16 MCS at a time (one
// Philox call per lane + ballot); records - exact sums of h and h^2 - are taken from shared memory, one thread per column.
struct Kpz2dRun {
  long long t0, n_mcs;
  const long long* rec_t;  // [nt] record times (device)
  int32_t rec_begin, nt;
  long long* rec_h;        // [nt][S]
  long long* rec_h2;
};

constexpr int kK5SThreads = 512;

__global__ void __launch_bounds__(kK5SThreads, 2) k2d_onchip(const __grid_constant__ Kpz2dDev D, const __grid_constant__ Kpz2dRun A) {
  extern __shared__ __align__(16) uint32_t k5s_smem[];
  const int s = blockIdx.x;
  const int RH = D.RW / 2;         // element-words (64 sites) per row = words per parity row
  // consecutive lanes own consecutive supergroups = blocks of 4 words of a parity row: one pad word per 4 words makes the
  // lane stride 5 words, so the 32 lanes of a load hit 32 different banks
  const int RHp = RH + (RH >> 2);
#define K5S_W(k) ((k) + ((k) >> 2))
  const int plane = D.Ly * RHp;
  uint32_t* EX = k5s_smem;
  uint32_t* OX = EX + plane;
  uint32_t* EY = OX + plane;
  uint32_t* OY = EY + plane;
  __shared__ long long red[2 * (kK5SThreads / 32)];
  uint32_t* gx = D.sx + (size_t)s * D.Ly * D.RW;
  uint32_t* gy = D.sy + (size_t)s * D.Ly * D.RW;
  for (int i = threadIdx.x; i < D.Ly * RH; i += kK5SThreads) {
    const int y = i / RH, k = i % RH;
    uint32_t e, o;
    nat_to_eo(gx[(size_t)y * D.RW + 2 * k], gx[(size_t)y * D.RW + 2 * k + 1], e, o);
    EX[y * RHp + K5S_W(k)] = e;
    OX[y * RHp + K5S_W(k)] = o;
    nat_to_eo(gy[(size_t)y * D.RW + 2 * k], gy[(size_t)y * D.RW + 2 * k + 1], e, o);
    EY[y * RHp + K5S_W(k)] = e;
    OY[y * RHp + K5S_W(k)] = o;
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const int lastf = D.t_p.value ? 31 - (__ffs(D.t_p.value) - 1) : -1;
  const int lastb = D.t_q.value ? 31 - (__ffs(D.t_q.value) - 1) : -1;
  int ri = A.rec_begin;
  long long next_rec = ri < A.nt ? A.rec_t[ri] : -1;
  uint32_t offbits = 0;
  auto draw_offsets = [&](long long m) {  // bit 2 k + ps = offset of pass ps of MCS (m & ~15) + k
    const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
    const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), D.keys);
    offbits = __ballot_sync(0xFFFFFFFFu, w.x & 1u);
  };
  if (D.offset_mode == 0) draw_offsets(A.t0);
  // fast path (see below): block-uniform
  const int sgr = RH / 4;  // supergroups per row
  const bool fast = (RH % 4) == 0 && lastf <= 1 && lastb <= 1;
  // T as masks over its two leading planes: always (T = 2^32), bit of plane 0, bit of plane 1, "plane 1 matters"
  const uint32_t pf_always = D.t_p.always ? ~0u : 0u, pf0 = 0u - (D.t_p.value >> 31), pf1 = 0u - ((D.t_p.value >> 30) & 1u);
  const uint32_t pb_always = D.t_q.always ? ~0u : 0u, pb0 = 0u - (D.t_q.value >> 31), pb1 = 0u - ((D.t_q.value >> 30) & 1u);
  const uint32_t pf_two = lastf >= 1 ? ~0u : 0u, pb_two = lastb >= 1 ? ~0u : 0u;
  for (long long m = A.t0; m < A.t0 + A.n_mcs; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    for (int ps = 0; ps < 2; ++ps) {
      const uint32_t o = D.offset_mode ? (uint32_t)ps : ((offbits >> (2 * ((int)m & 15) + ps)) & 1u);
      if (fast) {
        // Lx a multiple of 256 (the 4 element-words of a supergroup lie in ONE row, so they share the colour, the two
        // rows and - with the padding - consecutive word addresses) and thresholds of at most two planes (drawn
        // unconditionally: two independent Philox calls): straight-line code, every word loaded once and stored once.
        for (int G0 = 0; G0 < D.n_sg; G0 += kK5SThreads) {
          const int G = G0 + (int)threadIdx.x;
          if (G < D.n_sg) {
            const int y = G / sgr, kq = G - y * sgr;
            const uint32_t c = ((uint32_t)y + o) & 1u;
            const int b0 = y * RHp + 5 * kq, b1 = (y + 1 == D.Ly ? 0 : y + 1) * RHp + 5 * kq;
            uint32_t* PA = c ? OX : EX;   // the a side of the x-pair: the active sites themselves
            uint32_t* PY = c ? OY : EY;
            uint32_t a[4], e[5], b[4], ya[4], yb[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              a[k] = PA[b0 + k];
              ya[k] = PY[b0 + k];
              yb[k] = PY[b1 + k];
            }
            const int nxt = y * RHp + (kq + 1 == sgr ? 0 : 5 * (kq + 1));
            if (c) {
#pragma unroll
              for (int k = 0; k < 4; ++k) e[k] = EX[b0 + k];
              e[4] = EX[nxt];
#pragma unroll
              for (int k = 0; k < 4; ++k) b[k] = __funnelshift_r(e[k], e[k + 1], 1);
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) b[k] = OX[b0 + k];
            }
            const uint4 v0 = philox4x32_10((uint32_t)G, gs, tlo, ctr3(TAG_PAIR, (uint32_t)ps, 0u, thi), D.keys);
            const uint4 v1 = philox4x32_10((uint32_t)G, gs, tlo, ctr3(TAG_PAIR, (uint32_t)ps, 1u, thi), D.keys);
            const uint32_t R0[4] = {v0.x, v0.y, v0.z, v0.w}, R1[4] = {v1.x, v1.y, v1.z, v1.w};
            uint32_t hop[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const uint32_t cf = a[k] & ~b[k] & ya[k] & ~yb[k];  // both pairs (1,0)
              const uint32_t cb = ~a[k] & b[k] & ~ya[k] & yb[k];  // both pairs (0,1)
              // [U < T] from the two leading planes: plane 0 decides unless it equals T's bit, then plane 1
              const uint32_t lf = pf_always | (pf0 & ~R0[k]) | (~(R0[k] ^ pf0) & pf1 & ~R1[k] & pf_two);
              const uint32_t lb = pb_always | (pb0 & ~R0[k]) | (~(R0[k] ^ pb0) & pb1 & ~R1[k] & pb_two);
              hop[k] = (cf & lf) | (cb & lb);
            }
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              PA[b0 + k] = a[k] ^ hop[k];
              PY[b0 + k] = ya[k] ^ hop[k];
              PY[b1 + k] = yb[k] ^ hop[k];
            }
            if (c) {  // the b side is the even site one to the right: bit j + 1, carried into the next word
#pragma unroll
              for (int k = 1; k < 4; ++k) EX[b0 + k] = e[k] ^ (hop[k] << 1) ^ (hop[k - 1] >> 31);
              if (hop[0] << 1) atomicXor(&EX[b0], hop[0] << 1);  // word 0 also takes the carry of the previous thread
              if (hop[3] >> 31) atomicXor(&EX[nxt], 1u);
            } else {
#pragma unroll
              for (int k = 0; k < 4; ++k) OX[b0 + k] = b[k] ^ hop[k];
            }
          }
        }
      } else
      for (int G0 = 0; G0 < D.n_sg; G0 += kK5SThreads) {  // block-uniform trip count: every warp stays whole
        const int G = G0 + (int)threadIdx.x;
        const bool live_thread = G < D.n_sg;
        uint32_t cf[4], cb[4];
        int ey[4], ek[4];
        int yy = (4 * G) / RH, kk = (4 * G) - yy * RH;  // row and element-word of the supergroup's first 64 sites
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const int ew = 4 * G + k;
          cf[k] = cb[k] = 0u;
          ey[k] = yy;
          ek[k] = kk;
          if (++kk == RH) {  // the next element-word starts the next row
            kk = 0;
            ++yy;
          }
          if (live_thread && ew < D.n_ew) {
            const int y = ey[k], kb = ek[k];
            const uint32_t c = ((uint32_t)y + o) & 1u;
            const int r0 = y * RHp, r1 = (y + 1 == D.Ly ? 0 : y + 1) * RHp, w = K5S_W(kb);
            uint32_t a, b, ya, yb;
            if (c == 0u) {
              a = EX[r0 + w];
              b = OX[r0 + w];
              ya = EY[r0 + w];
              yb = EY[r1 + w];
            } else {
              a = OX[r0 + w];
              b = __funnelshift_r(EX[r0 + w], EX[r0 + K5S_W(kb + 1 == RH ? 0 : kb + 1)], 1);
              ya = OY[r0 + w];
              yb = OY[r1 + w];
            }
            cf[k] = a & ~b & ya & ~yb;  // both pairs (1,0)
            cb[k] = ~a & b & ~ya & yb;  // both pairs (0,1)
          }
        }
        uint32_t lt[4], eqf[4], eqb[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          lt[k] = (D.t_p.always ? cf[k] : 0u) | (D.t_q.always ? cb[k] : 0u);
          eqf[k] = (D.t_p.always || D.t_p.value == 0u) ? 0u : cf[k];
          eqb[k] = (D.t_q.always || D.t_q.value == 0u) ? 0u : cb[k];
        }
#pragma unroll 1
        for (int pl = 0; pl < 32; ++pl) {
          if (pl > lastf)
#pragma unroll
            for (int k = 0; k < 4; ++k) eqf[k] = 0u;
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
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const uint32_t hop = lt[k];  // accepted moves, bit j = the j-th active site of the element-word
          if (hop == 0u) continue;
          const int y = ey[k], kb = ek[k];
          const uint32_t c = ((uint32_t)y + o) & 1u;
          const int r0 = y * RHp, r1 = (y + 1 == D.Ly ? 0 : y + 1) * RHp, w = K5S_W(kb);
          if (c == 0u) {  // every word below is touched by this thread alone in this pass
            EX[r0 + w] ^= hop;
            OX[r0 + w] ^= hop;
            EY[r0 + w] ^= hop;
            EY[r1 + w] ^= hop;
          } else {
            OX[r0 + w] ^= hop;
            OY[r0 + w] ^= hop;
            OY[r1 + w] ^= hop;
            if (hop << 1) atomicXor(&EX[r0 + w], hop << 1);                       // site x + 1 = even site j + 1
            if (hop >> 31) atomicXor(&EX[r0 + K5S_W(kb + 1 == RH ? 0 : kb + 1)], 1u);  // ... of the next element-word
          }
        }
      }
      __syncthreads();  // the next pass reads what this one flipped
    }
    const long long t = m + 1;
    if (t == next_rec) {  // block-uniform
      long long s1 = 0, s2 = 0;
      for (int x = threadIdx.x; x < D.Lx; x += kK5SThreads) {
        // h(x,0) = 2 * (occupied bonds among sx[0][0..x]) - (x + 1): even sites 0..x are bits 0..x/2 of EX[0], odd ones
        // bits 0..(x-1)/2 of OX[0]
        const int ne = x / 2 + 1, no = (x + 1) / 2;
        int cnt = 0;
        for (int w = 0; w < (ne >> 5); ++w) cnt += __popc(EX[K5S_W(w)]);
        if (ne & 31) cnt += __popc(EX[K5S_W(ne >> 5)] & ((1u << (ne & 31)) - 1u));
        for (int w = 0; w < (no >> 5); ++w) cnt += __popc(OX[K5S_W(w)]);
        if (no & 31) cnt += __popc(OX[K5S_W(no >> 5)] & ((1u << (no & 31)) - 1u));
        int h = 2 * cnt - (x + 1);
        const uint32_t* col = (x & 1) ? OY : EY;
        const int jw = K5S_W((x >> 1) >> 5), jb = (x >> 1) & 31;
        for (int y = 0; y < D.Ly; ++y) {
          if (y > 0) h += 2 * (int)((col[y * RHp + jw] >> jb) & 1u) - 1;
          s1 += h;
          s2 += (long long)h * h;
        }
      }
#pragma unroll
      for (int d = 16; d >= 1; d >>= 1) {
        s1 += __shfl_down_sync(0xFFFFFFFFu, s1, d);
        s2 += __shfl_down_sync(0xFFFFFFFFu, s2, d);
      }
      const int warp = threadIdx.x >> 5;
      if (lane == 0) {
        red[warp] = s1;
        red[kK5SThreads / 32 + warp] = s2;
      }
      __syncthreads();
      if (threadIdx.x == 0) {
        long long a = 0, b = 0;
        for (int k = 0; k < kK5SThreads / 32; ++k) {
          a += red[k];
          b += red[kK5SThreads / 32 + k];
        }
        A.rec_h[(size_t)ri * D.S + s] = a;
        A.rec_h2[(size_t)ri * D.S + s] = b;
      }
      __syncthreads();
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
    if (D.offset_mode == 0 && ((int)t & 15) == 0) draw_offsets(t);
  }
  for (int i = threadIdx.x; i < D.Ly * RH; i += kK5SThreads) {
    const int y = i / RH, k = i % RH;
    uint32_t w0, w1;
    eo_to_nat(EX[y * RHp + K5S_W(k)], OX[y * RHp + K5S_W(k)], w0, w1);
    gx[(size_t)y * D.RW + 2 * k] = w0;
    gx[(size_t)y * D.RW + 2 * k + 1] = w1;
    eo_to_nat(EY[y * RHp + K5S_W(k)], OY[y * RHp + K5S_W(k)], w0, w1);
    gy[(size_t)y * D.RW + 2 * k] = w0;
    gy[(size_t)y * D.RW + 2 * k + 1] = w1;
  }
#undef K5S_W
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
