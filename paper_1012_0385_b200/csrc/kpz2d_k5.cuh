// kpz2d_k5.cuh — K5 / K5S: checkerboard sweep of the 2+1D generalisation ("two-sub-lattice
// updates, which can be generalized to checker-board lattice decomposition in two dimensions"): the dimer /
// octahedron move of ref. [7] - a site moves when its x-pair AND its y-pair of slopes are both (1,0) (forward, rate p) or
// both (0,1) (backward, rate q).  Product code (CUDA path); shares nothing with oracle/.
//
// Layout (device workspace and shared memory alike): the slopes are DE-INTERLEAVED by the parity of x, as the 1+1D
// kernels keep their rings: word k of row y of plane EX holds sx[y][x] of the even sites x = 64 k + 2 j in bit
// j, OX the odd sites x = 64 k + 2 j + 1, EY / OY the same for sy; RH = Lx / 64 words per row and plane.  The active sites
// of a row of colour c = (y + o) & 1 are x = 2 j + c: exactly the bits of the row's parity-c words, in the element order
// of the random stream (element y * Lx/2 + j of stream PAIR).  So a pass is 32-bit word logic with no bit gather:
//   c = 0: x-pair (EX[y][k], OX[y][k]),                             y-pair (EY[y][k], EY[y+1][k]);
//   c = 1: x-pair (OX[y][k], EX[y][k] >> 1 | EX[y][k+1] << 31),      y-pair (OY[y][k], OY[y+1][k]).
// Who writes what in one pass: a parity row of sy is touched by ONE row of sites (rows of colour 0 use EY[y], EY[y+1]; their
// neighbours y +- 1 have colour 1 and use OY), the a side of the x-pair by its own thread only; a colour-1 row shifts its
// flips into EX[y][k] and EX[y][k+1], and the first of a thread's words also takes the carry of the thread to its left:
// those two are atomic XORs, everything else plain stores.  The public ABI speaks the natural layout (bit x & 31 of word
// x >> 5); k2d_nat_to_eo / k2d_eo_to_nat convert at the boundary.
//
// Thread = one Philox supergroup = 128 consecutive elements = 4 element-words (4 x 64 sites).  Acceptance U < T MSB-first
// over bit-planes: thresholds of at most two planes (p = 0.75, 0.5, 0.25 ...) take two unconditional,
// independent Philox calls; anything else the lazy plane loop (planes drawn while a candidate of the warp is undecided).
// Fast path: Lx a multiple of 256 - the 4 element-words of a supergroup lie in one row, share the colour and sit in
// consecutive words (128-bit loads / stores on the streamed path).
//   k2d_pass    one launch = one colour pass of every sample, in place in HBM / L2 (lattices beyond shared memory);
//   k2d_onchip  one CTA per sample, persistent over the whole kpz2d_run, all four planes in shared memory (64 KiB for
//               512 x 512): global memory is touched at the start and the end of the launch only.
#pragma once
#include "common.cuh"

namespace kpz {

struct Kpz2dDev {
  PhiloxKeys keys;
  Thresh t_p, t_q;
  int32_t offset_mode, first_sample, S;
  int32_t Lx, Ly, RH;  // RH = Lx / 64 words per row and parity plane
  int32_t n_ew;        // element-words (64 sites) per sample = Ly * RH
  int32_t n_sg;        // supergroups per sample = ceil(n_ew / 4)
  uint32_t* EX;        // [S][Ly][RH] each
  uint32_t* OX;
  uint32_t* EY;
  uint32_t* OY;
};

struct Kpz2dRun {
  long long t0, n_mcs;
  const long long* rec_t;  // [nt] record times (device)
  int32_t rec_begin, nt;
  long long* rec_h;        // [nt][S]
  long long* rec_h2;
};

// flat start h = (x + y) & 1: sx = sy = (x + y) & 1, i.e. even sites carry y & 1, odd sites its complement
__global__ void k2d_init_flat(uint32_t* EX, uint32_t* OX, uint32_t* EY, uint32_t* OY, int S, int Ly, int RH) {
  const size_t n = (size_t)S * Ly * RH;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int y = (int)((i / RH) % Ly);
    const uint32_t e = (y & 1) ? 0xFFFFFFFFu : 0u;
    EX[i] = e;
    OX[i] = ~e;
    EY[i] = e;
    OY[i] = ~e;
  }
}

// natural words [rows][2 RH] <-> parity planes [rows][RH]
__global__ void k2d_nat_to_eo(const uint32_t* words, size_t n /* rows * RH */, uint32_t* E, uint32_t* O) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const uint2 w = reinterpret_cast<const uint2*>(words)[i];
    uint32_t e, o;
    nat_to_eo(w.x, w.y, e, o);
    E[i] = e;
    O[i] = o;
  }
}
__global__ void k2d_eo_to_nat(const uint32_t* E, const uint32_t* O, size_t n, uint32_t* words) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    uint32_t w0, w1;
    eo_to_nat(E[i], O[i], w0, w1);
    reinterpret_cast<uint2*>(words)[i] = make_uint2(w0, w1);
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

// The thresholds as the sweep uses them (per launch constants, computed once per thread).
struct Rates2d {
  Thresh tp, tq;
  int lastf, lastb;                      // last plane whose threshold bit is 1 (-1: none)
  uint32_t pf_always, pf0, pf1, pf_two;  // two-plane form of T(p): always; bit of plane 0; of plane 1; "plane 1 matters"
  uint32_t pb_always, pb0, pb1, pb_two;
  bool two;                              // both thresholds need at most two planes
};
__device__ __forceinline__ Rates2d make_rates2d(const Kpz2dDev& D) {
  Rates2d r;
  r.tp = D.t_p;
  r.tq = D.t_q;
  r.lastf = D.t_p.value ? 31 - (__ffs(D.t_p.value) - 1) : -1;
  r.lastb = D.t_q.value ? 31 - (__ffs(D.t_q.value) - 1) : -1;
  r.pf_always = D.t_p.always ? ~0u : 0u;
  r.pf0 = 0u - (D.t_p.value >> 31);
  r.pf1 = 0u - ((D.t_p.value >> 30) & 1u);
  r.pf_two = r.lastf >= 1 ? ~0u : 0u;
  r.pb_always = D.t_q.always ? ~0u : 0u;
  r.pb0 = 0u - (D.t_q.value >> 31);
  r.pb1 = 0u - ((D.t_q.value >> 30) & 1u);
  r.pb_two = r.lastb >= 1 ? ~0u : 0u;
  r.two = r.lastf <= 1 && r.lastb <= 1;
  return r;
}

// Accepted moves of one supergroup: cf / cb = forward- / backward-eligible elements of its 4 element-words.
// Must be called by whole warps (the lazy loop votes).  TWO: both thresholds need at most two planes (r.two).
template <bool TWO>
__device__ __forceinline__ void accept2d(uint32_t (&hop)[4], const uint32_t (&cf)[4], const uint32_t (&cb)[4], const Rates2d& r,
                                         const PhiloxKeys& K, uint32_t G, uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps) {
  if constexpr (TWO) {  // [U < T] from the two leading planes: plane 0 decides unless it equals T's bit, then plane 1
    const uint4 v0 = philox4x32_10(G, gs, tlo, ctr3(TAG_PAIR, ps, 0u, thi), K);
    const uint4 v1 = philox4x32_10(G, gs, tlo, ctr3(TAG_PAIR, ps, 1u, thi), K);
    const uint32_t R0[4] = {v0.x, v0.y, v0.z, v0.w}, R1[4] = {v1.x, v1.y, v1.z, v1.w};
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t lf = r.pf_always | (r.pf0 & ~R0[k]) | (~(R0[k] ^ r.pf0) & r.pf1 & ~R1[k] & r.pf_two);
      const uint32_t lb = r.pb_always | (r.pb0 & ~R0[k]) | (~(R0[k] ^ r.pb0) & r.pb1 & ~R1[k] & r.pb_two);
      hop[k] = (cf[k] & lf) | (cb[k] & lb);
    }
    return;
  } else {
  uint32_t eqf[4], eqb[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    hop[k] = (r.tp.always ? cf[k] : 0u) | (r.tq.always ? cb[k] : 0u);
    eqf[k] = (r.tp.always || r.tp.value == 0u) ? 0u : cf[k];
    eqb[k] = (r.tq.always || r.tq.value == 0u) ? 0u : cb[k];
  }
#pragma unroll 1
  for (int pl = 0; pl < 32; ++pl) {
    if (pl > r.lastf)
#pragma unroll
      for (int k = 0; k < 4; ++k) eqf[k] = 0u;  // an equal prefix can no longer become "less"
    if (pl > r.lastb)
#pragma unroll
      for (int k = 0; k < 4; ++k) eqb[k] = 0u;
    const uint32_t any = eqf[0] | eqf[1] | eqf[2] | eqf[3] | eqb[0] | eqb[1] | eqb[2] | eqb[3];
    if (!__any_sync(0xFFFFFFFFu, any != 0u)) break;
    const uint4 v = philox4x32_10(G, gs, tlo, ctr3(TAG_PAIR, ps, (uint32_t)pl, thi), K);
    const uint32_t R[4] = {v.x, v.y, v.z, v.w};
    const uint32_t tf = 0u - ((r.tp.value >> (31 - pl)) & 1u), tb = 0u - ((r.tq.value >> (31 - pl)) & 1u);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      hop[k] |= (eqf[k] & tf & ~R[k]) | (eqb[k] & tb & ~R[k]);
      eqf[k] &= ~(R[k] ^ tf);
      eqb[k] &= ~(R[k] ^ tb);
    }
  }
  }
}

// One colour pass of supergroup G of one sample whose planes start at EX, OX, EY, OY with row stride RS words; PAD
// (shared memory) inserts one pad word per 4 words of a row: consecutive lanes own consecutive blocks of 4 words, and a
// lane stride of 5 words spreads the 32 lanes of a load over 32 banks.  live = this thread holds a supergroup (every
// thread of the warp calls: the lazy loop votes).  ROWALIGNED: RH % 4 == 0, the supergroup lies in one row.
template <bool PAD, bool ROWALIGNED, bool TWO>
__device__ __forceinline__ void sweep_supergroup(uint32_t* EX, uint32_t* OX, uint32_t* EY, uint32_t* OY, int RS, int RH, int Ly,
                                                 int n_ew, int G, bool live, uint32_t o, const Rates2d& r,
                                                 const PhiloxKeys& K, uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps) {
  auto W = [](int k) { return PAD ? k + (k >> 2) : k; };
  if constexpr (ROWALIGNED) {
    const int sgr = RH / 4;  // supergroups per row
    const int y = live ? G / sgr : 0, kq = live ? G - y * sgr : 0;
    const uint32_t c = ((uint32_t)y + o) & 1u;
    const int b0 = y * RS + W(4 * kq), b1 = (y + 1 == Ly ? 0 : y + 1) * RS + W(4 * kq);
    const int nxt = y * RS + (kq + 1 == sgr ? 0 : W(4 * (kq + 1)));
    uint32_t* PA = c ? OX : EX;  // the a side of the x-pair: the active sites themselves
    uint32_t* PY = c ? OY : EY;
    uint32_t a[4] = {0, 0, 0, 0}, e[5] = {0, 0, 0, 0, 0}, b[4] = {0, 0, 0, 0}, ya[4] = {0, 0, 0, 0}, yb[4] = {0, 0, 0, 0};
    if (live) {
      if constexpr (!PAD) {  // 16-byte aligned: 128-bit loads
        const uint4 va = *reinterpret_cast<const uint4*>(PA + b0), v1 = *reinterpret_cast<const uint4*>(PY + b0),
                    v2 = *reinterpret_cast<const uint4*>(PY + b1);
        a[0] = va.x; a[1] = va.y; a[2] = va.z; a[3] = va.w;
        ya[0] = v1.x; ya[1] = v1.y; ya[2] = v1.z; ya[3] = v1.w;
        yb[0] = v2.x; yb[1] = v2.y; yb[2] = v2.z; yb[3] = v2.w;
        const uint4 vb = *reinterpret_cast<const uint4*>((c ? EX : OX) + b0);
        e[0] = vb.x; e[1] = vb.y; e[2] = vb.z; e[3] = vb.w;
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          a[k] = PA[b0 + k];
          ya[k] = PY[b0 + k];
          yb[k] = PY[b1 + k];
          e[k] = (c ? EX : OX)[b0 + k];
        }
      }
      if (c) {
        e[4] = EX[nxt];
#pragma unroll
        for (int k = 0; k < 4; ++k) b[k] = __funnelshift_r(e[k], e[k + 1], 1);
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) b[k] = e[k];
      }
    }
    uint32_t cf[4], cb[4], hop[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      cf[k] = a[k] & ~b[k] & ya[k] & ~yb[k];  // both pairs (1,0)
      cb[k] = ~a[k] & b[k] & ~ya[k] & yb[k];  // both pairs (0,1)
    }
    accept2d<TWO>(hop, cf, cb, r, K, (uint32_t)G, gs, tlo, thi, ps);
    if (!live) return;
    if constexpr (!PAD) {
      *reinterpret_cast<uint4*>(PA + b0) = make_uint4(a[0] ^ hop[0], a[1] ^ hop[1], a[2] ^ hop[2], a[3] ^ hop[3]);
      *reinterpret_cast<uint4*>(PY + b0) = make_uint4(ya[0] ^ hop[0], ya[1] ^ hop[1], ya[2] ^ hop[2], ya[3] ^ hop[3]);
      *reinterpret_cast<uint4*>(PY + b1) = make_uint4(yb[0] ^ hop[0], yb[1] ^ hop[1], yb[2] ^ hop[2], yb[3] ^ hop[3]);
    } else {
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        PA[b0 + k] = a[k] ^ hop[k];
        PY[b0 + k] = ya[k] ^ hop[k];
        PY[b1 + k] = yb[k] ^ hop[k];
      }
    }
    if (c) {  // the b side is the even site one to the right: bit j + 1, carried into the next word
#pragma unroll
      for (int k = 1; k < 4; ++k) EX[b0 + k] = e[k] ^ (hop[k] << 1) ^ (hop[k - 1] >> 31);
      if (hop[0] << 1) atomicXor(&EX[b0], hop[0] << 1);  // word 0 also takes the carry of the thread to the left
      if (hop[3] >> 31) atomicXor(&EX[nxt], 1u);
    } else {
      if constexpr (!PAD) {
        *reinterpret_cast<uint4*>(OX + b0) = make_uint4(b[0] ^ hop[0], b[1] ^ hop[1], b[2] ^ hop[2], b[3] ^ hop[3]);
      } else {
#pragma unroll
        for (int k = 0; k < 4; ++k) OX[b0 + k] = b[k] ^ hop[k];
      }
    }
  } else {
    // any Lx that is a multiple of 64: the supergroup's element-words may span rows (and colours); word by word
    uint32_t cf[4], cb[4], hop[4];
    int i0[4], i1[4], in[4];
    uint32_t cc[4];
    int yy = (4 * G) / RH, kk = (4 * G) - yy * RH;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      cf[k] = cb[k] = 0u;
      const int y = yy, kb = kk;
      if (++kk == RH) {  // the next element-word starts the next row
        kk = 0;
        ++yy;
      }
      const bool ok = live && 4 * G + k < n_ew;
      cc[k] = ((uint32_t)y + o) & 1u;
      i0[k] = y * RS + W(kb);
      i1[k] = (y + 1 >= Ly ? 0 : y + 1) * RS + W(kb);
      in[k] = y * RS + W(kb + 1 == RH ? 0 : kb + 1);
      if (ok) {
        uint32_t a, b, ya, yb;
        if (cc[k] == 0u) {
          a = EX[i0[k]];
          b = OX[i0[k]];
          ya = EY[i0[k]];
          yb = EY[i1[k]];
        } else {
          a = OX[i0[k]];
          b = __funnelshift_r(EX[i0[k]], EX[in[k]], 1);
          ya = OY[i0[k]];
          yb = OY[i1[k]];
        }
        cf[k] = a & ~b & ya & ~yb;
        cb[k] = ~a & b & ~ya & yb;
      }
    }
    accept2d<TWO>(hop, cf, cb, r, K, (uint32_t)G, gs, tlo, thi, ps);
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const uint32_t h = hop[k];  // candidates of a missing element-word are empty, so is h
      if (h == 0u) continue;
      if (cc[k] == 0u) {  // every word below is touched by this element-word alone in this pass
        EX[i0[k]] ^= h;
        OX[i0[k]] ^= h;
        EY[i0[k]] ^= h;
        EY[i1[k]] ^= h;
      } else {
        OX[i0[k]] ^= h;
        OY[i0[k]] ^= h;
        OY[i1[k]] ^= h;
        if (h << 1) atomicXor(&EX[i0[k]], h << 1);
        if (h >> 31) atomicXor(&EX[in[k]], 1u);
      }
    }
  }
}

// K5: one colour pass (MCS m, pass ps) of every sample, in place.  off[s] = colour offset o of this pass.
template <bool ROWALIGNED, bool TWO>
__global__ void __launch_bounds__(128) k2d_pass(const __grid_constant__ Kpz2dDev D, const unsigned char* __restrict__ off,
                                                long long m, int ps) {
  const long long gid = (long long)blockIdx.x * 128 + threadIdx.x;
  const bool live = gid < (long long)D.S * D.n_sg;
  const int s = live ? (int)(gid / D.n_sg) : 0;
  const int G = live ? (int)(gid - (long long)s * D.n_sg) : 0;
  const size_t base = (size_t)s * D.Ly * D.RH;
  const Rates2d r = make_rates2d(D);
  sweep_supergroup<false, ROWALIGNED, TWO>(D.EX + base, D.OX + base, D.EY + base, D.OY + base, D.RH, D.RH, D.Ly, D.n_ew, G, live,
                                      off[s], r, D.keys, (uint32_t)(D.first_sample + s), (uint32_t)m,
                                      (uint32_t)((unsigned long long)m >> 32), (uint32_t)ps);
}

// Exact sums of h and h^2 of one sample from its planes (row stride RS, PAD as above): thread = column x, strided by nthr.
// h(x,0) = 2 (occupied bonds among sx[0][0..x]) - (x + 1): even sites 0..x are bits 0..x/2 of EX[0], odd ones bits
// 0..(x-1)/2 of OX[0]; h(x,y) = h(x,y-1) + 2 sy[y][x] - 1.  MODE 1 also writes h[y][x].
template <bool PAD, int MODE>
__device__ __forceinline__ void column_sums(const uint32_t* EX, const uint32_t* OX, const uint32_t* EY, const uint32_t* OY, int RS,
                                            int Lx, int Ly, int x0, int nthr, long long& s1, long long& s2, int32_t* h_out) {
  auto W = [](int k) { return PAD ? k + (k >> 2) : k; };
  for (int x = x0; x < Lx; x += nthr) {
    const int ne = x / 2 + 1, no = (x + 1) / 2;
    int cnt = 0;
    for (int w = 0; w < (ne >> 5); ++w) cnt += __popc(EX[W(w)]);
    if (ne & 31) cnt += __popc(EX[W(ne >> 5)] & ((1u << (ne & 31)) - 1u));
    for (int w = 0; w < (no >> 5); ++w) cnt += __popc(OX[W(w)]);
    if (no & 31) cnt += __popc(OX[W(no >> 5)] & ((1u << (no & 31)) - 1u));
    int h = 2 * cnt - (x + 1);
    const uint32_t* col = (x & 1) ? OY : EY;
    const int jw = W((x >> 1) >> 5), jb = (x >> 1) & 31;
    for (int y = 0; y < Ly; ++y) {
      if (y > 0) h += 2 * (int)((col[(size_t)y * RS + jw] >> jb) & 1u) - 1;
      if (MODE == 1) h_out[(size_t)y * Lx + x] = h;
      s1 += h;
      s2 += (long long)h * h;
    }
  }
}

// block-wide sum of (s1, s2) into thread 0 (NW warps)
template <int NW>
__device__ __forceinline__ void block_sum2(long long& s1, long long& s2, long long* red /* [2 * NW] shared */) {
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    s1 += __shfl_down_sync(0xFFFFFFFFu, s1, d);
    s2 += __shfl_down_sync(0xFFFFFFFFu, s2, d);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
    red[warp] = s1;
    red[NW + warp] = s2;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    s1 = s2 = 0;
    for (int k = 0; k < NW; ++k) {
      s1 += red[k];
      s2 += red[NW + k];
    }
  }
  __syncthreads();
}

// MODE 0: exact sums over a sample (grid = S * nxb blocks of 256 columns, atomicAdd per block); MODE 1: heights of one sample.
template <int MODE>
__global__ void __launch_bounds__(256) k2d_heights(const uint32_t* __restrict__ EX, const uint32_t* __restrict__ OX,
                                                   const uint32_t* __restrict__ EY, const uint32_t* __restrict__ OY, int Lx, int Ly,
                                                   int RH, int nxb, unsigned long long* out_h, unsigned long long* out_h2,
                                                   int32_t* h_out) {
  __shared__ long long red[16];
  const int s = blockIdx.x / nxb, x = (blockIdx.x % nxb) * 256 + threadIdx.x;
  const size_t base = (size_t)s * Ly * RH;
  long long s1 = 0, s2 = 0;
  column_sums<false, MODE>(EX + base, OX + base, EY + base, OY + base, RH, Lx, Ly, x < Lx ? x : Lx, Lx, s1, s2, h_out);
  if (MODE == 0) {
    block_sum2<8>(s1, s2, red);
    if (threadIdx.x == 0) {
      atomicAdd(out_h + s, (unsigned long long)s1);  // exact: two's-complement wrap-around addition
      atomicAdd(out_h2 + s, (unsigned long long)s2);
    }
  }
}

// K5S: a whole sample on chip.  A pass is sweep_supergroup on shared memory followed by ONE __syncthreads (a pass reads only
// bits no other thread of the pass touches, so nothing else orders it); colour offsets are drawn in the kernel 16 MCS at a
// time (one Philox call per lane + ballot); records are taken from shared memory.
constexpr int kK5SThreads = 512;

template <bool ROWALIGNED, bool TWO>
__global__ void __launch_bounds__(kK5SThreads, 2) k2d_onchip(const __grid_constant__ Kpz2dDev D, const __grid_constant__ Kpz2dRun A) {
  extern __shared__ __align__(16) uint32_t k5s_smem[];
  __shared__ long long red[2 * (kK5SThreads / 32)];
  const int s = blockIdx.x;
  const int RH = D.RH, RS = RH + (RH >> 2);  // padded row stride
  const int plane = D.Ly * RS;
  uint32_t* EX = k5s_smem;
  uint32_t* OX = EX + plane;
  uint32_t* EY = OX + plane;
  uint32_t* OY = EY + plane;
  const size_t base = (size_t)s * D.Ly * RH;
  for (int i = threadIdx.x; i < D.Ly * RH; i += kK5SThreads) {
    const int y = i / RH, k = i - y * RH, j = y * RS + k + (k >> 2);
    EX[j] = D.EX[base + i];
    OX[j] = D.OX[base + i];
    EY[j] = D.EY[base + i];
    OY[j] = D.OY[base + i];
  }
  __syncthreads();
  const int lane = threadIdx.x & 31;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const Rates2d r = make_rates2d(D);
  int ri = A.rec_begin;
  long long next_rec = ri < A.nt ? A.rec_t[ri] : -1;
  uint32_t offbits = 0;
  auto draw_offsets = [&](long long m) {  // bit 2 k + ps = offset of pass ps of MCS (m & ~15) + k
    const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
    const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), D.keys);
    offbits = __ballot_sync(0xFFFFFFFFu, w.x & 1u);
  };
  if (D.offset_mode == 0) draw_offsets(A.t0);
  for (long long m = A.t0; m < A.t0 + A.n_mcs; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    for (int ps = 0; ps < 2; ++ps) {
      const uint32_t o = D.offset_mode ? (uint32_t)ps : ((offbits >> (2 * ((int)m & 15) + ps)) & 1u);
      for (int G0 = 0; G0 < D.n_sg; G0 += kK5SThreads) {  // block-uniform trip count: every warp stays whole
        const int G = G0 + (int)threadIdx.x;
        sweep_supergroup<true, ROWALIGNED, TWO>(EX, OX, EY, OY, RS, RH, D.Ly, D.n_ew, G < D.n_sg ? G : 0, G < D.n_sg, o, r, D.keys, gs,
                                           tlo, thi, (uint32_t)ps);
      }
      __syncthreads();  // the next pass reads what this one flipped
    }
    const long long t = m + 1;
    if (t == next_rec) {  // block-uniform
      long long s1 = 0, s2 = 0;
      column_sums<true, 0>(EX, OX, EY, OY, RS, D.Lx, D.Ly, (int)threadIdx.x, kK5SThreads, s1, s2, nullptr);
      block_sum2<kK5SThreads / 32>(s1, s2, red);
      if (threadIdx.x == 0) {
        A.rec_h[(size_t)ri * D.S + s] = s1;
        A.rec_h2[(size_t)ri * D.S + s] = s2;
      }
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
    if (D.offset_mode == 0 && ((int)t & 15) == 0) draw_offsets(t);
  }
  for (int i = threadIdx.x; i < D.Ly * RH; i += kK5SThreads) {
    const int y = i / RH, k = i - y * RH, j = y * RS + k + (k >> 2);
    D.EX[base + i] = EX[j];
    D.OX[base + i] = OX[j];
    D.EY[base + i] = EY[j];
    D.OY[base + i] = OY[j];
  }
}

}  // namespace kpz
