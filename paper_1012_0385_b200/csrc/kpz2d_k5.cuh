// kpz2d_k5.cuh — K5 / K5S / K5C: checkerboard sweep of the 2+1D generalisation ("two-sub-lattice
// updates, which can be generalized to checker-board lattice decomposition in two dimensions"): the dimer /
// octahedron move of ref. [7] - a site moves when its x-pair AND its y-pair of slopes are both (1,0) (forward, rate p) or
// both (0,1) (backward, rate q).  Product code (CUDA path); shares nothing with oracle/.
//
// Compiled twice: by nvcc into the library (generic in Lx, Ly, p, q: the kernels read them from Kpz2dDev) and, with
// K5J_LX / K5J_LY / K5J_TP... defined, at run time by NVRTC (csrc/jit.cu), where the shape and the thresholds are
// constants: the acceptance folds into one LOP3 per word and the address arithmetic disappears.  No host headers here.
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
// flips into EX[y][k] and EX[y][k+1], and the first of a thread's words also takes the carry of the thread to its left.
// The public ABI speaks the natural layout (bit x & 31 of word x >> 5); k2d_nat_to_eo / k2d_eo_to_nat (kpz2d_api.cu)
// convert at the boundary.
//
// Thread = one Philox supergroup = 128 consecutive elements = 4 element-words (4 x 64 sites).  Acceptance U < T MSB-first
// over bit-planes: thresholds of at most two planes (p = 0.75, 0.5, 0.25 ...) take two unconditional,
// independent Philox calls; anything else the lazy plane loop (planes drawn while a candidate of the warp is undecided).
// Fast path (ROWALIGNED): Lx a multiple of 256 - the 4 element-words of a supergroup lie in one row, share the colour and
// sit in 16 consecutive bytes (128-bit loads / stores, in shared memory too: consecutive lanes own consecutive 16-byte
// blocks, so a warp's access is conflict-free without padding).  Threads are mapped to supergroups BY ROW PARITY (first
// all even rows, then all odd rows), so the colour is uniform over a warp - over the whole CTA on chip - and each colour
// runs its own straight-line code.
//   K5  (pass_body: k2d_pass / kpz2d_k5_pass_jit)  one launch = one colour pass of every sample, in place in HBM / L2
//       (lattices beyond every on-chip variant); consecutive passes by programmatic dependent launch;
//   K5S (onchip_body: k2d_onchip / kpz2d_k5s_jit)  one CTA per sample, persistent over the whole kpz2d_run, all four planes
//       in shared memory (64 KiB for 512 x 512), rows stored by parity (even rows first): global memory is touched at the
//       start and the end of the launch only; planes drawn one sweep ahead around a split barrier;
//   K5C (cluster_body: kpz2d_k5c_jit)  the same with a sample spread over a thread-block cluster of 2 ... 16 CTAs, the
//       neighbour CTA's first row through distributed shared memory (1024 x 1024, 2048 x 2048).
#pragma once
#include "rtc_prelude.cuh"
#include "philox.cuh"
#include "sweep_types.cuh"
#include "height_lut.cuh"

#ifndef K5J_XRALL
#define K5J_XRALL 0  // 1: every warp of K5C reaches row y + 1 through shared::cluster addresses (debug)
#endif

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

// The shape as the kernels use it: kernel parameters under nvcc, compile-time constants under NVRTC.
struct Shape2d {
  int Lx, Ly, RH, n_ew, n_sg;
};
__device__ __forceinline__ Shape2d shape2d(const Kpz2dDev& D) {
#ifdef K5J_LX
  (void)D;
  return Shape2d{K5J_LX, K5J_LY, K5J_LX / 64, K5J_LX / 64 * K5J_LY, (K5J_LX / 64 * K5J_LY + 3) / 4};
#else
  return Shape2d{D.Lx, D.Ly, D.RH, D.n_ew, D.n_sg};
#endif
}

// The thresholds as the sweep uses them (per launch constants, computed once per thread; literals under NVRTC).
struct Rates2d {
  Thresh tp, tq;
  int lastf, lastb;                      // last plane whose threshold bit is 1 (-1: none)
  uint32_t pf_always, pf0, pf1, pf_two;  // two-plane form of T(p): always; bit of plane 0; of plane 1; "plane 1 matters"
  uint32_t pb_always, pb0, pb1, pb_two;
};
__device__ __forceinline__ int last_plane(uint32_t v) {  // 31 - ctz(v), -1 for 0; written so that a literal folds
  int last = -1;
#pragma unroll
  for (int b = 0; b < 32; ++b)
    if ((v >> (31 - b)) & 1u) last = b;
  return last;
}
__device__ __forceinline__ Rates2d make_rates2d(const Kpz2dDev& D) {
  Rates2d r;
#ifdef K5J_LX
  (void)D;
  r.tp.value = K5J_TP;
  r.tp.always = K5J_TP_ALWAYS;
  r.tq.value = K5J_TQ;
  r.tq.always = K5J_TQ_ALWAYS;
  r.lastf = last_plane(K5J_TP);
  r.lastb = last_plane(K5J_TQ);
#else
  r.tp = D.t_p;
  r.tq = D.t_q;
  r.lastf = D.t_p.value ? 31 - (__ffs(D.t_p.value) - 1) : -1;
  r.lastb = D.t_q.value ? 31 - (__ffs(D.t_q.value) - 1) : -1;
#endif
  r.pf_always = r.tp.always ? ~0u : 0u;
  r.pf0 = 0u - (r.tp.value >> 31);
  r.pf1 = 0u - ((r.tp.value >> 30) & 1u);
  r.pf_two = r.lastf >= 1 ? ~0u : 0u;
  r.pb_always = r.tq.always ? ~0u : 0u;
  r.pb0 = 0u - (r.tq.value >> 31);
  r.pb1 = 0u - ((r.tq.value >> 30) & 1u);
  r.pb_two = r.lastb >= 1 ? ~0u : 0u;
  return r;
}

// The two leading bit-planes of the 128 uniforms of supergroup G in colour pass (time, ps): two independent Philox calls.
struct Planes2 {
  uint4 v0, v1;
};
__device__ __forceinline__ Planes2 draw_two(const PhiloxKeys& K, uint32_t G, uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps) {
  Planes2 R;
  R.v0 = philox4x32_10(G, gs, tlo, ctr3(TAG_PAIR, ps, 0u, thi), K);
  R.v1 = philox4x32_10(G, gs, tlo, ctr3(TAG_PAIR, ps, 1u, thi), K);
  return R;
}
// [U < T] from the two leading planes: plane 0 decides unless it equals T's bit, then plane 1
__device__ __forceinline__ void accept_two(uint32_t (&hop)[4], const uint32_t (&cf)[4], const uint32_t (&cb)[4], const Rates2d& r,
                                           const Planes2& R) {
  const uint32_t R0[4] = {R.v0.x, R.v0.y, R.v0.z, R.v0.w}, R1[4] = {R.v1.x, R.v1.y, R.v1.z, R.v1.w};
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    const uint32_t lf = r.pf_always | (r.pf0 & ~R0[k]) | (~(R0[k] ^ r.pf0) & r.pf1 & ~R1[k] & r.pf_two);
    const uint32_t lb = r.pb_always | (r.pb0 & ~R0[k]) | (~(R0[k] ^ r.pb0) & r.pb1 & ~R1[k] & r.pb_two);
    hop[k] = (cf[k] & lf) | (cb[k] & lb);
  }
}

// Accepted moves of one supergroup: cf / cb = forward- / backward-eligible elements of its 4 element-words.
// Must be called by whole warps (the lazy loop votes).  TWO: both thresholds need at most two planes.
template <bool TWO>
__device__ __forceinline__ void accept2d(uint32_t (&hop)[4], const uint32_t (&cf)[4], const uint32_t (&cb)[4], const Rates2d& r,
                                         const PhiloxKeys& K, uint32_t G, uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps) {
  if constexpr (TWO) {
    accept_two(hop, cf, cb, r, draw_two(K, G, gs, tlo, thi, ps));
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

// Distributed shared memory of a thread-block cluster (K5C): a 32-bit shared::cluster address names a word of any CTA
// of the cluster (mapa), loads / stores on it reach that CTA's shared memory; barrier.cluster orders them.
__device__ __forceinline__ uint32_t smem_addr(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ uint32_t cluster_ctarank() {
  uint32_t r;
  asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
  return r;
}
__device__ __forceinline__ uint32_t mapa(uint32_t cta_addr, uint32_t rank) {
  uint32_t r;
  asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(cta_addr), "r"(rank));
  return r;
}
__device__ __forceinline__ uint4 ld4_cluster(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared::cluster.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void st4_cluster(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  asm volatile("st.shared::cluster.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ int ld_cluster_s32(uint32_t a) {
  int v;
  asm volatile("ld.shared::cluster.s32 %0, [%1];" : "=r"(v) : "r"(a) : "memory");
  return v;
}
__device__ __forceinline__ void cluster_arrive() { asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory"); }
__device__ __forceinline__ void cluster_wait() { asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory"); }

__device__ __forceinline__ uint4 ld4(const uint32_t* p) { return *reinterpret_cast<const uint4*>(p); }
__device__ __forceinline__ void st4(uint32_t* p, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
  *reinterpret_cast<uint4*>(p) = make_uint4(x, y, z, w);
}

// Fast path: one supergroup (4 consecutive element-words) of a row of colour C.  P0 = word offset of the supergroup in
// its own row (the same in every plane, a multiple of 4: 16-byte accesses), P1 = the same words of row y + 1, NX = the
// word that follows the supergroup in its row (wrapping to the row's first word).  live = this thread holds a supergroup
// (every thread of the warp calls: the lazy loop votes).
// RIW ("row in warp"): the sgr supergroups of a row are sgr consecutive lanes of ONE warp and the warp is whole: the
// word to the right and the carry from the left then travel by shuffle and every store is a plain 128-bit store;
// otherwise word NX is loaded and the two carries are atomic XORs.
// pre != nullptr (a compile-time fact at every call site): the two planes were drawn earlier (software pipeline).
// XR: the words of row y + 1 are reached through the shared::cluster address xr1 (they may lie in the next CTA of the
// cluster: K5C) instead of PY + P1.
template <bool TWO, int C, bool RIW, bool XR = false>
__device__ __forceinline__ void sweep_row_supergroup(uint32_t* EX, uint32_t* OX, uint32_t* EY, uint32_t* OY, int P0, int P1, int NX,
                                                     int kq, int sgr, uint32_t G, bool live, const Rates2d& r, const PhiloxKeys& K,
                                                     uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps,
                                                     const Planes2* pre = nullptr, uint32_t xr1 = 0) {
  uint32_t* PA = C ? OX : EX;  // the a side of the x-pair: the active sites themselves
  uint32_t* PB = C ? EX : OX;  // the b side: the neighbour to the right
  uint32_t* PY = C ? OY : EY;
  uint4 va = make_uint4(0, 0, 0, 0), vb = va, v0 = va, v1 = va;
  uint32_t e4 = 0;
  if (live) {
    va = ld4(PA + P0);
    vb = ld4(PB + P0);
    v0 = ld4(PY + P0);
    v1 = XR ? ld4_cluster(xr1) : ld4(PY + P1);
    if (C && !RIW) e4 = PB[NX];
  }
  const int lane = (int)(threadIdx.x & 31u);
  if (C && RIW) e4 = __shfl_sync(0xFFFFFFFFu, vb.x, kq + 1 == sgr ? lane - (sgr - 1) : lane + 1);
  const uint32_t a[4] = {va.x, va.y, va.z, va.w}, e[5] = {vb.x, vb.y, vb.z, vb.w, e4};
  const uint32_t ya[4] = {v0.x, v0.y, v0.z, v0.w}, yb[4] = {v1.x, v1.y, v1.z, v1.w};
  uint32_t b[4], cf[4], cb[4], hop[4];
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    b[k] = C ? __funnelshift_r(e[k], e[k + 1], 1) : e[k];  // colour 1: the even site one to the right
    cf[k] = a[k] & ~b[k] & ya[k] & ~yb[k];                 // both pairs (1,0)
    cb[k] = ~a[k] & b[k] & ~ya[k] & yb[k];                 // both pairs (0,1)
  }
  if (pre)
    accept_two(hop, cf, cb, r, *pre);
  else
    accept2d<TWO>(hop, cf, cb, r, K, G, gs, tlo, thi, ps);
  uint32_t cin = 0;
  if (C && RIW) cin = __shfl_sync(0xFFFFFFFFu, hop[3] >> 31, kq == 0 ? lane + (sgr - 1) : lane - 1);
  if (!live) return;
  st4(PA + P0, a[0] ^ hop[0], a[1] ^ hop[1], a[2] ^ hop[2], a[3] ^ hop[3]);
  st4(PY + P0, ya[0] ^ hop[0], ya[1] ^ hop[1], ya[2] ^ hop[2], ya[3] ^ hop[3]);
  if (XR)
    st4_cluster(xr1, yb[0] ^ hop[0], yb[1] ^ hop[1], yb[2] ^ hop[2], yb[3] ^ hop[3]);
  else
    st4(PY + P1, yb[0] ^ hop[0], yb[1] ^ hop[1], yb[2] ^ hop[2], yb[3] ^ hop[3]);
  if (C) {  // the b side is bit j + 1 of EX: the flips move up by one bit, the top bit into the next word
    const uint32_t f1 = __funnelshift_l(hop[0], hop[1], 1), f2 = __funnelshift_l(hop[1], hop[2], 1),
                   f3 = __funnelshift_l(hop[2], hop[3], 1);
    if (RIW) {
      st4(EX + P0, e[0] ^ (hop[0] << 1) ^ cin, e[1] ^ f1, e[2] ^ f2, e[3] ^ f3);
    } else {  // word 0 also takes the carry of the thread to the left, word NX this thread's
      EX[P0 + 1] = e[1] ^ f1;
      EX[P0 + 2] = e[2] ^ f2;
      EX[P0 + 3] = e[3] ^ f3;
      if (hop[0] << 1) atomicXor(&EX[P0], hop[0] << 1);
      if (hop[3] >> 31) atomicXor(&EX[NX], 1u);
    }
  } else {
    st4(OX + P0, b[0] ^ hop[0], b[1] ^ hop[1], b[2] ^ hop[2], b[3] ^ hop[3]);
  }
}

// Any Lx that is a multiple of 64: the supergroup's element-words may span rows (and colours); word by word, rows in
// natural order with stride RH.
template <bool TWO>
__device__ __forceinline__ void sweep_ragged_supergroup(uint32_t* EX, uint32_t* OX, uint32_t* EY, uint32_t* OY, int RH, int Ly,
                                                        int n_ew, int G, bool live, uint32_t o, const Rates2d& r,
                                                        const PhiloxKeys& K, uint32_t gs, uint32_t tlo, uint32_t thi, uint32_t ps) {
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
    i0[k] = y * RH + kb;
    i1[k] = (y + 1 >= Ly ? 0 : y + 1) * RH + kb;
    in[k] = y * RH + (kb + 1 == RH ? 0 : kb + 1);
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

// K5: one colour pass (MCS m, pass ps) of every sample, in place.  off[s] = colour offset o of this pass.  Thread =
// (sample, supergroup); on the fast path the supergroups of a sample are taken by row parity, so a warp has one colour.
// PDL (programmatic dependent launch; the host sets the launch attribute): the launch of the NEXT pass may begin while this
// one is still running - its threads draw their planes, which depend on nothing in memory, and only then wait
// (griddepcontrol.wait) for this pass to be complete and visible.  Hides the launch gap between two passes.
template <bool ROWALIGNED, bool TWO, bool PDL = false>
__device__ __forceinline__ void pass_body(const Kpz2dDev& D, const unsigned char* __restrict__ off, long long m, int ps) {
  if constexpr (PDL) asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
  const Shape2d sh = shape2d(D);
  const long long gid = (long long)blockIdx.x * 128 + threadIdx.x;
  const bool live = gid < (long long)D.S * sh.n_sg;
  const int s = live ? (int)(gid / sh.n_sg) : 0;
  const int i = live ? (int)(gid - (long long)s * sh.n_sg) : 0;
  const size_t base = (size_t)s * sh.Ly * sh.RH;
  uint32_t *EX = D.EX + base, *OX = D.OX + base, *EY = D.EY + base, *OY = D.OY + base;
  const Rates2d r = make_rates2d(D);
  const uint32_t gs = (uint32_t)(D.first_sample + s), tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
  if constexpr (ROWALIGNED) {
    const int sgr = sh.RH / 4, nh = sh.n_sg / 2;  // supergroups per row; per row parity
    const int h = i >= nh ? 1 : 0, ii = i - h * nh;
    const int rr = ii / sgr, kq = ii - rr * sgr, y = 2 * rr + h;
    const int P0 = y * sh.RH + 4 * kq, P1 = (y + 1 == sh.Ly ? 0 : y + 1) * sh.RH + 4 * kq;
    const int NX = y * sh.RH + (kq + 1 == sgr ? 0 : 4 * (kq + 1));
    const uint32_t G = (uint32_t)(y * sgr + kq);
    Planes2 R;
    const Planes2* pre = nullptr;
    if constexpr (PDL && TWO) {  // drawn before anything of the previous pass is needed
      R = draw_two(D.keys, G, gs, tlo, thi, (uint32_t)ps);
      asm volatile("" ::"r"(R.v0.x), "r"(R.v0.y), "r"(R.v0.z), "r"(R.v0.w), "r"(R.v1.x), "r"(R.v1.y), "r"(R.v1.z), "r"(R.v1.w));
      pre = &R;
    }
    if constexpr (PDL) asm volatile("griddepcontrol.wait;" ::: "memory");
    const uint32_t o = off[s];
    // one colour per warp whenever nh is a multiple of 32; a warp that straddles samples or parities goes word by word
    const unsigned c1 = __ballot_sync(0xFFFFFFFFu, (((uint32_t)h + o) & 1u) != 0u);
    if (c1 == 0xFFFFFFFFu)
      sweep_row_supergroup<TWO, 1, false>(EX, OX, EY, OY, P0, P1, NX, kq, sgr, G, live, r, D.keys, gs, tlo, thi, (uint32_t)ps, pre);
    else if (c1 == 0u)
      sweep_row_supergroup<TWO, 0, false>(EX, OX, EY, OY, P0, P1, NX, kq, sgr, G, live, r, D.keys, gs, tlo, thi, (uint32_t)ps, pre);
    else
      sweep_ragged_supergroup<TWO>(EX, OX, EY, OY, sh.RH, sh.Ly, sh.n_ew, (int)G, live, o, r, D.keys, gs, tlo, thi, (uint32_t)ps);
  } else {
    if constexpr (PDL) asm volatile("griddepcontrol.wait;" ::: "memory");
    sweep_ragged_supergroup<TWO>(EX, OX, EY, OY, sh.RH, sh.Ly, sh.n_ew, i, live, off[s], r, D.keys, gs, tlo, thi, (uint32_t)ps);
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

// Sums over one row (RH even-site words ex, RH odd-site words ox) of the heights relative to the height before its
// site 0, with the byte table of height_lut.cuh (8 sites per lookup): S1 = sum, S2 = sum of squares.
__device__ __forceinline__ void row_relative_sums(const uint32_t* ex, const uint32_t* ox, int RH, const uint32_t* lut,
                                                  long long& S1, long long& S2) {
  long long R = 0;
  S1 = S2 = 0;
  for (int k = 0; k < RH; k += 4) {
    const int nw = RH - k < 4 ? RH - k : 4;
    uint32_t P[4], Q[4];
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      P[w] = w < nw ? ex[k + w] : 0u;
      Q[w] = w < nw ? ox[k + w] : 0u;
    }
    int rg, s1g, s2g;
    unit_relative_sums_lut(P, Q, nw, lut, rg, s1g, s2g);
    const long long n = 64LL * nw;
    S1 += n * R + s1g;
    S2 += n * R * R + 2 * R * s1g + s2g;
    R += rg;
  }
}

// Exact sums of h and h^2 of a sample in shared memory, ROW BY ROW: inside row y the heights integrate along x exactly as
// on a 1+1D ring, h(x,y) = B(y) + sum_{x'<=x} (2 sx[y][x'] - 1), so a thread takes a row (row_relative_sums) and the row
// bases come from one block-wide scan of column 0: B(y) = h(0,y) - (2 sx[y][0] - 1), h(0,y) = h(0,0) + sum_{y'=1..y}
// (2 sy[y'][0] - 1).  Equal to the column-wise definition on every single-valued surface - which the
// dynamics preserve (every move flips the four slopes around one site) - and about ten times cheaper than walking each
// column bit by bit.  NT threads, all call.
// The planes hold rows yg0 .. yg0 + Ly - 1 of the sample (K5C: the rows of one CTA of the cluster; else yg0 = 0);
// carry = h(0, yg0 - 1), or h(0,0) when yg0 = 0.
template <int NT>
__device__ __forceinline__ void row_sums_onchip(const uint32_t* EX, const uint32_t* OX, const uint32_t* EY, int RH, int half, int Lx,
                                                int Ly, int yg0, int carry, const uint32_t* lut, int* scan /* [NT / 32] shared */,
                                                long long& s1, long long& s2) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int y0 = 0; y0 < Ly; y0 += NT) {   // block-uniform trip count
    const int y = y0 + (int)threadIdx.x;
    const bool live = y < Ly;
    const int row = (live ? (half ? (y >> 1) + (y & 1) * half : y) : 0) * RH;
    const int d = (live && yg0 + y > 0) ? 2 * (int)(EY[row] & 1u) - 1 : 0;  // h(0,y) - h(0,y-1)
    int incl = d;
#pragma unroll
    for (int k = 1; k < 32; k <<= 1) {
      const int v = __shfl_up_sync(0xFFFFFFFFu, incl, k);
      if (lane >= k) incl += v;
    }
    __syncthreads();
    if (lane == 31) scan[warp] = incl;
    __syncthreads();
    int add = 0, total = 0;
#pragma unroll
    for (int k = 0; k < NT / 32; ++k) {
      const int t = scan[k];
      if (k < warp) add += t;
      total += t;
    }
    if (live) {
      const long long B = (long long)(carry + add + incl) - (2 * (int)(EX[row] & 1u) - 1);  // height before site (0, y)
      long long S1, S2;  // of the row, relative to B
      row_relative_sums(EX + row, OX + row, RH, lut, S1, S2);
      s1 += (long long)Lx * B + S1;
      s2 += (long long)Lx * B * B + 2 * B * S1 + S2;
    }
    carry += total;
  }
}

// Split barrier of a CTA (one arrival per warp): arrive after a pass's stores, wait before the next pass's loads, with
// work that needs no shared memory (the next pass's Philox calls) in between.
__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.shared::cta.b64 st, [%0];\n}" ::"r"(bar) : "memory");
}
// keep: values that must have been computed BEFORE the wait (the compiler may not sink them past it)
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, const Planes2& keep) {
  asm volatile(
      "{\n.reg .pred p;\n"
      "K5_WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra K5_WAIT_%=;\n}" ::"r"(bar),
      "r"(parity), "r"(keep.v0.x), "r"(keep.v0.y), "r"(keep.v0.z), "r"(keep.v0.w), "r"(keep.v1.x), "r"(keep.v1.y), "r"(keep.v1.z),
      "r"(keep.v1.w)
      : "memory");
}

// K5S: a whole sample on chip.  A pass is the sweep on shared memory followed by ONE __syncthreads (a pass reads only
// bits no other thread of the pass touches, so nothing else orders it); colour offsets are drawn in the kernel 16 MCS at a
// time (one Philox call per lane + ballot); records are taken from shared memory.
constexpr int kK5SThreads = 512;

// PIPE (fast path with two-plane thresholds and at most one supergroup per thread and row parity): the planes of the
// next sweep are drawn one sweep ahead, and the CTA barrier after a pass is split (mbarrier) around that draw.
template <bool ROWALIGNED, bool TWO, bool RIW, bool PIPE>
__device__ __forceinline__ void onchip_body(const Kpz2dDev& D, const Kpz2dRun& A) {
  extern __shared__ __align__(16) uint32_t k5s_smem[];
  __shared__ long long red[2 * (kK5SThreads / 32)];
  __shared__ uint32_t lut[256];   // byte table of the heights (height_lut.cuh), for the records
  __shared__ int scan[kK5SThreads / 32];
  if (threadIdx.x < 256) lut[threadIdx.x] = height_lut_entry((int)threadIdx.x);
  const Shape2d sh = shape2d(D);
  const int s = blockIdx.x;
  const int RH = sh.RH, Ly = sh.Ly;
  const int half = ROWALIGNED ? Ly / 2 : 0;  // fast path: rows kept by parity, row y in slot (y >> 1) + (y & 1) * half
  const int plane = Ly * RH;
  uint32_t* EX = k5s_smem;
  uint32_t* OX = EX + plane;
  uint32_t* EY = OX + plane;
  uint32_t* OY = EY + plane;
  const size_t base = (size_t)s * plane;
  for (int i = threadIdx.x; i < plane; i += kK5SThreads) {
    const int y = i / RH, k = i - y * RH, j = (half ? (y >> 1) + (y & 1) * half : y) * RH + k;
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
  const int sgr = RH / 4, nh = sh.n_sg / 2;  // fast path: supergroups per row; per row parity
  // PIPE: this thread's supergroup of each row parity, fixed for the whole run
  __shared__ unsigned long long mbar_word;
  const uint32_t mbar = smem_addr(&mbar_word);
  uint32_t phase = 0;
  const bool pl_live = nh >= kK5SThreads || (int)threadIdx.x < nh;  // a constant when every thread holds a supergroup
  const int pl_i = pl_live ? (int)threadIdx.x : 0, pl_rr = pl_i / sgr, pl_kq = pl_i - pl_rr * sgr;
  const uint32_t pl_G0 = (uint32_t)(2 * pl_rr * sgr + pl_kq), pl_G1 = pl_G0 + (uint32_t)sgr;
  Planes2 pl_R;
  if constexpr (PIPE) {
    if (threadIdx.x == 0) mbar_init(mbar, kK5SThreads / 32);
    __syncthreads();
    pl_R = draw_two(D.keys, pl_G0, gs, (uint32_t)A.t0, (uint32_t)((unsigned long long)A.t0 >> 32), 0u);
  }
  for (long long m = A.t0; m < A.t0 + A.n_mcs; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    for (int ps = 0; ps < 2; ++ps) {
      const uint32_t o = D.offset_mode ? (uint32_t)ps : ((offbits >> (2 * ((int)m & 15) + ps)) & 1u);
      if constexpr (PIPE) {
        const int P0e = pl_rr * RH + 4 * pl_kq, P0o = P0e + half * RH;  // own row: even rows first, then odd rows
        const int P1o = (pl_rr + 1 == half ? 0 : pl_rr + 1) * RH + 4 * pl_kq;  // row y + 1 of an odd row: the next even row
        const int nxw = pl_kq + 1 == sgr ? 0 : 4 * (pl_kq + 1);
        // even rows (colour o), with the planes drawn one sweep ago; then draw those of the odd rows
        if (o)
          sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0e, P0o, pl_rr * RH + nxw, pl_kq, sgr, pl_G0, pl_live, r, D.keys, gs, tlo, thi,
                                            (uint32_t)ps, &pl_R);
        else
          sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0e, P0o, pl_rr * RH + nxw, pl_kq, sgr, pl_G0, pl_live, r, D.keys, gs, tlo, thi,
                                            (uint32_t)ps, &pl_R);
        pl_R = draw_two(D.keys, pl_G1, gs, tlo, thi, (uint32_t)ps);
        if (o)
          sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0o, P1o, (pl_rr + half) * RH + nxw, pl_kq, sgr, pl_G1, pl_live, r, D.keys, gs,
                                            tlo, thi, (uint32_t)ps, &pl_R);
        else
          sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0o, P1o, (pl_rr + half) * RH + nxw, pl_kq, sgr, pl_G1, pl_live, r, D.keys, gs,
                                            tlo, thi, (uint32_t)ps, &pl_R);
        __syncwarp();
        if (lane == 0) mbar_arrive(mbar);
        {  // the first sweep of the next pass, drawn while the other warps finish this one
          const long long mn = ps ? m + 1 : m;
          pl_R = draw_two(D.keys, pl_G0, gs, (uint32_t)mn, (uint32_t)((unsigned long long)mn >> 32), (uint32_t)(ps ^ 1));
        }
        mbar_wait(mbar, phase, pl_R);
        phase ^= 1u;
        continue;
      }
      if constexpr (ROWALIGNED) {
        for (int h = 0; h < 2; ++h) {  // even rows, then odd rows: one colour for the whole CTA
          const bool c1 = (((uint32_t)h + o) & 1u) != 0u;
          for (int i0 = 0; i0 < nh; i0 += kK5SThreads) {  // block-uniform trip count: every warp stays whole
            const int i = i0 + (int)threadIdx.x;
            const bool live = i < nh;
            const int ii = live ? i : 0;
            const int rr = ii / sgr, kq = ii - rr * sgr;
            const int s0 = rr + h * half, s1 = h ? (rr + 1 == half ? 0 : rr + 1) : rr + half;
            const int P0 = s0 * RH + 4 * kq, P1 = s1 * RH + 4 * kq, NX = s0 * RH + (kq + 1 == sgr ? 0 : 4 * (kq + 1));
            const uint32_t G = (uint32_t)((2 * rr + h) * sgr + kq);
            if (c1)
              sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0, P1, NX, kq, sgr, G, live, r, D.keys, gs, tlo, thi, (uint32_t)ps);
            else
              sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0, P1, NX, kq, sgr, G, live, r, D.keys, gs, tlo, thi, (uint32_t)ps);
          }
        }
      } else {
        for (int G0 = 0; G0 < sh.n_sg; G0 += kK5SThreads) {
          const int G = G0 + (int)threadIdx.x;
          sweep_ragged_supergroup<TWO>(EX, OX, EY, OY, RH, Ly, sh.n_ew, G < sh.n_sg ? G : 0, G < sh.n_sg, o, r, D.keys, gs, tlo, thi,
                                       (uint32_t)ps);
        }
      }
      __syncthreads();  // the next pass reads what this one flipped
    }
    const long long t = m + 1;
    if (t == next_rec) {  // block-uniform
      long long s1 = 0, s2 = 0;
      row_sums_onchip<kK5SThreads>(EX, OX, EY, RH, half, sh.Lx, Ly, 0, 2 * (int)(EX[0] & 1u) - 1, lut, scan, s1, s2);  // row 0 = slot 0
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
  for (int i = threadIdx.x; i < plane; i += kK5SThreads) {
    const int y = i / RH, k = i - y * RH, j = (half ? (y >> 1) + (y & 1) * half : y) * RH + k;
    D.EX[base + i] = EX[j];
    D.OX[base + i] = OX[j];
    D.EY[base + i] = EY[j];
    D.OY[base + i] = OY[j];
  }
}

// mbarrier operations at cluster scope (K5C neighbour synchronisation): a CTA's barrier also takes arrivals from the
// two neighbouring CTAs of the cluster, sent through its shared::cluster address.
__device__ __forceinline__ void mbar_init_cluster(uint32_t bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_arrive_rel_cluster(uint32_t bar) {
  asm volatile("{\n.reg .b64 st;\nmbarrier.arrive.release.cluster.shared::cta.b64 st, [%0];\n}" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_remote(uint32_t cluster_bar) {
  asm volatile("mbarrier.arrive.release.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_bar) : "memory");
}
__device__ __forceinline__ void mbar_wait_acq_cluster(uint32_t bar, uint32_t parity) {
  asm volatile(
      "{\n.reg .pred p;\n"
      "K5C_WAIT_%=:\n"
      "mbarrier.try_wait.parity.acquire.cluster.shared::cta.b64 p, [%0], %1;\n"
      "@!p bra K5C_WAIT_%=;\n}" ::"r"(bar),
      "r"(parity)
      : "memory");
}

// K5C: a sample spread over a thread-block cluster of CS CTAs (lattices beyond the shared memory of one SM, e.g.
// 1024 x 1024 = 256 KiB of slopes; also: more, smaller CTAs balance better over the 148 SMs).  CTA q holds rows
// q Ly/CS .. (q + 1) Ly/CS - 1 in its own shared memory, by parity as K5S does; the only words of another CTA a sweep
// touches are the first even row of CTA q + 1 (row y + 1 of this CTA's last odd row), read and written through
// distributed shared memory.  Synchronisation after a colour pass, split (arrive ... wait) around the Philox calls of the
// next pass: NBR = false (the default: measured faster): one barrier.cluster; NBR = true ("K5J_NBR=1"): the CTAs
// synchronise with their two NEIGHBOURS only - CTA q
// may start pass k + 1 when its own warps, the warps of CTA q - 1 that hold that CTA's last odd row (they write q's row
// 0) and the warps of CTA q + 1 that hold its row 0 (q's last odd row reads it) have finished pass k.  That is an
// mbarrier per CTA with NW + n_edge + n_row0 arrivals, the foreign ones sent through distributed shared memory; two
// barriers alternate, since a neighbour may run one pass ahead (never two: its own barrier waits for this CTA's warps).
// One supergroup per thread and row parity (NT >= Ly/CS/2 * Lx/256); run-time specialised only.
template <bool TWO, bool RIW, int CS, int NT, bool NBR>
__device__ __forceinline__ void cluster_body(const Kpz2dDev& D, const Kpz2dRun& A) {
  extern __shared__ __align__(16) uint32_t k5s_smem[];
  __shared__ long long red[2 * (NT / 32)];
  __shared__ uint32_t lut[256];
  __shared__ int scan[NT / 32];
  __shared__ int col0[2];  // [0]: sum over this CTA's rows of h(0,y) - h(0,y-1); [1]: h(0,0) (CTA 0)
  for (int i = threadIdx.x; i < 256; i += NT) lut[i] = height_lut_entry(i);
  const Shape2d sh = shape2d(D);
  const uint32_t q = cluster_ctarank();
  const int s = blockIdx.x / CS;
  const int RH = sh.RH, LyC = sh.Ly / CS, half = LyC / 2, plane = LyC * RH, yg0 = (int)q * LyC;
  uint32_t* EX = k5s_smem;
  uint32_t* OX = EX + plane;
  uint32_t* EY = OX + plane;
  uint32_t* OY = EY + plane;
  const size_t base = (size_t)s * sh.Ly * RH + (size_t)q * plane;  // this CTA's rows in the workspace
  for (int i = threadIdx.x; i < plane; i += NT) {
    const int y = i / RH, k = i - y * RH, j = ((y >> 1) + (y & 1) * half) * RH + k;
    EX[j] = D.EX[base + i];
    OX[j] = D.OX[base + i];
    EY[j] = D.EY[base + i];
    OY[j] = D.OY[base + i];
  }
  cluster_arrive();  // every CTA of the cluster holds its rows before a neighbour reaches into them
  cluster_wait();
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
  // this thread's supergroup of each row parity, fixed for the whole run
  const int sgr = RH / 4, nh = half * sgr;
  const bool live = nh >= NT || (int)threadIdx.x < nh;
  const int ti = live ? (int)threadIdx.x : 0, rr = ti / sgr, kq = ti - rr * sgr;
  const uint32_t G0 = (uint32_t)((yg0 + 2 * rr) * sgr + kq), G1 = G0 + (uint32_t)sgr;
  const int P0e = rr * RH + 4 * kq, P0o = P0e + half * RH, nxw = kq + 1 == sgr ? 0 : 4 * (kq + 1);
  // row y + 1 of an odd row: the next even row - of the next CTA (cyclically) for this CTA's last odd row
  const bool edge = rr + 1 == half;
  const int P1o = (edge ? 0 : rr + 1) * RH + 4 * kq;
  const uint32_t nbr = edge ? (q + 1 == (uint32_t)CS ? 0u : q + 1u) : q;
  const uint32_t xrE = mapa(smem_addr(EY + P1o), nbr), xrO = mapa(smem_addr(OY + P1o), nbr);
  const bool has_edge = __any_sync(0xFFFFFFFFu, live && edge);      // this warp holds (part of) the CTA's last odd row
  const bool has_row0 = __any_sync(0xFFFFFFFFu, live && rr == 0);    // ... of the CTA's first even row
  const bool warp_edge = has_edge || K5J_XRALL;
  __shared__ unsigned long long nbar[2];
  const uint32_t bar0 = smem_addr(&nbar[0]), bar1 = smem_addr(&nbar[1]);
  const uint32_t q_next = q + 1 == (uint32_t)CS ? 0u : q + 1u, q_prev = q == 0 ? (uint32_t)CS - 1u : q - 1u;
  const uint32_t nx0 = mapa(bar0, q_next), nx1 = mapa(bar1, q_next), pv0 = mapa(bar0, q_prev), pv1 = mapa(bar1, q_prev);
  uint32_t npass = 0;  // colour passes done by this launch
  if constexpr (NBR) {
    if (threadIdx.x == 0) {
      const int a = (half - 1) * sgr, b = half * sgr - 1;  // threads of the last odd row; row 0: threads 0 .. sgr - 1
      const uint32_t count = (uint32_t)(NT / 32 + (b / 32 - a / 32 + 1) + (sgr + 31) / 32);
      mbar_init_cluster(bar0, count);
      mbar_init_cluster(bar1, count);
      mbar_fence_init();
    }
    cluster_arrive();  // the barriers exist before a neighbour arrives on them
    cluster_wait();
  }
  Planes2 R;
  const Planes2* pre = TWO ? &R : nullptr;
  if constexpr (TWO) R = draw_two(D.keys, G0, gs, (uint32_t)A.t0, (uint32_t)((unsigned long long)A.t0 >> 32), 0u);
  for (long long m = A.t0; m < A.t0 + A.n_mcs; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    for (int ps = 0; ps < 2; ++ps) {
      const uint32_t o = D.offset_mode ? (uint32_t)ps : ((offbits >> (2 * ((int)m & 15) + ps)) & 1u);
      if (o)  // even rows: colour o
        sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0e, P0o, rr * RH + nxw, kq, sgr, G0, live, r, D.keys, gs, tlo, thi,
                                          (uint32_t)ps, pre);
      else
        sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0e, P0o, rr * RH + nxw, kq, sgr, G0, live, r, D.keys, gs, tlo, thi,
                                          (uint32_t)ps, pre);
      if constexpr (TWO) R = draw_two(D.keys, G1, gs, tlo, thi, (uint32_t)ps);
      // odd rows: colour 1 - o; only the warp that holds the CTA's last odd row goes through shared::cluster addresses
      if (warp_edge) {
        if (o)
          sweep_row_supergroup<TWO, 0, RIW, true>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs,
                                                  tlo, thi, (uint32_t)ps, pre, xrE);
        else
          sweep_row_supergroup<TWO, 1, RIW, true>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs,
                                                  tlo, thi, (uint32_t)ps, pre, xrO);
      } else {
        if (o)
          sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs, tlo,
                                            thi, (uint32_t)ps, pre);
        else
          sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs, tlo,
                                            thi, (uint32_t)ps, pre);
      }
      const bool odd_pass = (npass & 1u) != 0u;
      if constexpr (NBR) {
        __syncwarp();
        if (lane == 0) {
          mbar_arrive_rel_cluster(odd_pass ? bar1 : bar0);
          if (has_edge) mbar_arrive_remote(odd_pass ? nx1 : nx0);
          if (has_row0) mbar_arrive_remote(odd_pass ? pv1 : pv0);
        }
      } else {
        cluster_arrive();
      }
      if constexpr (TWO) {  // the first sweep of the next pass, drawn while the other CTAs finish this one
        const long long mn = ps ? m + 1 : m;
        R = draw_two(D.keys, G0, gs, (uint32_t)mn, (uint32_t)((unsigned long long)mn >> 32), (uint32_t)(ps ^ 1));
        asm volatile("" ::"r"(R.v0.x), "r"(R.v0.y), "r"(R.v0.z), "r"(R.v0.w), "r"(R.v1.x), "r"(R.v1.y), "r"(R.v1.z), "r"(R.v1.w));
      }
      if constexpr (NBR)
        mbar_wait_acq_cluster(odd_pass ? bar1 : bar0, (npass >> 1) & 1u);
      else
        cluster_wait();
      ++npass;
    }
    const long long t = m + 1;
    if (t == next_rec) {  // cluster-uniform
      int d = 0;  // column 0 of sy over this CTA's rows
      for (int y = threadIdx.x; y < LyC; y += NT)
        if (yg0 + y > 0) d += 2 * (int)(EY[((y >> 1) + (y & 1) * half) * RH] & 1u) - 1;
#pragma unroll
      for (int k = 16; k >= 1; k >>= 1) d += __shfl_xor_sync(0xFFFFFFFFu, d, k);
      if (lane == 0) scan[threadIdx.x >> 5] = d;
      __syncthreads();
      if (threadIdx.x == 0) {
        int tot = 0;
        for (int k = 0; k < NT / 32; ++k) tot += scan[k];
        col0[0] = tot;
        col0[1] = 2 * (int)(EX[0] & 1u) - 1;  // meaningful in CTA 0: its slot 0 is row 0 of the sample
      }
      cluster_arrive();
      cluster_wait();
      int carry = ld_cluster_s32(mapa(smem_addr(&col0[1]), 0u));  // h(0,0)
      for (uint32_t k = 0; k < q; ++k) carry += ld_cluster_s32(mapa(smem_addr(&col0[0]), k));
      long long s1 = 0, s2 = 0;
      row_sums_onchip<NT>(EX, OX, EY, RH, half, sh.Lx, LyC, yg0, carry, lut, scan, s1, s2);
      block_sum2<NT / 32>(s1, s2, red);
      if (threadIdx.x == 0) {  // the host cleared the records of this run: exact two's-complement wrap-around addition
        atomicAdd((unsigned long long*)A.rec_h + (size_t)ri * D.S + s, (unsigned long long)s1);
        atomicAdd((unsigned long long*)A.rec_h2 + (size_t)ri * D.S + s, (unsigned long long)s2);
      }
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
    if (D.offset_mode == 0 && ((int)t & 15) == 0) draw_offsets(t);
  }
  for (int i = threadIdx.x; i < plane; i += NT) {
    const int y = i / RH, k = i - y * RH, j = ((y >> 1) + (y & 1) * half) * RH + k;
    D.EX[base + i] = EX[j];
    D.OX[base + i] = OX[j];
    D.EY[base + i] = EY[j];
    D.OY[base + i] = OY[j];
  }
  cluster_arrive();  // no CTA leaves while a neighbour may still read its col0
  cluster_wait();
}

// K5C, two samples per cluster ("K5J_DUAL"): every CTA holds its rows of TWO samples and sweeps them alternately - A's
// pass k, B's pass k, A's pass k + 1, ... - so the cluster barrier that publishes a pass of one sample completes while
// the CTA sweeps the other sample: sweep(p); [wait for sweep p - 1's barrier]; arrive for sweep p; sweep(p + 1) ...
// The last cluster of an odd ensemble holds one sample and waits before every sweep.  Same rows, addresses and
// distributed-shared-memory accesses as cluster_body; the planes are drawn inside the sweep.
template <bool TWO, bool RIW, int CS, int NT>
__device__ __forceinline__ void cluster_body_dual(const Kpz2dDev& D, const Kpz2dRun& A) {
  extern __shared__ __align__(16) uint32_t k5s_smem[];
  __shared__ long long red[2 * (NT / 32)];
  __shared__ uint32_t lut[256];
  __shared__ int scan[NT / 32];
  __shared__ int col0[2];
  for (int i = threadIdx.x; i < 256; i += NT) lut[i] = height_lut_entry(i);
  const Shape2d sh = shape2d(D);
  const uint32_t q = cluster_ctarank();
  const int s0 = (int)(blockIdx.x / CS) * 2, ns = D.S - s0 < 2 ? D.S - s0 : 2;
  const int RH = sh.RH, LyC = sh.Ly / CS, half = LyC / 2, plane = LyC * RH, yg0 = (int)q * LyC;
  const int set = 4 * plane;  // words of one sample's four planes: EX, OX, EY, OY at 0, plane, 2 plane, 3 plane
  for (int j = 0; j < ns; ++j) {
    const size_t base = (size_t)(s0 + j) * sh.Ly * RH + (size_t)q * plane;
    uint32_t* P = k5s_smem + j * set;
    for (int i = threadIdx.x; i < plane; i += NT) {
      const int y = i / RH, k = i - y * RH, w = ((y >> 1) + (y & 1) * half) * RH + k;
      P[w] = D.EX[base + i];
      P[plane + w] = D.OX[base + i];
      P[2 * plane + w] = D.EY[base + i];
      P[3 * plane + w] = D.OY[base + i];
    }
  }
  cluster_arrive();
  cluster_wait();
  const int lane = threadIdx.x & 31;
  const Rates2d r = make_rates2d(D);
  int ri = A.rec_begin;
  long long next_rec = ri < A.nt ? A.rec_t[ri] : -1;
  uint32_t offbits[2] = {0u, 0u};
  auto draw_offsets = [&](long long m) {
    for (int j = 0; j < ns; ++j) {
      const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
      const uint4 w = philox4x32_10(0u, (uint32_t)(D.first_sample + s0 + j), (uint32_t)mb,
                                    ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), D.keys);
      offbits[j] = __ballot_sync(0xFFFFFFFFu, w.x & 1u);
    }
  };
  if (D.offset_mode == 0) draw_offsets(A.t0);
  const int sgr = RH / 4, nh = half * sgr;
  const bool live = nh >= NT || (int)threadIdx.x < nh;
  const int ti = live ? (int)threadIdx.x : 0, rr = ti / sgr, kq = ti - rr * sgr;
  const uint32_t G0 = (uint32_t)((yg0 + 2 * rr) * sgr + kq), G1 = G0 + (uint32_t)sgr;
  const int P0e = rr * RH + 4 * kq, P0o = P0e + half * RH, nxw = kq + 1 == sgr ? 0 : 4 * (kq + 1);
  const bool edge = rr + 1 == half;
  const int P1o = (edge ? 0 : rr + 1) * RH + 4 * kq;
  const uint32_t nbr = edge ? (q + 1 == (uint32_t)CS ? 0u : q + 1u) : q;
  const bool warp_edge = __any_sync(0xFFFFFFFFu, live && edge);
  bool pending = false;  // an arrival on the cluster barrier that has not been waited for, made after a sweep of sample pend_j
  int pend_j = 0;
  auto settle = [&]() {
    if (pending) cluster_wait();
    pending = false;
  };
  auto sweep = [&](int j, uint32_t tlo, uint32_t thi, uint32_t ps, uint32_t o) {
    uint32_t* EX = k5s_smem + j * set;
    uint32_t* OX = EX + plane;
    uint32_t* EY = OX + plane;
    uint32_t* OY = EY + plane;
    const uint32_t gs = (uint32_t)(D.first_sample + s0 + j);
    if (o)
      sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0e, P0o, rr * RH + nxw, kq, sgr, G0, live, r, D.keys, gs, tlo, thi, ps);
    else
      sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0e, P0o, rr * RH + nxw, kq, sgr, G0, live, r, D.keys, gs, tlo, thi, ps);
    if (warp_edge) {
      if (o)
        sweep_row_supergroup<TWO, 0, RIW, true>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs,
                                                tlo, thi, ps, nullptr, mapa(smem_addr(EY + P1o), nbr));
      else
        sweep_row_supergroup<TWO, 1, RIW, true>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs,
                                                tlo, thi, ps, nullptr, mapa(smem_addr(OY + P1o), nbr));
    } else {
      if (o)
        sweep_row_supergroup<TWO, 0, RIW>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs, tlo, thi, ps);
      else
        sweep_row_supergroup<TWO, 1, RIW>(EX, OX, EY, OY, P0o, P1o, (rr + half) * RH + nxw, kq, sgr, G1, live, r, D.keys, gs, tlo, thi, ps);
    }
  };
  for (long long m = A.t0; m < A.t0 + A.n_mcs; ++m) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    for (int ps = 0; ps < 2; ++ps) {
      for (int j = 0; j < ns; ++j) {
        if (pending && pend_j == j) settle();  // this sample's previous pass must be published (one-sample cluster only)
        const uint32_t o = D.offset_mode ? (uint32_t)ps : ((offbits[j] >> (2 * ((int)m & 15) + ps)) & 1u);
        sweep(j, tlo, thi, (uint32_t)ps, o);
        settle();  // the other sample's barrier has had this whole sweep to complete
        cluster_arrive();
        pending = true;
        pend_j = j;
      }
    }
    const long long t = m + 1;
    if (t == next_rec) {  // cluster-uniform
      settle();
      for (int j = 0; j < ns; ++j) {
        const uint32_t* EX = k5s_smem + j * set;
        const uint32_t* OX = EX + plane;
        const uint32_t* EY = OX + plane;
        int d = 0;
        for (int y = threadIdx.x; y < LyC; y += NT)
          if (yg0 + y > 0) d += 2 * (int)(EY[((y >> 1) + (y & 1) * half) * RH] & 1u) - 1;
#pragma unroll
        for (int k = 16; k >= 1; k >>= 1) d += __shfl_xor_sync(0xFFFFFFFFu, d, k);
        __syncthreads();  // scan / col0 of the previous sample have been read
        if (lane == 0) scan[threadIdx.x >> 5] = d;
        __syncthreads();
        if (threadIdx.x == 0) {
          int tot = 0;
          for (int k = 0; k < NT / 32; ++k) tot += scan[k];
          col0[0] = tot;
          col0[1] = 2 * (int)(EX[0] & 1u) - 1;
        }
        cluster_arrive();
        cluster_wait();
        int carry = ld_cluster_s32(mapa(smem_addr(&col0[1]), 0u));
        for (uint32_t k = 0; k < q; ++k) carry += ld_cluster_s32(mapa(smem_addr(&col0[0]), k));
        cluster_arrive();  // every CTA has read col0 before it is written for the next sample
        cluster_wait();
        long long s1 = 0, s2 = 0;
        row_sums_onchip<NT>(EX, OX, EY, RH, half, sh.Lx, LyC, yg0, carry, lut, scan, s1, s2);
        block_sum2<NT / 32>(s1, s2, red);
        if (threadIdx.x == 0) {
          atomicAdd((unsigned long long*)A.rec_h + (size_t)ri * D.S + s0 + j, (unsigned long long)s1);
          atomicAdd((unsigned long long*)A.rec_h2 + (size_t)ri * D.S + s0 + j, (unsigned long long)s2);
        }
      }
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
    if (D.offset_mode == 0 && ((int)t & 15) == 0) draw_offsets(t);
  }
  settle();
  for (int j = 0; j < ns; ++j) {
    const size_t base = (size_t)(s0 + j) * sh.Ly * RH + (size_t)q * plane;
    const uint32_t* P = k5s_smem + j * set;
    for (int i = threadIdx.x; i < plane; i += NT) {
      const int y = i / RH, k = i - y * RH, w = ((y >> 1) + (y & 1) * half) * RH + k;
      D.EX[base + i] = P[w];
      D.OX[base + i] = P[plane + w];
      D.EY[base + i] = P[2 * plane + w];
      D.OY[base + i] = P[3 * plane + w];
    }
  }
  cluster_arrive();
  cluster_wait();
}

#ifdef K5J_LX
// ---- entry points of the run-time specialised build (NVRTC; csrc/jit.cu) -----------------------------------------
constexpr bool kJRowAligned = (K5J_LX % 256) == 0;
constexpr int kJSgr = K5J_LX / 256;                   // supergroups per row (fast path)
constexpr int kJNh = K5J_LX / 256 * K5J_LY / 2;       // supergroups per row parity
constexpr bool kJRiw = kJRowAligned && kJSgr <= 32 && (32 % (kJSgr > 0 ? kJSgr : 1)) == 0 && (kJNh % 32) == 0 && K5J_RIW;
constexpr bool kJPipe = kJRowAligned && (K5J_TWO != 0) && kJNh <= kK5SThreads && K5J_PIPE;

// K5J_ENTRY: the one entry point this compilation is for (1 K5S, 2 K5C, 3 K5) - the others are left out, which
// shortens the NVRTC run; 0 or undefined: all of them.
#ifndef K5J_ENTRY
#define K5J_ENTRY 0
#endif
#if K5J_ENTRY == 0 || K5J_ENTRY == 1
extern "C" __global__ void __launch_bounds__(kK5SThreads, K5J_MINB)
    kpz2d_k5s_jit(const __grid_constant__ Kpz2dDev D, const __grid_constant__ Kpz2dRun A) {
  onchip_body<kJRowAligned, K5J_TWO != 0, kJRiw, kJPipe>(D, A);
}
#endif
#if K5J_CS > 1 && (K5J_ENTRY == 0 || K5J_ENTRY == 2)
constexpr int kJNhC = K5J_LX / 256 * (K5J_LY / K5J_CS) / 2;  // supergroups per row parity and CTA
constexpr bool kJRiwC = kJRowAligned && kJSgr <= 32 && (32 % (kJSgr > 0 ? kJSgr : 1)) == 0 && (kJNhC % 32) == 0 && K5J_RIW;
static_assert(kJRowAligned && (K5J_LY % (2 * K5J_CS)) == 0 && kJNhC <= K5J_THREADS, "K5C: shape the host must not ask for");
extern "C" __global__ void __cluster_dims__(K5J_CS, 1, 1) __launch_bounds__(K5J_THREADS, K5J_MINB)
    kpz2d_k5c_jit(const __grid_constant__ Kpz2dDev D, const __grid_constant__ Kpz2dRun A) {
  if constexpr (K5J_DUAL != 0)
    cluster_body_dual<K5J_TWO != 0, kJRiwC, K5J_CS, K5J_THREADS>(D, A);
  else
    cluster_body<K5J_TWO != 0, kJRiwC, K5J_CS, K5J_THREADS, K5J_NBR != 0>(D, A);
}
#endif
#if K5J_ENTRY == 0 || K5J_ENTRY == 3
extern "C" __global__ void __launch_bounds__(128)
    kpz2d_k5_pass_jit(const __grid_constant__ Kpz2dDev D, const unsigned char* __restrict__ off, long long m, int ps) {
  pass_body<kJRowAligned, K5J_TWO != 0, K5J_PDL != 0>(D, off, m, ps);
}
#endif
#else
// ---- the generic kernels of the library build --------------------------------------------------------------------
template <bool ROWALIGNED, bool TWO>
__global__ void __launch_bounds__(128) k2d_pass(const __grid_constant__ Kpz2dDev D, const unsigned char* __restrict__ off,
                                                long long m, int ps) {
  pass_body<ROWALIGNED, TWO>(D, off, m, ps);
}
template <bool ROWALIGNED, bool TWO>
__global__ void __launch_bounds__(kK5SThreads, 2) k2d_onchip(const __grid_constant__ Kpz2dDev D, const __grid_constant__ Kpz2dRun A) {
  onchip_body<ROWALIGNED, TWO, false, false>(D, A);
}
#endif

}  // namespace kpz
