// k4_lanes_jit.cuh — K4 v2: two-lane opposite-direction lattice gas with turning points, specialised at run time
// (NVRTC, jit.cu) on the ring size and the four thresholds (north_star (4); PAPER.md:253-275;
// DESIGN §R12-R17).  One CTA per sample, persistent over the whole lanes_run.
//
// Layout on chip: NATURAL bit order (bit i&31 of word i>>5 = site i), because the dominant random streams of this
// model are per SITE (lane changes, turning points): one Philox call is one bit-plane of 128 consecutive sites = 4
// natural words.  A thread owns exactly one such supergroup: 4 words of lane A, lane B and the turning-point mask
// in registers (L=16384: 128 threads = 4 warps per sample, 1024 warps on the chip for config 5).
//   * in-lane hops are word-local bit logic: with sh = (X >> 1 | next word << 31), lane A (right) hops where
//     X & ~sh & pairmask(o), lane B (left) where ~X & sh & pairmask(o); offset 1 needs bit 0 of the next thread's
//     word 0 and sends one carry bit back (ring closure = wrap-around of that exchange);
//   * lane changes (K4J_PRE = 1, default): whether a site WOULD let a particle change lane in step st of MCS m - "is a
//     turning point and U(SWITCH_st, m, site) < T(omega)" - does not depend on the occupations.  So every warp computes
//     these acceptance masks for its 32 supergroups for a CHUNK of MCS ahead (precompute_chunk) and parks them in shared
//     memory; the sweep itself then only ANDs them with "source occupied, target empty".  This takes the lazy MSB-first
//     comparison - a chain of dependent Philox calls - off the latency-critical, barrier-coupled path of the sweep
//     (measured: with ~1.7 warps per SMSP every dependent trip cost ~400 clk) and turns it into throughput work with
//     full SIMT efficiency: all lanes draw the first K4J_DIRECT planes of their items, items that are still undecided
//     go to a per-warp queue, and every further trip of the warp pops 32 queued (supergroup, MCS, step, plane) entries
//     - whatever items they belong to - draws their planes, and pushes back those still undecided.  No lane ever idles
//     while another waits for a deeper plane.  Candidates are the ~6 turning points of a supergroup (4.0 planes per
//     supergroup and step on average) instead of the ~1.3 live ones (1.8 planes), but the warp draws 5.3 planes per
//     32 supergroups where the SIMT-lazy loop over live sites drew 8.8.  Results are identical: the comparison of one
//     element still runs plane by plane, MSB first.
//     K4J_PRE = 0 keeps the live-site evaluation inside the sweep (K4J_EAGER planes drawn one MCS ahead, resolve_packed);
//   * hop counters by POPC of two merged hop words (hops of one pass sit on one bit parity), occupancy profile at
//     epoch ends by warp-transposed, coalesced red.global.add.
//
// Compile-time configuration (-D, set by lanes_api.cu): K4J_W = L/32, K4J_TPA, K4J_TPB, K4J_TOMEGA, K4J_TTURN
// (thresholds in [0, 2^32]), K4J_OFFSET_MODE, K4J_TW0 and K4J_INDEP (site-wise crossing model), K4J_EAGER,
// K4J_SMAX, K4J_TRIP, K4J_PRE, K4J_CHUNK, K4J_DIRECT, K4J_VPROF.
#pragma once
#include "sweep_types.cuh"

#ifndef K4J_HALOCHECK  // debug: sequence numbers on the shared-memory halo slots (see k1_sweep_jit.cuh, K1J_HALOCHECK)
#define K4J_HALOCHECK 0
#endif
#ifndef K4J_W
#error "k4_lanes_jit.cuh needs K4J_W, K4J_TPA, K4J_TPB, K4J_TOMEGA, K4J_TTURN, K4J_OFFSET_MODE"
#endif
#ifndef K4J_TW0
#define K4J_TW0 0ull  // crossing threshold at unflagged sites: 0 = turning-point model, else §R18
#endif
#ifndef K4J_INDEP
#define K4J_INDEP 0   // 1: the B->A crossings read their own flag set (D.V)
#endif
#ifndef K4J_PRE
#define K4J_PRE 1    // 1: lane-change acceptance masks precomputed per chunk of MCS (see above); 0: evaluated in the sweep
#endif
#ifndef K4J_CHUNK
#define K4J_CHUNK 16  // MCS per precomputed chunk (lanes_api.cu sizes the dynamic shared memory with the same number)
#endif
#ifndef K4J_VPROF
#define K4J_VPROF 6   // occupancy profile: epoch-end snapshots are counted in this many bit-sliced planes in shared memory
#endif                //   and flushed to the per-site counters every 2^K4J_VPROF - 1 snapshots (0: added to them directly)

#ifndef K4J_DIRECT
#define K4J_DIRECT 4  // planes every lane draws for each of its items before undecided items go to the queue
#endif
#ifndef K4J_EAGER
#define K4J_EAGER 6  // K4J_PRE = 0: lane-change planes drawn one MCS ahead
#endif
#ifndef K4J_SMAX
#define K4J_SMAX 1   // packed trips: at most this many consecutive planes per trip (1 = plane by plane; a power of two)
#endif
#ifndef K4J_TRIP
#define K4J_TRIP 2  // planes per trip of the unpacked loop (turning-point redraw, in-lane rates < 1 with K4J_SMAX = 1)
#endif
#if K4J_SMAX != 1 && K4J_SMAX != 2 && K4J_SMAX != 4 && K4J_SMAX != 8 && K4J_SMAX != 16 && K4J_SMAX != 32
#error "K4J_SMAX must be a power of two in [1, 32]"
#endif

namespace kpz {
namespace k4j {

constexpr int W = K4J_W;
constexpr int U = (W + 3) / 4;
constexpr bool SINGLE_WARP = U <= 32;
constexpr bool PARTIAL = (W % 4) != 0;
constexpr int NTHREADS = (U + 31) / 32 * 32;
constexpr int VPROF = (K4J_VPROF > 0 && NTHREADS <= 256) ? K4J_VPROF : 0;  // bit-sliced snapshot counters (see add_profile_v)
// Small rings (the paper's L = 512 ... 2048): U <= 16 supergroups fill only U lanes, so a warp sweeps SPW = 32 / U
// independent samples side by side; offsets and record sums become per-lane values (segments of U lanes).
constexpr int SPW = (!PARTIAL && U <= 16 && (U & (U - 1)) == 0) ? 32 / U : 1;
constexpr uint64_t TPA = K4J_TPA, TPB = K4J_TPB, TOMEGA = K4J_TOMEGA, TTURN = K4J_TTURN;
constexpr uint64_t kOne = 1ull << 32;
constexpr uint32_t FULL = 0xFFFFFFFFu;

__host__ __device__ constexpr int planes_of(uint64_t T) {
  if (T == 0 || T >= kOne) return 0;
  int z = 0;
  while (!((T >> z) & 1ull)) ++z;
  return 32 - z;
}
constexpr uint64_t TW0 = K4J_TW0;
constexpr bool CROSS = TW0 != 0;  // every site can be crossed: two rate classes, chosen by the site's flag
constexpr int NPW = planes_of(TOMEGA) > planes_of(TW0) ? planes_of(TOMEGA) : planes_of(TW0);
constexpr int EAGER = K4J_EAGER < NPW ? K4J_EAGER : NPW;
constexpr int EAGERA = EAGER > 0 ? EAGER : 1;

template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
  return d;
}

// One MSB-first comparison step with plane `pl` of the uniforms (R = that plane's bits): lt = already decided
// U < T, eq = prefix still equal to T's.
template <uint64_t T>
__device__ __forceinline__ void plane_step(uint32_t (&lt)[4], uint32_t (&eq)[4], const uint32_t (&R)[4], int pl) {
  const uint32_t tb = 0u - (((uint32_t)T >> (31 - pl)) & 1u);  // callers: 0 < T < 2^32
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    lt[w] |= eq[w] & tb & ~R[w];
    eq[w] &= ~(R[w] ^ tb);
  }
}

// Finish U < T for the still-undecided elements `eq` of supergroup G of stream c3 (tag | pass | time_hi), starting at
// plane pl0.  K4J_TRIP planes per trip, trips are warp-uniform (a warp leaves when none of its lanes is undecided).
template <uint64_t T>
__device__ __forceinline__ void resolve(uint32_t (&lt)[4], uint32_t (&eq)[4], const PhiloxKeys& K, uint32_t G,
                                        uint32_t gs, uint32_t tlo, uint32_t c3, int pl0) {
  constexpr int NP = planes_of(T);
#pragma unroll 1
  for (int pl = pl0; pl < NP; pl += K4J_TRIP) {
    if (!__any_sync(FULL, (eq[0] | eq[1] | eq[2] | eq[3]) != 0u)) break;
    uint32_t R[K4J_TRIP][4];
#pragma unroll
    for (int t = 0; t < K4J_TRIP; ++t) {  // independent calls: their rounds interleave
      if (pl + t < NP) {                   // (warp-uniform) never draw a plane T does not reach
        const uint4 v = philox4x32_10(G, gs, tlo, c3 | ((uint32_t)(pl + t) << 22), K);
        R[t][0] = v.x; R[t][1] = v.y; R[t][2] = v.z; R[t][3] = v.w;
      } else {
        R[t][0] = R[t][1] = R[t][2] = R[t][3] = 0u;
      }
    }
#pragma unroll
    for (int t = 0; t < K4J_TRIP; ++t)
      if (pl + t < NP) plane_step<T>(lt, eq, R[t], pl + t);
  }
}

// Per-warp exchange area of the packed trips.
struct PackSmem {
  uint4 plane[32];         // plane[j] = the 128 bits lane j drew
  unsigned char owner[32];  // owner[r] = lane of the r-th undecided supergroup of the warp
};

// Finish the comparison for the undecided elements of every lane of the warp, starting at plane pl0 (< NP planes in
// all).  Each trip: n = lanes still undecided.  While n > 16 (or K4J_SMAX = 1) every lane draws the next plane of its
// own supergroup.  Once n <= 32 / s the 32 lanes are dealt out as (undecided supergroup i, plane pl + t), i < 32 / s,
// t < s: lane j draws plane pl + (j / npad) of the supergroup owned by the (j mod npad)-th undecided lane, every lane
// parks its 128 bits in shared memory, and an owner then applies planes pl .. pl + s - 1 IN ORDER - the comparison is
// the plane-by-plane one, only the drawing is spread over the idle lanes.  step(lt, eq, R, pl) is one MSB-first step.
template <class Step>
__device__ __forceinline__ void resolve_packed(uint32_t (&lt)[4], uint32_t (&eq)[4], const PhiloxKeys& K, uint32_t G,
                                               uint32_t gs, uint32_t tlo, uint32_t c3, int pl0, int NP, PackSmem* xs,
                                               Step step) {
  const int lane = threadIdx.x & 31;
  int pl = pl0;
#pragma unroll 1
  while (pl < NP) {  // warp-uniform
    const bool und = (eq[0] | eq[1] | eq[2] | eq[3]) != 0u;
    const uint32_t mask = __ballot_sync(FULL, und);
    if (!mask) break;
    const int n = __popc(mask);
    int lg = 0;  // log2 of the planes of this trip
    if (K4J_SMAX >= 2 && n <= 16) lg = 1;
    if (K4J_SMAX >= 4 && n <= 8) lg = 2;
    if (K4J_SMAX >= 8 && n <= 4) lg = 3;
    if (K4J_SMAX >= 16 && n <= 2) lg = 4;
    if (K4J_SMAX >= 32 && n <= 1) lg = 5;
    if (lg == 0) {
      const uint4 v = philox4x32_10(G, gs, tlo, c3 | ((uint32_t)pl << 22), K);
      const uint32_t R[4] = {v.x, v.y, v.z, v.w};
      step(lt, eq, R, pl);
      pl += 1;
    } else {
      const int npad = 32 >> lg;
      const int rank = __popc(mask & ((1u << lane) - 1u));
      if (und) xs->owner[rank] = (unsigned char)lane;
      __syncwarp();
      const int i = lane & (npad - 1), t = lane >> (5 - lg);
      const int src = i < n ? (int)xs->owner[i] : lane;  // spare lanes redraw a plane of their own: never read
      const uint32_t Gs = __shfl_sync(FULL, G, src), gss = __shfl_sync(FULL, gs, src);
      const int q = pl + t < 32 ? pl + t : 31;
      xs->plane[lane] = philox4x32_10(Gs, gss, tlo, c3 | ((uint32_t)q << 22), K);
      __syncwarp();
      const int mine = rank & (npad - 1);  // decided lanes read somebody's planes: eq = 0 makes the step a no-op
#pragma unroll 1
      for (int tt = 0; tt < (1 << lg); ++tt) {
        if (pl + tt < NP) {  // warp-uniform
          const uint4 v = xs->plane[mine + tt * npad];
          const uint32_t R[4] = {v.x, v.y, v.z, v.w};
          step(lt, eq, R, pl + tt);
        }
      }
      __syncwarp();  // the slots are rewritten by the next trip
      pl += 1 << lg;
    }
  }
}

// [U < T] over the `live` elements of one supergroup, from plane 0.
template <uint64_t T>
__device__ __forceinline__ void lazy_less(uint32_t (&lt)[4], const uint32_t (&live)[4], const PhiloxKeys& K, uint32_t G,
                                          uint32_t gs, uint32_t tlo, uint32_t c3) {
  uint32_t eq[4];
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    lt[w] = (T >= kOne) ? live[w] : 0u;
    eq[w] = (T >= kOne || T == 0) ? 0u : live[w];
  }
  if (T > 0 && T < kOne) resolve<T>(lt, eq, K, G, gs, tlo, c3, 0);
}
// Same through packed trips (every lane of the warp must call it).
template <uint64_t T>
__device__ __forceinline__ void lazy_less_packed(uint32_t (&lt)[4], const uint32_t (&live)[4], const PhiloxKeys& K,
                                                 uint32_t G, uint32_t gs, uint32_t tlo, uint32_t c3, PackSmem* xs) {
  uint32_t eq[4];
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    lt[w] = (T >= kOne) ? live[w] : 0u;
    eq[w] = (T >= kOne || T == 0) ? 0u : live[w];
  }
  if (T > 0 && T < kOne)
    resolve_packed(lt, eq, K, G, gs, tlo, c3, 0, planes_of(T), xs,
                   [](uint32_t (&l)[4], uint32_t (&e)[4], const uint32_t (&R)[4], int pl) { plane_step<T>(l, e, R, pl); });
}

// ---- bit gathers between site order and pair order ------------------------------------------------------------------
__device__ __forceinline__ uint32_t compress_even(uint32_t x) {  // even-position bits -> low 16 bits
  x &= 0x55555555u;
  x = (x | (x >> 1)) & 0x33333333u;
  x = (x | (x >> 2)) & 0x0F0F0F0Fu;
  x = (x | (x >> 4)) & 0x00FF00FFu;
  x = (x | (x >> 8)) & 0x0000FFFFu;
  return x;
}
__device__ __forceinline__ uint32_t spread_even(uint32_t x) {  // low 16 bits -> even positions
  x &= 0x0000FFFFu;
  x = (x | (x << 8)) & 0x00FF00FFu;
  x = (x | (x << 4)) & 0x0F0F0F0Fu;
  x = (x | (x << 2)) & 0x33333333u;
  x = (x | (x << 1)) & 0x55555555u;
  return x;
}

// ---- neighbour exchange: the value held by thread `src` of this sample ---------------------------------------------
// (`parity` counts the exchanges of the CTA; the slot set alternates with it)
#if K4J_HALOCHECK
__device__ unsigned int* g_halo_check;  // = LanesRunArgs.check
#endif
constexpr int HALO_WORDS = (K4J_HALOCHECK ? 4 : 2) * NTHREADS;
__device__ __forceinline__ uint32_t unit_exchange(uint32_t mine, int src, uint32_t* halo, int& parity) {
  if (SINGLE_WARP) {
    return __shfl_sync(FULL, mine, src);
  } else {
    uint32_t* slot = halo + (parity & 1) * NTHREADS;
    slot[threadIdx.x] = mine;
#if K4J_HALOCHECK
    slot[2 * NTHREADS + threadIdx.x] = (uint32_t)parity;
#endif
    __syncthreads();
    const uint32_t v = slot[src];
#if K4J_HALOCHECK
    if (slot[2 * NTHREADS + src] != (uint32_t)parity) atomicAdd(g_halo_check, 1u);
#endif
    parity += 1;
    return v;
  }
}

// Same, reading the values of two threads after one publication (one barrier).
__device__ __forceinline__ void unit_exchange2(uint32_t mine, int src1, int src2, uint32_t& v1, uint32_t& v2,
                                               uint32_t* halo, int& parity) {
  if (SINGLE_WARP) {
    v1 = __shfl_sync(FULL, mine, src1);
    v2 = __shfl_sync(FULL, mine, src2);
  } else {
    uint32_t* slot = halo + (parity & 1) * NTHREADS;
    slot[threadIdx.x] = mine;
#if K4J_HALOCHECK
    slot[2 * NTHREADS + threadIdx.x] = (uint32_t)parity;
#endif
    __syncthreads();
    v1 = slot[src1];
    v2 = slot[src2];
#if K4J_HALOCHECK
    if (slot[2 * NTHREADS + src1] != (uint32_t)parity || slot[2 * NTHREADS + src2] != (uint32_t)parity)
      atomicAdd(g_halo_check, 1u);
#endif
    parity += 1;
  }
}

struct Unit {
  int u;     // supergroup index of this thread within the sample
  int nwn;   // valid words (4; 2 in the last thread of a ragged ring; 0 for an idle lane)
  int nxt, prv;
  uint32_t gs;  // global sample index
};

// In-lane pass of one lane: RIGHT (lane A): (1,0)->(0,1) on pairs (a, a+1); else (lane B) (0,1)->(1,0).
// o = offset of the pass; next0 = bit 0 of the next thread's word 0 (old value; only used when o = 1).
// Returns the carry: 1 if the hop over this thread's last pair flips bit 0 of the next thread (o = 1 only).
template <bool RIGHT, uint64_t TP>
__device__ __forceinline__ uint32_t lane_pass(uint32_t (&X)[4], const Unit& un, uint32_t o, uint32_t next0,
                                              const PhiloxKeys& K, uint32_t tag, uint32_t tlo, uint32_t c3time,
                                              unsigned long long& hops, PackSmem* xs) {
  uint32_t hop[4];
  const uint32_t amask = o ? 0xAAAAAAAAu : 0x55555555u;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    uint32_t nx = (w < 3) ? X[w < 3 ? w + 1 : 3] : next0;
    if (PARTIAL) nx = (w + 1 < un.nwn) ? nx : next0;
    const uint32_t sh = __funnelshift_r(X[w], nx, 1);
    hop[w] = RIGHT ? lop3<0x20>(X[w], sh, amask) : lop3<0x08>(X[w], sh, amask);  // X & ~sh & m : ~X & sh & m
    if (PARTIAL) hop[w] = (w < un.nwn) ? hop[w] : 0u;
  }
  if (TP < kOne) {
    // candidates in PAIR order (in-lane uniforms are per pair): this thread's 64 pairs are words
    // 2(u&1), 2(u&1)+1 of pair supergroup u>>1
    const uint32_t lv0 = compress_even(hop[0] >> o) | (compress_even(hop[1] >> o) << 16);
    const uint32_t lv1 = compress_even(hop[2] >> o) | (compress_even(hop[3] >> o) << 16);
    const bool hi = (un.u & 1) != 0;
    uint32_t live[4] = {hi ? 0u : lv0, hi ? 0u : lv1, hi ? lv0 : 0u, hi ? lv1 : 0u};
    uint32_t acc[4];
    lazy_less_packed<TP>(acc, live, K, (uint32_t)(un.u >> 1), un.gs, tlo, ctr3(tag, 0, 0, 0) | c3time, xs);
    const uint32_t a0 = hi ? acc[2] : acc[0], a1 = hi ? acc[3] : acc[1];
    hop[0] = spread_even(a0) << o;
    hop[1] = spread_even(a0 >> 16) << o;
    hop[2] = spread_even(a1) << o;
    hop[3] = spread_even(a1 >> 16) << o;
  }
  // a hop flips both sites of its pair: hop | hop << 1, the bit shifted out of a word enters the next one
  uint32_t out;
  if (!PARTIAL) {
    X[3] ^= hop[3] | __funnelshift_l(hop[2], hop[3], 1);
    X[2] ^= hop[2] | __funnelshift_l(hop[1], hop[2], 1);
    X[1] ^= hop[1] | __funnelshift_l(hop[0], hop[1], 1);
    X[0] ^= hop[0] | (hop[0] << 1);
    out = hop[3] >> 31;
  } else {
    uint32_t carry = 0;
    out = 0;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      X[w] ^= hop[w] | (hop[w] << 1) | carry;
      carry = hop[w] >> 31;
      if (w + 1 == un.nwn) {  // the carry of the last valid word leaves the thread
        out = carry;
        carry = 0;
      }
    }
  }
  // hops of one pass sit on one bit parity, so two hop words merge into one POPC
  hops += __popc(hop[0] | __funnelshift_l(hop[1], hop[1], 1)) + __popc(hop[2] | __funnelshift_l(hop[3], hop[3], 1));
  return out;
}

// The eager planes of the two lane-change steps of one MCS: r[step][plane][word].
struct Eager {
  uint32_t r[2][EAGERA][4];
};

__device__ __forceinline__ void draw_eager(Eager& E, const PhiloxKeys& K, const Unit& un, long long m) {
  const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
#pragma unroll
  for (int st = 0; st < 2; ++st) {
#pragma unroll
    for (int pl = 0; pl < EAGER; ++pl) {
      const uint4 v = philox4x32_10((uint32_t)un.u, un.gs, tlo,
                                    ctr3(st == 0 ? TAG_SWITCH_AB : TAG_SWITCH_BA, 0, (uint32_t)pl, thi), K);
      E.r[st][pl][0] = v.x;
      E.r[st][pl][1] = v.y;
      E.r[st][pl][2] = v.z;
      E.r[st][pl][3] = v.w;
    }
  }
}

// Two rate classes: elements with flag F compare with T(omega) (bit b1 of this plane), the others with
// T(w_unflagged) (bit b0).
__device__ __forceinline__ void plane_step2(uint32_t (&lt)[4], uint32_t (&eq)[4], const uint32_t (&R)[4],
                                            const uint32_t (&F)[4], uint32_t b1, uint32_t b0) {
  const uint32_t B1 = 0u - b1, B0 = 0u - b0;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint32_t tb = (F[w] & B1) | (~F[w] & B0);
    lt[w] |= eq[w] & tb & ~R[w];
    eq[w] &= ~(R[w] ^ tb);
  }
}
__host__ __device__ constexpr uint32_t tbit(uint64_t T, int pl) { return (uint32_t)((T >> (31 - pl)) & 1ull); }

// ---- precomputed lane-change acceptance (K4J_PRE) ---------------------------------------------------------------------
constexpr int CHUNK = K4J_CHUNK;
constexpr int DIRECT = K4J_DIRECT < NPW ? K4J_DIRECT : NPW;
constexpr int QCAP = 128;  // queue entries per warp (a power of two >= 32 + 64 + 32)
static_assert(CHUNK >= 1 && CHUNK <= 256, "K4J_CHUNK: the chunk index has 8 bits in a queue entry");

// Per-warp shared memory of the precompute.
struct WarpSmem {
  uint4 acc[CHUNK][2][32];  // acc[k][st][lane]: sites of the lane's supergroup that accept a lane change in step st of
                            //   MCS m0 + k (st 0: A->B, 1: B->A) - candidates only (turning points / every site)
  uint4 qeq[QCAP];          // queue of undecided items: their elements whose prefix still equals the threshold's ...
  uint32_t qid[QCAP];       //   ... and lane | k << 5 | st << 13 | next plane << 14
  uint4 flag[2][32];        // site-wise crossing model: the flag words of every lane for step 0 / 1 (rate class per site)
};

__host__ __device__ constexpr uint32_t dyn_tbit(uint64_t T, int pl) {
  return (T > 0 && T < kOne) ? (((uint32_t)T >> (31 - pl)) & 1u) : 0u;
}
// One MSB-first comparison step of a lane-change item with plane pl; F = flag words (rate class per site, CROSS only).
__device__ __forceinline__ void change_step(uint32_t (&lt)[4], uint32_t (&eq)[4], const uint32_t (&R)[4],
                                            const uint32_t (&F)[4], int pl) {
  if constexpr (!CROSS) plane_step<TOMEGA>(lt, eq, R, pl);
  else plane_step2(lt, eq, R, F, dyn_tbit(TOMEGA, pl), dyn_tbit(TW0, pl));
}
// Candidates of one item: lt = accepted whatever U is, eq = needs planes.  F = flags of the step, nwn = valid words.
__device__ __forceinline__ void change_init(uint32_t (&lt)[4], uint32_t (&eq)[4], const uint32_t (&F)[4], int nwn) {
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    if constexpr (!CROSS) {
      lt[w] = (TOMEGA >= kOne) ? F[w] : 0u;
      eq[w] = (TOMEGA > 0 && TOMEGA < kOne) ? F[w] : 0u;
    } else {
      constexpr uint32_t AL1 = TOMEGA >= kOne ? ~0u : 0u, AL0 = TW0 >= kOne ? ~0u : 0u;
      constexpr uint32_t PA1 = (TOMEGA > 0 && TOMEGA < kOne) ? ~0u : 0u, PA0 = (TW0 > 0 && TW0 < kOne) ? ~0u : 0u;
      const uint32_t valid = w < nwn ? FULL : 0u;
      lt[w] = valid & ((F[w] & AL1) | (~F[w] & AL0));
      eq[w] = valid & ((F[w] & PA1) | (~F[w] & PA0));
    }
  }
}

struct Queue {
  uint32_t head, tail;  // warp-uniform
};

// Append the lanes' undecided items (und) to the queue.
__device__ __forceinline__ void queue_push(WarpSmem* ws, Queue& q, bool und, const uint32_t (&eq)[4], uint32_t id) {
  const int lane = threadIdx.x & 31;
  const uint32_t mask = __ballot_sync(FULL, und);
  if (und) {
    const uint32_t j = (q.tail + (uint32_t)__popc(mask & ((1u << lane) - 1u))) & (QCAP - 1);
    ws->qeq[j] = make_uint4(eq[0], eq[1], eq[2], eq[3]);
    ws->qid[j] = id;
  }
  q.tail += (uint32_t)__popc(mask);
}

// One trip of the warp over up to 32 queued entries: each lane draws the next plane of ITS entry (whatever lane, MCS
// and step that entry belongs to), applies it, ORs newly accepted sites into the entry's mask and queues the entry
// again while it is undecided.  Entries are unique per (lane, k, st), so the read-modify-write of acc needs no atomic.
__device__ __forceinline__ void queue_trip(WarpSmem* ws, uint4 (*acc)[2][32], Queue& q, const PhiloxKeys& K, uint32_t G,
                                           uint32_t gs, long long m0) {
  const int lane = threadIdx.x & 31;
  const uint32_t nv = q.tail - q.head < 32u ? q.tail - q.head : 32u;
  const bool valid = (uint32_t)lane < nv;
  const uint32_t j = (q.head + (uint32_t)lane) & (QCAP - 1);
  const uint32_t id = valid ? ws->qid[j] : 0u;
  const uint4 e = ws->qeq[j];
  q.head += nv;
  const int le = (int)(id & 31u), k = (int)((id >> 5) & 255u), st = (int)((id >> 13) & 1u), pl = (int)(id >> 14);
  const uint32_t Gs = __shfl_sync(FULL, G, le), gss = __shfl_sync(FULL, gs, le);
  const unsigned long long mm = (unsigned long long)(m0 + k);
  const uint4 v = philox4x32_10(Gs, gss, (uint32_t)mm,
                                ctr3(st ? TAG_SWITCH_BA : TAG_SWITCH_AB, 0, (uint32_t)pl, (uint32_t)(mm >> 32)), K);
  const uint32_t R[4] = {v.x, v.y, v.z, v.w};
  uint32_t F[4] = {0u, 0u, 0u, 0u};
  if constexpr (CROSS) {
    const uint4 f = ws->flag[st][le];
    F[0] = f.x; F[1] = f.y; F[2] = f.z; F[3] = f.w;
  }
  uint32_t lt[4] = {0u, 0u, 0u, 0u};
  uint32_t eq[4] = {valid ? e.x : 0u, valid ? e.y : 0u, valid ? e.z : 0u, valid ? e.w : 0u};
  change_step(lt, eq, R, F, pl);
  if ((lt[0] | lt[1] | lt[2] | lt[3]) != 0u) {
    uint4 a = acc[k][st][le];
    a.x |= lt[0]; a.y |= lt[1]; a.z |= lt[2]; a.w |= lt[3];
    acc[k][st][le] = a;
  }
  __syncwarp();  // the popped slots may be reused by the pushes below
  queue_push(ws, q, (eq[0] | eq[1] | eq[2] | eq[3]) != 0u && pl + 1 < NPW, eq, id + (1u << 14));
  __syncwarp();
}

// Acceptance masks of this warp's supergroups for MCS m0 .. m0 + n - 1 (n <= CHUNK), both lane-change steps.
// F0 / F1 = the lane's flag words of step 0 / 1 (turning points; u_i / v_i), fixed over the chunk.
__device__ __forceinline__ void precompute_chunk(WarpSmem* ws, uint4 (*acc)[2][32], const PhiloxKeys& K, const Unit& un,
                                                 const uint32_t (&F0)[4], const uint32_t (&F1)[4], long long m0, int n) {
  const int lane = threadIdx.x & 31;
  if constexpr (CROSS) {
    ws->flag[0][lane] = make_uint4(F0[0], F0[1], F0[2], F0[3]);
    ws->flag[1][lane] = make_uint4(F1[0], F1[1], F1[2], F1[3]);
  }
  __syncwarp();
  Queue q{0u, 0u};
#pragma unroll 1
  for (int k = 0; k < n; ++k) {
    const unsigned long long mm = (unsigned long long)(m0 + k);
    const uint32_t tlo = (uint32_t)mm, thi = (uint32_t)(mm >> 32);
    uint32_t lt0[4], eq0[4], lt1[4], eq1[4];
    change_init(lt0, eq0, F0, un.nwn);
    change_init(lt1, eq1, F1, un.nwn);
    if (NPW > 0) {
      uint32_t R0[DIRECT > 0 ? DIRECT : 1][4], R1[DIRECT > 0 ? DIRECT : 1][4];
#pragma unroll
      for (int pl = 0; pl < DIRECT; ++pl) {  // 2 * DIRECT independent calls: their rounds interleave
        const uint4 a = philox4x32_10((uint32_t)un.u, un.gs, tlo, ctr3(TAG_SWITCH_AB, 0, (uint32_t)pl, thi), K);
        const uint4 b = philox4x32_10((uint32_t)un.u, un.gs, tlo, ctr3(TAG_SWITCH_BA, 0, (uint32_t)pl, thi), K);
        R0[pl][0] = a.x; R0[pl][1] = a.y; R0[pl][2] = a.z; R0[pl][3] = a.w;
        R1[pl][0] = b.x; R1[pl][1] = b.y; R1[pl][2] = b.z; R1[pl][3] = b.w;
      }
#pragma unroll
      for (int pl = 0; pl < DIRECT; ++pl) {
        change_step(lt0, eq0, R0[pl], F0, pl);
        change_step(lt1, eq1, R1[pl], F1, pl);
      }
    }
    acc[k][0][lane] = make_uint4(lt0[0], lt0[1], lt0[2], lt0[3]);
    acc[k][1][lane] = make_uint4(lt1[0], lt1[1], lt1[2], lt1[3]);
    __syncwarp();
    const uint32_t id = (uint32_t)lane | ((uint32_t)k << 5) | ((uint32_t)DIRECT << 14);
    queue_push(ws, q, DIRECT < NPW && (eq0[0] | eq0[1] | eq0[2] | eq0[3]) != 0u, eq0, id);
    queue_push(ws, q, DIRECT < NPW && (eq1[0] | eq1[1] | eq1[2] | eq1[3]) != 0u, eq1, id | (1u << 13));
    __syncwarp();
    while (q.tail - q.head >= 32u) queue_trip(ws, acc, q, K, (uint32_t)un.u, un.gs, m0);
  }
  while (q.tail != q.head) queue_trip(ws, acc, q, K, (uint32_t)un.u, un.gs, m0);
  __syncwarp();
}

// Lane changes SRC -> DST where the source is occupied, the target empty and U < T(site) (§R18):
// turning-point model: T = T(omega) at flagged sites F, no crossing elsewhere; site-wise crossing model: T(omega) at
// flagged sites, T(w_unflagged) elsewhere.
__device__ __forceinline__ void lane_change(uint32_t (&SRC)[4], uint32_t (&DST)[4], const uint32_t (&F)[4],
                                            const uint32_t (&r)[EAGERA][4], const PhiloxKeys& K, const Unit& un,
                                            uint32_t tag, uint32_t tlo, uint32_t thi, PackSmem* xs) {
  uint32_t lt[4], eq[4];
  if constexpr (!CROSS) {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t live = lop3<0x20>(SRC[w], DST[w], F[w]);  // SRC & ~DST & F
      lt[w] = (TOMEGA >= kOne) ? live : 0u;
      eq[w] = (TOMEGA >= kOne || TOMEGA == 0) ? 0u : live;
    }
    if (TOMEGA > 0 && TOMEGA < kOne) {
#pragma unroll
      for (int pl = 0; pl < EAGER; ++pl) plane_step<TOMEGA>(lt, eq, r[pl], pl);
      if (EAGER < NPW)
        resolve_packed(lt, eq, K, (uint32_t)un.u, un.gs, tlo, ctr3(tag, 0, 0, thi), EAGER, NPW, xs,
                       [](uint32_t (&l)[4], uint32_t (&e)[4], const uint32_t (&R)[4], int pl) {
                         plane_step<TOMEGA>(l, e, R, pl);
                       });
    }
  } else {
    constexpr uint32_t AL1 = TOMEGA >= kOne ? ~0u : 0u, AL0 = TW0 >= kOne ? ~0u : 0u;          // always accepted
    constexpr uint32_t PA1 = (TOMEGA > 0 && TOMEGA < kOne) ? ~0u : 0u, PA0 = TW0 < kOne ? ~0u : 0u;  // needs planes
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t live = SRC[w] & ~DST[w];
      lt[w] = live & ((F[w] & AL1) | (~F[w] & AL0));
      eq[w] = live & ((F[w] & PA1) | (~F[w] & PA0));
    }
#pragma unroll
    for (int pl = 0; pl < EAGER; ++pl) plane_step2(lt, eq, r[pl], F, tbit(TOMEGA, pl), tbit(TW0, pl));
    if (EAGER < NPW)
      resolve_packed(lt, eq, K, (uint32_t)un.u, un.gs, tlo, ctr3(tag, 0, 0, thi), EAGER, NPW, xs,
                     [&F](uint32_t (&l)[4], uint32_t (&e)[4], const uint32_t (&R)[4], int pl) {
                       plane_step2(l, e, R, F, ((uint32_t)TOMEGA >> (31 - pl)) & (TOMEGA < kOne ? 1u : 0u),
                                   ((uint32_t)TW0 >> (31 - pl)) & (TW0 < kOne ? 1u : 0u));
                     });
  }
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    SRC[w] ^= lt[w];
    DST[w] ^= lt[w];
  }
}

// The same with the acceptance mask precomputed (K4J_PRE): acc = candidate sites whose uniform is below their threshold.
__device__ __forceinline__ void lane_change_pre(uint32_t (&SRC)[4], uint32_t (&DST)[4], const uint4 acc) {
  const uint32_t a[4] = {acc.x, acc.y, acc.z, acc.w};
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    const uint32_t mv = lop3<0x20>(SRC[w], DST[w], a[w]);  // SRC & ~DST & acc
    SRC[w] ^= mv;
    DST[w] ^= mv;
  }
}

// Quenched-per-epoch turning-point mask of this thread's supergroup: all 128 sites are live.
__device__ __forceinline__ void draw_turn(uint32_t (&T)[4], const PhiloxKeys& K, const Unit& un,
                                          unsigned long long epoch, uint32_t tag) {
  const uint32_t live[4] = {FULL, FULL, FULL, FULL};
  lazy_less<TTURN>(T, live, K, (uint32_t)un.u, un.gs, (uint32_t)epoch, ctr3(tag, 0, 0, (uint32_t)(epoch >> 32)));
#pragma unroll
  for (int w = 0; w < 4; ++w) T[w] = (w < un.nwn) ? T[w] : 0u;
}

// Epoch-end occupancy profile: occ[site] += bit.  The warp transposes its 32 x 4 words so that lane l
// adds the bits of sites 32 j + l: every red.global.add of the warp covers 128 consecutive bytes.
__device__ __forceinline__ void add_profile(const uint32_t (&X)[4], uint32_t* occ, int S) {
  const int lane = threadIdx.x & 31;
#pragma unroll 1
  for (int t = 0; t < 32; ++t) {
    // source lane t of this warp holds supergroup g of sample smp
    const int thr = (int)(threadIdx.x & ~31u) + t;
    const int smp = SPW > 1 ? (int)blockIdx.x * SPW + thr / U : (int)blockIdx.x;
    const int g = SPW > 1 ? thr % U : thr;
    const bool ok = smp < S && g < U;
    uint32_t* dst = occ + (size_t)smp * (32 * W) + 128 * g;
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t v = __shfl_sync(FULL, X[w], t);
      const int site = 128 * g + 32 * w + lane;
      if (ok && ((v >> lane) & 1u) && site < 32 * W) atomicAdd(dst + 32 * w + lane, 1u);
    }
  }
}

// The same through bit-sliced counters (K4J_VPROF planes per lane array, one uint4 per plane and thread, in shared memory):
// an epoch-end snapshot is ONE ripple-carry addition of the thread's 128 occupation bits to its 128 vertical counters
// (two planes touched on average) instead of 128 shuffles and up to 128 atomics per warp; flush_profile() adds the
// counters to the per-site uint32 profile every 2^K4J_VPROF - 1 snapshots and at the end of the launch.  The sites of a
// thread belong to it alone, so the flush is a plain read-modify-write.
__device__ __forceinline__ void add_profile_v(const uint32_t (&X)[4], uint4* cnt /* [VPROF][NTHREADS], this thread's column */) {
  uint32_t c[4] = {X[0], X[1], X[2], X[3]};
#pragma unroll 1
  for (int p = 0; p < VPROF; ++p) {
    if ((c[0] | c[1] | c[2] | c[3]) == 0u) break;
    const uint4 t = cnt[p * NTHREADS];
    cnt[p * NTHREADS] = make_uint4(t.x ^ c[0], t.y ^ c[1], t.z ^ c[2], t.w ^ c[3]);
    c[0] &= t.x; c[1] &= t.y; c[2] &= t.z; c[3] &= t.w;
  }
}
__device__ __forceinline__ void flush_profile(uint4* cnt, uint32_t* occ_unit /* this thread's 128 counters */, int nwn) {
  uint32_t pl[VPROF > 0 ? VPROF : 1][4];
  uint32_t any = 0u;
#pragma unroll
  for (int p = 0; p < VPROF; ++p) {
    const uint4 t = cnt[p * NTHREADS];
    pl[p][0] = t.x; pl[p][1] = t.y; pl[p][2] = t.z; pl[p][3] = t.w;
    any |= t.x | t.y | t.z | t.w;
    cnt[p * NTHREADS] = make_uint4(0u, 0u, 0u, 0u);
  }
  if (any == 0u) return;
#pragma unroll
  for (int w = 0; w < 4; ++w) {
    if (w < nwn) {
#pragma unroll 1
      for (int b = 0; b < 32; ++b) {
        uint32_t v = 0u;
#pragma unroll
        for (int p = 0; p < VPROF; ++p) v |= ((pl[p][w] >> b) & 1u) << p;
        if (v) occ_unit[32 * w + b] += v;
      }
    }
  }
}

__device__ __forceinline__ uint32_t draw_offsets16(const PhiloxKeys& K, uint32_t gs, long long m) {
  const int lane = threadIdx.x & 31;
  const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
  const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), K);
  return __ballot_sync(FULL, w.x & 1u);
}

}  // namespace k4j
}  // namespace kpz

// grid = S samples, block = NTHREADS; thread u = supergroup u (idle when u >= U, but it joins every barrier / shuffle).
#ifndef K4J_MINB  // CTAs per SM the kernel is compiled for (0: left to the compiler).  1: with ~1.7 warps per SMSP registers
#define K4J_MINB 1  // are free, and the compiler's looser schedule is worth +2 % on config 5 (measured)
#endif
#if K4J_MINB > 0
extern "C" __global__ void __launch_bounds__(kpz::k4j::NTHREADS, K4J_MINB)
#else
extern "C" __global__ void __launch_bounds__(kpz::k4j::NTHREADS)
#endif
lanes_k4_sweep_jit(const __grid_constant__ kpz::LanesDev D, const __grid_constant__ kpz::LanesRunArgs R) {
  using namespace kpz;
  using namespace kpz::k4j;
  __shared__ uint32_t halo[SINGLE_WARP ? 1 : HALO_WORDS];
#if K4J_HALOCHECK
  if (threadIdx.x == 0) g_halo_check = R.check;  // every CTA writes the same pointer
  __syncthreads();
#endif
  __shared__ unsigned long long red[SINGLE_WARP ? 1 : 4 * 32];
  __shared__ PackSmem pack[NTHREADS / 32];
  const int tid = (int)threadIdx.x;
  PackSmem* const xs = pack + (tid >> 5);
  // dynamic shared memory (lanes_api.cu sizes it): K4J_PRE: NTHREADS / 32 WarpSmem; then the bit-sliced profile counters
  extern __shared__ __align__(16) unsigned char k4_dyn_smem[];
  WarpSmem* const ws = reinterpret_cast<WarpSmem*>(k4_dyn_smem) + (tid >> 5);
  uint4* const vcnt = reinterpret_cast<uint4*>(k4_dyn_smem + (K4J_PRE ? sizeof(WarpSmem) * (NTHREADS / 32) : 0));
  // vcnt[(lane array * VPROF + plane) * NTHREADS + tid]: a thread touches its own column only
  if (VPROF > 0)
    for (int p = 0; p < 2 * VPROF; ++p) vcnt[p * NTHREADS + tid] = make_uint4(0u, 0u, 0u, 0u);
  // SPW == 1: CTA = sample, thread = supergroup.  SPW > 1: CTA = one warp = SPW samples, lane = (sample, supergroup).
  int sub = 0, s = (int)blockIdx.x, lane0 = 0;
  const int lane = threadIdx.x & 31;
  Unit un;
  un.u = tid;
  bool active = un.u < U;
  if constexpr (SPW > 1) {
    sub = tid / U;
    s = (int)blockIdx.x * SPW + sub;
    un.u = tid % U;
    lane0 = sub * U;
    active = s < D.S;
  }
  un.nwn = !active ? 0 : (PARTIAL ? min(4, W - 4 * un.u) : 4);
  un.nxt = lane0 + ((un.u + 1 >= U) ? 0 : un.u + 1);
  un.prv = lane0 + ((un.u == 0) ? U - 1 : un.u - 1);
  un.gs = (uint32_t)(D.first_sample + s);
  const unsigned long long row = (unsigned long long)s * D.Wp + 4ull * (active ? un.u : 0);
  int parity = 0;

  uint32_t A[4] = {0, 0, 0, 0}, B[4] = {0, 0, 0, 0}, T[4] = {0, 0, 0, 0};
  uint32_t V[4] = {0, 0, 0, 0};  // flags of the B->A crossings when they are a set of their own (K4J_INDEP)
  if (active) {
    const uint4 a = *reinterpret_cast<const uint4*>(D.A + row);
    const uint4 b = *reinterpret_cast<const uint4*>(D.B + row);
    A[0] = a.x; A[1] = a.y; A[2] = a.z; A[3] = a.w;
    B[0] = b.x; B[1] = b.y; B[2] = b.z; B[3] = b.w;
    const uint4 t = *reinterpret_cast<const uint4*>(D.T + row);
    T[0] = t.x; T[1] = t.y; T[2] = t.z; T[3] = t.w;
    if (K4J_INDEP) {
      const uint4 v = *reinterpret_cast<const uint4*>(D.V + row);
      V[0] = v.x; V[1] = v.y; V[2] = v.z; V[3] = v.w;
    }
  }
  unsigned long long jA = 0, jB = 0;
  int ri = R.rec_begin;
  long long next_rec = ri < R.nt ? R.rec_t[ri] : -1;
  const long long t_end = R.t0 + R.n_mcs;
  const long long period = D.period;
  long long m = R.t0;
  // epoch bookkeeping without a 64-bit division per MCS
  long long epoch = period > 0 ? m / period : 0;
  long long in_epoch = period > 0 ? m - epoch * period : 0;  // m mod period
  uint32_t offbits = 0;
  auto draw_offsets = [&]() {
    if constexpr (SPW == 1) {
      offbits = draw_offsets16(D.keys, un.gs, m);
    } else {
#pragma unroll 1
      for (int k = 0; k < SPW; ++k) {  // one ballot per sample of this warp; each lane keeps its own sample's
        const uint32_t b = draw_offsets16(D.keys, (uint32_t)(D.first_sample + (int)blockIdx.x * SPW + k), m);
        if (k == sub) offbits = b;
      }
    }
  };
  if (K4J_OFFSET_MODE == 0) draw_offsets();

  auto block_sum4 = [&](unsigned long long v0, unsigned long long v1, unsigned long long v2, unsigned long long v3,
                        unsigned long long (&out)[4]) {
    unsigned long long v[4] = {v0, v1, v2, v3};
#pragma unroll
    for (int k = 0; k < 4; ++k)
#pragma unroll
      for (int d = (SPW > 1 ? U : 32) / 2; d >= 1; d >>= 1) v[k] += __shfl_down_sync(FULL, v[k], d, SPW > 1 ? U : 32);
    if (SINGLE_WARP) {
#pragma unroll
      for (int k = 0; k < 4; ++k) out[k] = v[k];  // valid in the first lane of each sample
    } else {
      const int warp = tid >> 5;
      __syncthreads();
      if (lane == 0)
#pragma unroll
        for (int k = 0; k < 4; ++k) red[k * 32 + warp] = v[k];
      __syncthreads();
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        unsigned long long a = 0;
        for (int w = 0; w < NTHREADS / 32; ++w) a += red[k * 32 + w];
        out[k] = a;
      }
    }
  };

  Eager EA, EB;
  if (!K4J_PRE) draw_eager(EA, D.keys, un, m);
  int nflush = 0;  // snapshots in the bit-sliced profile counters

  auto redraw_flags = [&]() {  // a new epoch starts at MCS m
    if (period > 0 && m > 0 && in_epoch == 0) {
      draw_turn(T, D.keys, un, (unsigned long long)epoch, TAG_TURN);
      if (K4J_INDEP) draw_turn(V, D.keys, un, (unsigned long long)epoch, TAG_TURN_V);
    }
  };

  // One MCS m.  K4J_PRE: the lane-change acceptance masks are entry kc of the precomputed chunk.  Otherwise: with the
  // eager lane-change planes Ec drawn one step earlier; draws those of MCS m+1 into En.
  auto mcs = [&](const Eager& Ec, Eager& En, int kc) {
    const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
    if (!K4J_PRE) {
      redraw_flags();
      draw_eager(En, D.keys, un, m + 1);
    }
#pragma unroll
    for (int pass = 0; pass < 2; ++pass) {
      const uint32_t o = K4J_OFFSET_MODE ? (uint32_t)pass : ((offbits >> (2 * ((int)m & 15) + pass)) & 1u);
      // in-lane hops of both lanes with the same offset
      const uint32_t c3t = ((uint32_t)pass << 27) | thi;
      if (TPA >= kOne && TPB >= kOne) {
        // rate 1 in both lanes (config 5): the hop over a thread boundary is decided by old bits alone,
        // so both sides compute it from ONE exchange: first bits go to the previous thread, last bits to the next
        uint32_t nx = 0, in = 0;
        if (SPW > 1 || o) {  // (per-lane offsets when a warp holds several samples: every lane joins the shuffle)
          uint32_t lastA = A[3], lastB = B[3];
          if (PARTIAL) {
            lastA = un.nwn >= 4 ? A[3] : A[1];
            lastB = un.nwn >= 4 ? B[3] : B[1];
          }
          const uint32_t mine = (A[0] & 1u) | ((B[0] & 1u) << 1) | ((lastA >> 31) << 2) | ((lastB >> 31) << 3);
          uint32_t vn, vp;
          unit_exchange2(mine, un.nxt, un.prv, vn, vp, halo, parity);
          nx = (active && o) ? (vn & 3u) : 0u;  // idle threads hold all-zero words and must not see a neighbour bit
          // lane A: particle on the previous thread's last site, hole on my first; lane B: the other way round
          in = (active && o) ? (((vp >> 2) & ~A[0] & 1u) | ((~(vp >> 3) & B[0] & 1u) << 1)) : 0u;
        }
        lane_pass<true, TPA>(A, un, o, nx & 1u, D.keys, TAG_PAIR, tlo, c3t, jA, xs);
        lane_pass<false, TPB>(B, un, o, nx >> 1, D.keys, TAG_PAIR_B, tlo, c3t, jB, xs);
        A[0] ^= in & 1u;
        B[0] ^= in >> 1;
      } else {
        uint32_t nx = 0;
        if (SPW > 1 || o) {
          nx = unit_exchange((A[0] & 1u) | ((B[0] & 1u) << 1), un.nxt, halo, parity);
          if (!active || !o) nx = 0;
        }
        const uint32_t cA = lane_pass<true, TPA>(A, un, o, nx & 1u, D.keys, TAG_PAIR, tlo, c3t, jA, xs);
        const uint32_t cB = lane_pass<false, TPB>(B, un, o, nx >> 1, D.keys, TAG_PAIR_B, tlo, c3t, jB, xs);
        if (SPW > 1 || o) {  // the carries are zero in an offset-0 pass
          const uint32_t in = unit_exchange(cA | (cB << 1), un.prv, halo, parity);
          if (active) {
            A[0] ^= in & 1u;
            B[0] ^= in >> 1;
          }
        }
      }
      // lane changes at turning points: A->B after pass 0, B->A after pass 1
      if (K4J_PRE) {
        if (pass == 0) lane_change_pre(A, B, ws->acc[kc][0][lane]);
        else lane_change_pre(B, A, ws->acc[kc][1][lane]);
      } else {
        if (pass == 0) lane_change(A, B, T, Ec.r[0], D.keys, un, TAG_SWITCH_AB, tlo, thi, xs);
        else lane_change(B, A, K4J_INDEP ? V : T, Ec.r[1], D.keys, un, TAG_SWITCH_BA, tlo, thi, xs);
      }
    }
    ++m;  // t = m from here on
    if (period > 0 && ++in_epoch == period) {
      in_epoch = 0;
      ++epoch;
      if (VPROF > 0) {  // occupancy profile at epoch ends
        add_profile_v(A, vcnt + tid);
        add_profile_v(B, vcnt + VPROF * NTHREADS + tid);
        if (++nflush == (1 << VPROF) - 1) {
          if (active) {
            flush_profile(vcnt + tid, D.occA + (size_t)s * (32 * W) + 128 * un.u, un.nwn);
            flush_profile(vcnt + VPROF * NTHREADS + tid, D.occB + (size_t)s * (32 * W) + 128 * un.u, un.nwn);
          }
          nflush = 0;
        }
      } else {
        add_profile(A, D.occA, D.S);
        add_profile(B, D.occB, D.S);
      }
    }
    if (m == next_rec) {
      unsigned long long tot[4];
      block_sum4(jA, jB, (unsigned long long)(__popc(A[0]) + __popc(A[1]) + __popc(A[2]) + __popc(A[3])),
                 (unsigned long long)(__popc(B[0]) + __popc(B[1]) + __popc(B[2]) + __popc(B[3])), tot);
      if (SPW > 1 ? (un.u == 0 && active) : tid == 0) {
        const size_t cell = (size_t)ri * D.S + s, plane = (size_t)R.nt * D.S;
        R.rec[cell] = (long long)(D.JA[s] + tot[0]);
        R.rec[plane + cell] = (long long)(D.JB[s] + tot[1]);
        R.rec[2 * plane + cell] = (long long)tot[2];
        R.rec[3 * plane + cell] = (long long)tot[3];
      }
      ++ri;
      next_rec = ri < R.nt ? R.rec_t[ri] : -1;
    }
    if (K4J_OFFSET_MODE == 0 && ((int)m & 15) == 0) draw_offsets();
  };

  if (K4J_PRE) {
    while (m < t_end) {  // chunks end at epoch ends: the flags are fixed over a chunk
      long long n = t_end - m < (long long)CHUNK ? t_end - m : (long long)CHUNK;
      if (period > 0 && period - in_epoch < n) n = period - in_epoch;
      redraw_flags();
      precompute_chunk(ws, ws->acc, D.keys, un, T, K4J_INDEP ? V : T, m, (int)n);
      for (int kc = 0; kc < (int)n; ++kc) mcs(EA, EA, kc);
    }
  } else {
    while (m < t_end) {
      mcs(EA, EB, 0);
      if (m >= t_end) break;
      mcs(EB, EA, 0);
    }
  }

  {
    unsigned long long tot[4];
    block_sum4(jA, jB, 0, 0, tot);
    if (SPW > 1 ? (un.u == 0 && active) : tid == 0) {
      D.JA[s] += tot[0];
      D.JB[s] += tot[1];
    }
  }
  if (VPROF > 0 && active && nflush > 0) {
    flush_profile(vcnt + tid, D.occA + (size_t)s * (32 * W) + 128 * un.u, un.nwn);
    flush_profile(vcnt + VPROF * NTHREADS + tid, D.occB + (size_t)s * (32 * W) + 128 * un.u, un.nwn);
  }
  if (active) {
    *reinterpret_cast<uint4*>(D.A + row) = make_uint4(A[0], A[1], A[2], A[3]);
    *reinterpret_cast<uint4*>(D.B + row) = make_uint4(B[0], B[1], B[2], B[3]);
    *reinterpret_cast<uint4*>(D.T + row) = make_uint4(T[0], T[1], T[2], T[3]);
    if (K4J_INDEP) *reinterpret_cast<uint4*>(D.V + row) = make_uint4(V[0], V[1], V[2], V[3]);
  }
}
