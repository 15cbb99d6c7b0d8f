// k1_sweep_jit.cuh — K1 v2: the on-chip per-sample sweep specialised at run time (NVRTC, see jit.cu) on the
// ring size and on the four acceptance thresholds (north_star (1),(3)).
//
// Why specialise.  The sweep is integer work bound by alu-pipe slots (LOP3 / SHF and - because it
// also takes an alu slot - IMAD.WIDE issue at 0.5 warp-instr/clk/SMSP; a Philox call is 20 IMAD.WIDE + 20 LOP3).  With
// the thresholds known at compile time the lazy MSB-first comparison U < T folds into a fixed boolean
// function of the few bit-planes T needs, so the pair logic costs 3-4 LOP3 per 32 pairs instead of ~15, the plane count
// is a constant, and the Philox calls of the NEXT MCS (counter-based, state-independent) are issued in the same basic
// block as the logic of the current one.  One source, three entry points: kpz_k1_sweep_jit (a CTA per sample, the whole
// run on chip), kpz_k3t_sweep_jit (K1J_TILE: 32-unit windows of a long ring, 32 MCS per trip through HBM) and
// kpz_k3_pass_jit (K1J_STREAM: one sub-lattice pass per launch).
//
// Compile-time configuration (all -D macros, set by jit.cu):
//   K1J_PW            pair-words (64-site groups) per sample = L/64
//   K1J_T0..K1J_T3    thresholds T(p), T(p_slow), T(q), T(q_slow) as integers in [0, 2^32]
//   K1J_DIS           0 no disorder tags, 1 slow-p tags, 2 slow-p and slow-q tags
//   K1J_OFFSET_MODE   0 drawn offsets, 1 alternating
//   K1J_VARIANT       code shape of the drawn-offset sweep (see below and pass_branchfree)
//
// Layout on chip: as K1 v1 (kpz_k1.cuh): thread = one unit = 128 pairs = one Philox supergroup, 4 even-site words
// P[4] and 4 odd-site words Q[4] in registers; frame 0 pairs (P,Q) = sites (2k,2k+1), frame 1 pairs (Q,P') with P'
// = P shifted by one even site.  The lattice is in frame 0 at every MCS boundary.
#pragma once
#include "sweep_types.cuh"
#include "height_lut.cuh"

#ifndef K1J_VARIANT  // code shape of the drawn-offset sweep on the LUT path:
#ifdef K1J_TILE      //   0: one code path per offset pair (4-way switch) with the Philox rounds repeated inside each;
#define K1J_VARIANT 2  // 1: branch-free (roles by mask, shifts by the offset): one basic block per MCS, most slots;
#else                //   2: 4-way switch after the Philox rounds: fewest alu slots, no overlap inside a warp.
#define K1J_VARIANT 1  // Measured: per-sample kernel (1.7 warps per SMSP) 1 >> 0, 2 (config 2: 19.3 / 17.4 / 16.0
#endif               // TSU/s); blocked stream (many warps hide the latency) 2 > 1 (20.8 vs 19.4 TSU/s).
#endif
#ifndef K1J_PACK
#define K1J_PACK 1  // small rings: several samples per warp (SPW below)
#endif
#ifndef K1J_REFRAME
#ifdef K1J_TILE
#define K1J_REFRAME 1  // merged frame changes: measured +5 % on the blocked stream (many warps per SM) ...
#else
#define K1J_REFRAME 0  // ... and -3 % / -9 % on the per-sample kernel (1.7 warps per SMSP), which keeps frame 0 per pass
#endif
#endif
#ifndef K1J_EAGER  // GENERAL path: planes drawn unconditionally; deeper planes are evaluated lazily
#ifdef K1J_TILE
#define K1J_EAGER 12  // blocked stream, planes drawn right before use: a warp needs ~12 planes anyway (8: -9 %, 16: -16 %)
#else
#define K1J_EAGER 8   // drawn one MCS ahead (6: -5 %, 10: -3 %)
#endif
#endif
#ifndef K1J_AHEAD  // 1: the planes of MCS m+1 are drawn while MCS m runs (two register sets); 0 (blocked stream only):
#ifdef K1J_TILE    // drawn right before use - fewer registers, more resident warps (config 4: +3.6 %)
#define K1J_AHEAD 0
#else
#define K1J_AHEAD 1
#endif
#endif
#if !defined(K1J_TILE) && K1J_AHEAD == 0
#error "K1J_AHEAD = 0 is implemented by the blocked-stream kernel only"
#endif
#ifndef K1J_TRIP  // GENERAL path: planes per lazy trip
#if defined(K1J_TILE) || defined(K1J_STREAM)
#define K1J_TRIP 1  // many warps per SM: pipe-bound, never draw a plane that may not be needed (config 4: +5 %)
#else
#define K1J_TRIP 2  // 1.7 warps per SMSP: latency-bound, two independent calls per trip (p = 0.8 at L = 1024: +5 %)
#endif
#endif
#ifndef K1J_UPT   // units (Philox supergroups of 256 sites) per thread of the per-sample kernel.  2: a ring of 64 units is
#define K1J_UPT 1  // ONE warp - no __syncthreads, no shared-memory halo, two independent units of pair logic per thread
#endif             // (L = 16384: see DESIGN §5); rings whose unit count is even and not ragged only.
#if (defined(K1J_TILE) || defined(K1J_STREAM)) && K1J_UPT != 1
#error "K1J_UPT > 1 is implemented by the per-sample kernel only"
#endif
#ifndef K1J_QUEUE  // per-sample kernel, > 0: the run is cut into chunks of K1J_QUEUE MCS and the CTAs pull (sample, chunk)
#define K1J_QUEUE 0  // items from a counter in chunk-major order, parking the ring in HBM between chunks (exact: the RNG is
#endif               // counter-based, it is run(a); run(b)).  Balances rings over SMSPs that hold different numbers of warps.
#ifndef K1J_PDL  // pass-by-pass stream (K3): programmatic dependent launch of consecutive passes (set by the host)
#define K1J_PDL 0
#endif
#ifndef K1J_HALOCHECK  // debug (compute-sanitizer's racecheck is closed on the GPU pool): every word published through
#define K1J_HALOCHECK 0  // the shared-memory halo carries the number of its exchange; a reader that finds another number
#endif                   // - a slot not yet written, or already overwritten by a later exchange - counts an error
#ifndef K1J_PW
#error "k1_sweep_jit.cuh needs K1J_PW, K1J_T0..3, K1J_DIS, K1J_OFFSET_MODE"
#endif

namespace kpz {
namespace k1j {

constexpr int PW = K1J_PW;
constexpr int PWp = (PW + 3) / 4 * 4;
constexpr int U = PWp / 4;                 // units (Philox supergroups) per sample
constexpr int UPT = K1J_UPT;               // units per thread
constexpr int NW = 4 * UPT;                // pair-words per thread
constexpr int UT = (U + UPT - 1) / UPT;    // threads per sample
constexpr bool PARTIAL = (PW % 4) != 0;
static_assert(UPT == 1 || (!PARTIAL && U % UPT == 0), "several units per thread: whole units, evenly divided");
#ifdef K1J_TILE
constexpr bool TILE = true;   // K3T: a warp sweeps a 32-unit window of a long ring (kpz_k3t_sweep_jit below)
#else
constexpr bool TILE = false;
#endif
constexpr bool SINGLE_WARP = TILE || UT <= 32;
// Small rings: a ring of U <= 16 units (L = 256 U sites, U a power of two) fills only U lanes, so a warp sweeps
// SPW = 32 / U independent samples side by side; every per-sample quantity (offsets, frame, record sums) is then a
// per-lane value and the shuffles run inside segments of U lanes.
// (K1J_PACK=0 turns packing off; measured, it never helps.)
constexpr int SPW = (K1J_PACK && !TILE && !PARTIAL && UT <= 16 && (UT & (UT - 1)) == 0) ? 32 / UT : 1;
constexpr int DIS = K1J_DIS;
constexpr int NTHREADS = (UT + 31) / 32 * 32;
constexpr uint64_t T0 = K1J_T0, T1 = K1J_T1, T2 = K1J_T2, T3 = K1J_T3;
constexpr uint64_t kOne = 1ull << 32;

// bit-planes U < T can depend on: 0 for T in {0, 2^32}, else 32 - ctz(T)
__host__ __device__ constexpr int planes_of(uint64_t T) {
  if (T == 0 || T >= kOne) return 0;
  int z = 0;
  while (!((T >> z) & 1ull)) ++z;
  return 32 - z;
}
__host__ __device__ constexpr int cmax(int a, int b) { return a > b ? a : b; }
constexpr int NPS = cmax(cmax(planes_of(T0), planes_of(T2)),
                         cmax(DIS >= 1 ? planes_of(T1) : 0, DIS >= 2 ? planes_of(T3) : 0));
// Rate selection "sel" of a pair depends on a (which side holds the particle), the tags and the planes.  With at most
// three such words it is ONE LOP3 (select_word); otherwise the GENERAL path compares plane by plane: the first NEAG
// planes are drawn one MCS ahead like everything else, deeper planes only while some active pair of the warp is
// still undecided (lazy, two planes per trip) - this is how non-dyadic rates such as p = 0.8 or 0.9 run.
constexpr int SEL_NVARS = 1 + (DIS >= 1) + (DIS >= 2) + NPS;
constexpr bool GENERAL = SEL_NVARS > 3;
constexpr int NEAG = !GENERAL ? NPS : (NPS < K1J_EAGER ? NPS : K1J_EAGER);
constexpr int NPSA = NEAG > 0 ? NEAG : 1;  // array extent

// The eagerly drawn random bit-planes of one MCS of one unit: r[pass][plane][word].
struct Planes {
  uint32_t r[2][NPSA][NW];
};

__device__ __forceinline__ void draw_planes(Planes& R, const PhiloxKeys& K, uint32_t G, uint32_t gs, long long m) {
  const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
#pragma unroll
  for (int pass = 0; pass < 2; ++pass) {
#pragma unroll
    for (int pl = 0; pl < NEAG; ++pl) {
#pragma unroll
      for (int j = 0; j < UPT; ++j) {  // G = the thread's first supergroup
        const uint4 v = philox4x32_10(G + j, gs, tlo, ctr3(TAG_PAIR, (uint32_t)pass, (uint32_t)pl, thi), K);
        R.r[pass][pl][4 * j + 0] = v.x;
        R.r[pass][pl][4 * j + 1] = v.y;
        R.r[pass][pl][4 * j + 2] = v.z;
        R.r[pass][pl][4 * j + 3] = v.w;
      }
    }
  }
}

// ---- pair logic as explicit LOP3s --------------------------------------------------------------------------------
template <int LUT>
__device__ __forceinline__ uint32_t lop3(uint32_t a, uint32_t b, uint32_t c) {
  uint32_t d;
  asm("lop3.b32 %0, %1, %2, %3, %4;" : "=r"(d) : "r"(a), "r"(b), "r"(c), "n"(LUT));
  return d;
}

// [U < T] for one pair whose leading plane bits are r0, r1 (compile-time evaluation of the same MSB-first rule).
__host__ __device__ constexpr int accept_bits(uint64_t T, int r0, int r1) {
  if (T >= kOne) return 1;
  if (T == 0) return 0;
  const int np = planes_of(T);
  for (int pl = 0; pl < np && pl < 2; ++pl) {
    const int t = (int)((T >> (31 - pl)) & 1ull), x = pl == 0 ? r0 : r1;
    if (t && !x) return 1;
    if (t != x) return 0;
  }
  return 0;
}
// On an active pair (a != b) the side a alone tells which move is attempted: a = 1 forward with the p class of the
// a site, a = 0 backward with the q class of the b site.  sel = "the attempted move is accepted".
__host__ __device__ constexpr int sel_bit(int a, int spa, int sqb, int r0, int r1) {
  return a ? accept_bits(spa ? T1 : T0, r0, r1) : accept_bits(sqb ? T3 : T2, r0, r1);
}
// When sel depends on at most three words (a + tags + planes) it is ONE LOP3 with this table; inputs in the order
// a, [spa], [sqb], [plane 0], [plane 1].
__host__ __device__ constexpr int sel_lut() {
  int lut = 0;
  for (int i = 0; i < 8; ++i) {
    const int in[3] = {(i >> 2) & 1, (i >> 1) & 1, i & 1};
    int k = 1, spa = 0, sqb = 0, r0 = 0, r1 = 0;
    if (DIS >= 1) spa = in[k < 3 ? k : 2], ++k;
    if (DIS >= 2) sqb = in[k < 3 ? k : 2], ++k;
    if (NPS >= 1) r0 = in[k < 3 ? k : 2], ++k;
    if (NPS >= 2) r1 = in[k < 3 ? k : 2], ++k;
    lut |= sel_bit(in[0], spa, sqb, r0, r1) << i;
  }
  return lut;
}

// sel for one word (LUT path only): a = departure side of a forward hop; spa / sqb = the tags of the pair's a / b site.
__device__ __forceinline__ uint32_t select_word(uint32_t a, uint32_t spa, uint32_t sqb, const uint32_t (&r)[NPSA][NW],
                                                int w) {
  uint32_t in[3] = {a, 0u, 0u};
  int k = 1;
  if (DIS >= 1) in[k < 3 ? k++ : 2] = spa;
  if (DIS >= 2) in[k < 3 ? k++ : 2] = sqb;
  if (NPS >= 1) in[k < 3 ? k++ : 2] = r[0][w];
  if (NPS >= 2) in[k < 3 ? k++ : 2] = r[NEAG >= 2 ? 1 : 0][w];
  return lop3<sel_lut()>(in[0], in[1], in[2]);
}

// GENERAL path helpers.
__host__ __device__ constexpr uint32_t tbit(uint64_t T, int pl) { return (uint32_t)((T >> (31 - pl)) & 1ull); }
__host__ __device__ constexpr uint32_t is_always(uint64_t T) { return T >= kOne ? 1u : 0u; }
__host__ __device__ constexpr uint32_t is_partial(uint64_t T) { return (T > 0 && T < kOne) ? 1u : 0u; }

// MSB-first comparison of ONE rate class against its constant threshold T: eq = pairs of the class whose prefix still
// equals T's, lt |= pairs decided "U < T".  A plane whose T bit is 0 costs one LOP3 per word, a 1 bit two; once T has no
// bit left below, an equal prefix can no longer become "less" and the class drops out.
template <uint64_t T>
__device__ __forceinline__ void class_planes_eager(uint32_t (&lt)[NW], uint32_t (&eq)[NW], const uint32_t (&r)[NPSA][NW]) {
  if constexpr (T > 0 && T < kOne) {
#pragma unroll
    for (int pl = 0; pl < NEAG; ++pl) {
#pragma unroll
      for (int w = 0; w < NW; ++w) {
        if (pl >= planes_of(T)) {
          eq[w] = 0u;
        } else if (tbit(T, pl)) {
          lt[w] |= eq[w] & ~r[pl][w];
          eq[w] &= r[pl][w];
        } else {
          eq[w] &= ~r[pl][w];
        }
      }
    }
  }
}
template <uint64_t T>
__device__ __forceinline__ void class_plane_lazy(uint32_t (&lt)[NW], uint32_t (&eq)[NW], const uint32_t (&R)[NW], int pl) {
  if constexpr (T > 0 && T < kOne) {
    if (pl >= planes_of(T)) {  // warp-uniform
#pragma unroll
      for (int w = 0; w < NW; ++w) eq[w] = 0u;
    } else {
      const uint32_t tb = 0u - ((uint32_t)(T >> (31 - pl)) & 1u);
#pragma unroll
      for (int w = 0; w < NW; ++w) {
        lt[w] |= eq[w] & tb & ~R[w];
        eq[w] &= ~(R[w] ^ tb);
      }
    }
  }
}

// flips of the 32 pairs of each word of one pass: x = active pairs, a = side holding the particle's departure site.
// The pairs are split into their rate classes (0 = p, 1 = p_slow, 2 = q, 3 = q_slow) once; every class then compares
// against its own constant threshold.
__device__ __forceinline__ void general_flips(uint32_t (&lt)[NW], const uint32_t (&x)[NW], const uint32_t (&a)[NW],
                                              const uint32_t (&spa)[NW], const uint32_t (&sqb)[NW],
                                              const uint32_t (&r)[NPSA][NW], const PhiloxKeys& K, uint32_t G, uint32_t gs,
                                              uint32_t tlo, uint32_t c3) {
  uint32_t e0[NW], e1[NW], e2[NW], e3[NW];
#pragma unroll
  for (int w = 0; w < NW; ++w) {
    const uint32_t xp = x[w] & a[w], xq = x[w] & ~a[w];
    const uint32_t m0 = DIS >= 1 ? (xp & ~spa[w]) : xp, m1 = DIS >= 1 ? (xp & spa[w]) : 0u;
    const uint32_t m2 = DIS >= 2 ? (xq & ~sqb[w]) : xq, m3 = DIS >= 2 ? (xq & sqb[w]) : 0u;
    lt[w] = (is_always(T0) ? m0 : 0u) | (is_always(T1) ? m1 : 0u) | (is_always(T2) ? m2 : 0u) | (is_always(T3) ? m3 : 0u);
    e0[w] = is_partial(T0) ? m0 : 0u;
    e1[w] = is_partial(T1) ? m1 : 0u;
    e2[w] = is_partial(T2) ? m2 : 0u;
    e3[w] = is_partial(T3) ? m3 : 0u;
  }
  class_planes_eager<T0>(lt, e0, r);
  if (DIS >= 1) class_planes_eager<T1>(lt, e1, r);
  class_planes_eager<T2>(lt, e2, r);
  if (DIS >= 2) class_planes_eager<T3>(lt, e3, r);
  if (NEAG < NPS) {
    const unsigned alive = __activemask();  // the streamed pass kernel's last warp may be partly retired
#pragma unroll 1
    for (int pl = NEAG; pl < NPS; pl += K1J_TRIP) {
      uint32_t any = 0u;
#pragma unroll
      for (int w = 0; w < NW; ++w) any |= e0[w] | e1[w] | e2[w] | e3[w];
      if (!__any_sync(alive, any != 0u)) break;
      uint32_t R[K1J_TRIP][NW];
#pragma unroll
      for (int t = 0; t < K1J_TRIP; ++t) {  // independent calls: their rounds interleave
        const int q = pl + t < 32 ? pl + t : 31;
#pragma unroll
        for (int j = 0; j < UPT; ++j) {
          const uint4 v = philox4x32_10(G + j, gs, tlo, c3 | ((uint32_t)q << 22), K);
          R[t][4 * j + 0] = v.x; R[t][4 * j + 1] = v.y; R[t][4 * j + 2] = v.z; R[t][4 * j + 3] = v.w;
        }
      }
#pragma unroll
      for (int t = 0; t < K1J_TRIP; ++t) {
        if (pl + t < NPS) {
          class_plane_lazy<T0>(lt, e0, R[t], pl + t);
          if (DIS >= 1) class_plane_lazy<T1>(lt, e1, R[t], pl + t);
          class_plane_lazy<T2>(lt, e2, R[t], pl + t);
          if (DIS >= 2) class_plane_lazy<T3>(lt, e3, R[t], pl + t);
        }
      }
    }
  }
}

// One sub-lattice pass with the roles known at compile time (§R3).
__device__ __forceinline__ void pass_logic(uint32_t (&a)[NW], uint32_t (&b)[NW], const uint32_t (&spa)[NW],
                                           const uint32_t (&sqb)[NW], const uint32_t (&r)[NPSA][NW]) {
#pragma unroll
  for (int w = 0; w < NW; ++w) {
    const uint32_t sel = select_word(a[w], spa[w], sqb[w], r, w);
    const uint32_t na = lop3<0xD8>(a[w], b[w], sel);  // a ^ ((a ^ b) & sel)
    const uint32_t nb = lop3<0xE4>(a[w], b[w], sel);  // b ^ ((a ^ b) & sel)
    a[w] = na;
    b[w] = nb;
  }
}

// ---- neighbour word exchange (a5): the value held by unit `src` of this sample ---------------------------------
// `parity` counts the exchanges of the CTA; the slot set alternates with it, so that a warp that runs ahead writes the
// set nobody reads any more (one barrier per exchange).
#if K1J_HALOCHECK
__device__ unsigned int* g_halo_check;  // = KpzRunArgs.check
#endif
constexpr int HALO_WORDS = (K1J_HALOCHECK ? 8 : 4) * NTHREADS;  // [2 sets][2 words per thread] (+ the same for the tags)
__device__ __forceinline__ uint32_t unit_exchange(uint32_t mine, int src, uint32_t* halo, int& parity) {
  if (SINGLE_WARP) {
    return __shfl_sync(0xFFFFFFFFu, mine, src);
  } else {
    uint32_t* slot = halo + (parity & 1) * NTHREADS;
    slot[threadIdx.x] = mine;
#if K1J_HALOCHECK
    slot[4 * NTHREADS + threadIdx.x] = (uint32_t)parity;
#endif
    __syncthreads();
    const uint32_t v = slot[src];
#if K1J_HALOCHECK
    if (slot[4 * NTHREADS + src] != (uint32_t)parity) atomicAdd(g_halo_check, 1u);
#endif
    parity += 1;
    return v;
  }
}

struct Unit {
  int nw;   // valid words of this thread (NW, fewer in the last unit of a ragged ring, 0 for an idle lane)
  int nxt;  // thread holding the next sites (ring closure: the last unit's successor is unit 0)
  int prv;
};

// frame 0 -> 1: P'[w] = P[w] >> 1 | next << 31, h = word 0 of the next unit
// (sh = 1; sh = 0 leaves P as it is: the branch-free sweep passes the offset itself)
__device__ __forceinline__ void shift_up_words(uint32_t (&P)[NW], int nw, uint32_t h, uint32_t sh) {
  if (!PARTIAL) {
#pragma unroll
    for (int w = 0; w < NW - 1; ++w) P[w] = __funnelshift_r(P[w], P[w + 1], sh);
    P[NW - 1] = __funnelshift_r(P[NW - 1], h, sh);
  } else {
#pragma unroll
    for (int w = 0; w < 4; ++w) {
      const uint32_t next = (w + 1 < nw) ? P[w + 1 < 4 ? w + 1 : 3] : h;
      P[w] = (w < nw) ? __funnelshift_r(P[w], next, sh) : 0u;
    }
  }
}
// frame 1 -> 0: P[w] = P'[w] << 1 | prev >> 31, h = last valid word of the previous unit
__device__ __forceinline__ void shift_down_words(uint32_t (&P)[NW], int nw, uint32_t h, uint32_t sh) {
  if (!PARTIAL) {
#pragma unroll
    for (int w = NW - 1; w > 0; --w) P[w] = __funnelshift_l(P[w - 1], P[w], sh);
    P[0] = __funnelshift_l(h, P[0], sh);
  } else {
#pragma unroll
    for (int w = 3; w >= 0; --w) {
      const uint32_t prev = (w > 0) ? P[w > 0 ? w - 1 : 0] : h;
      P[w] = (w < nw) ? __funnelshift_l(prev, P[w], sh) : 0u;
    }
  }
}
__device__ __forceinline__ void frame_up(uint32_t (&P)[NW], const Unit& un, uint32_t* halo, int& parity,
                                         uint32_t sh = 1u) {
  const uint32_t h = unit_exchange(P[0], un.nxt, halo, parity);
  shift_up_words(P, un.nw, h, sh);
}
__device__ __forceinline__ void frame_down(uint32_t (&P)[NW], const Unit& un, uint32_t* halo, int& parity,
                                           uint32_t sh = 1u) {
  uint32_t last = P[NW - 1];
  if (PARTIAL) last = un.nw >= 4 ? P[3] : un.nw == 3 ? P[2] : un.nw == 2 ? P[1] : P[0];
  const uint32_t h = unit_exchange(last, un.prv, halo, parity);
  shift_down_words(P, un.nw, h, sh);
}

// Frame change `from` -> `to` (each 0 or 1, warp-uniform run-time values) with ONE neighbour exchange: every unit
// publishes its first and its last valid word; the shift down by `from` uses the previous unit's last word, and the
// shift up by `to` needs the next unit's first word AFTER that unit's own shift down - which is a function of words
// this unit already holds (its own last word is the next unit's incoming word).
__device__ __forceinline__ void reframe(uint32_t (&P)[NW], const Unit& un, uint32_t from, uint32_t to, uint32_t* halo,
                                        int& parity) {
  uint32_t last = P[NW - 1];
  if (PARTIAL) last = un.nw >= 4 ? P[3] : un.nw == 3 ? P[2] : un.nw == 2 ? P[1] : P[0];
  uint32_t hn, hp;  // next unit's first word, previous unit's last word
  if (SINGLE_WARP) {
    hn = __shfl_sync(0xFFFFFFFFu, P[0], un.nxt);
    hp = __shfl_sync(0xFFFFFFFFu, last, un.prv);
  } else {
    uint32_t* slot = halo + (parity & 1) * (2 * NTHREADS);
    slot[2 * threadIdx.x] = P[0];
    slot[2 * threadIdx.x + 1] = last;
#if K1J_HALOCHECK
    slot[4 * NTHREADS + 2 * threadIdx.x] = (uint32_t)parity;
#endif
    __syncthreads();
    hn = slot[2 * un.nxt];
    hp = slot[2 * un.prv + 1];
#if K1J_HALOCHECK
    if (slot[4 * NTHREADS + 2 * un.nxt] != (uint32_t)parity || slot[4 * NTHREADS + 2 * un.prv] != (uint32_t)parity)
      atomicAdd(g_halo_check, 1u);
#endif
    parity += 1;
  }
  hn = __funnelshift_l(last, hn, from);  // the next unit's first word after ITS shift down
  shift_down_words(P, un.nw, hp, from);
  shift_up_words(P, un.nw, hn, to);
}

// Quenched tags in the frames the passes use them in.
struct Tags {
  uint32_t spa0[NW];  // slow-p at even sites  (a side of frame 0)
  uint32_t spa1[NW];  // slow-p at odd sites   (a side of frame 1)
  uint32_t sqb0[NW];  // slow-q at odd sites   (b side of frame 0)
  uint32_t sqb1[NW];  // slow-q at even sites, shifted to frame 1 (b side of frame 1)
};

// One MCS with the offsets (O0, O1) of its two passes known at compile time; frame 0 on entry and exit.
template <int O0, int O1>
__device__ __forceinline__ void mcs_logic(uint32_t (&P)[NW], uint32_t (&Q)[NW], const Tags& G, const Planes& R,
                                          const Unit& un, uint32_t* halo, int& parity) {
  if (O0) frame_up(P, un, halo, parity);
  if (O0) pass_logic(Q, P, G.spa1, G.sqb1, R.r[0]);
  else pass_logic(P, Q, G.spa0, G.sqb0, R.r[0]);
  if (O1 && !O0) frame_up(P, un, halo, parity);
  if (!O1 && O0) frame_down(P, un, halo, parity);
  if (O1) pass_logic(Q, P, G.spa1, G.sqb1, R.r[1]);
  else pass_logic(P, Q, G.spa0, G.sqb0, R.r[1]);
  if (O1) frame_down(P, un, halo, parity);
}

// Branch-free form (K1J_VARIANT 1): the offset o of a pass is a run-time, warp-uniform value.  P is brought to frame
// o by reframe() (funnel shifts by 0 or 1 bit), the a side is picked by a mask (P and Q enter the update
// symmetrically, so only the rate selection needs to know which of them is a): the whole MCS is one basic block,
// which the scheduler fills with the Philox rounds of the next MCS.  P must be in frame o on entry.
__device__ __forceinline__ void pass_branchfree(uint32_t (&P)[NW], uint32_t (&Q)[NW], const Tags& G,
                                                const uint32_t (&r)[NPSA][NW], const Unit& un, uint32_t o,
                                                uint32_t* halo, int& parity, const PhiloxKeys& K, uint32_t Gu,
                                                uint32_t gs, uint32_t tlo, uint32_t c3) {
  const uint32_t M = 0u - o;  // all ones in frame 1
  if constexpr (!GENERAL) {
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      const uint32_t a = lop3<0xCA>(M, Q[w], P[w]);  // frame 1: a = odd site (Q); frame 0: a = even site (P)
      uint32_t spa = 0u, sqb = 0u;
      if (DIS >= 1) spa = lop3<0xCA>(M, G.spa1[w], G.spa0[w]);
      if (DIS >= 2) sqb = lop3<0xCA>(M, G.sqb1[w], G.sqb0[w]);
      const uint32_t sel = select_word(a, spa, sqb, r, w);
      const uint32_t np = lop3<0xD8>(P[w], Q[w], sel);
      const uint32_t nq = lop3<0xE4>(P[w], Q[w], sel);
      P[w] = np;
      Q[w] = nq;
    }
  } else {
    uint32_t a[NW], x[NW], spa[NW], sqb[NW], lt[NW];
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      a[w] = lop3<0xCA>(M, Q[w], P[w]);
      x[w] = P[w] ^ Q[w];
      spa[w] = DIS >= 1 ? lop3<0xCA>(M, G.spa1[w], G.spa0[w]) : 0u;
      sqb[w] = DIS >= 2 ? lop3<0xCA>(M, G.sqb1[w], G.sqb0[w]) : 0u;
    }
    general_flips(lt, x, a, spa, sqb, r, K, Gu, gs, tlo, c3);
#pragma unroll
    for (int w = 0; w < NW; ++w) {
      P[w] ^= lt[w];
      Q[w] ^= lt[w];
    }
  }
}

// ---- K2 fused: heights h_x = inclusive prefix of (2n-1), exact sums per sample (a6, a7) -----------
// 8 sites at a time through the byte table of height_lut.cuh.
__device__ __forceinline__ void record_sums(const uint32_t (&P)[NW], const uint32_t (&Q)[NW], int nw,
                                            const uint32_t* lut, long long* scratch, long long* out_h,
                                            long long* out_h2, bool writer) {
  int r = 0, s1 = 0, s2 = 0;
  if (nw > 0) unit_relative_sums_lut<NW>(P, Q, nw, lut, r, s1, s2);
  const int lane = threadIdx.x & 31;
  constexpr int SEG = SPW > 1 ? UT : 32;  // lanes of one sample inside a warp
  const int pos = lane & (SEG - 1);
  int incl = r;  // inclusive scan of the unit totals: the height before unit u is the sum over units < u
#pragma unroll
  for (int d = 1; d < SEG; d <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, d, SEG);
    if (pos >= d) incl += v;
  }
  long long base = (long long)(incl - r);
  if (!SINGLE_WARP) {
    const int warp = threadIdx.x >> 5;
    int* wtot = reinterpret_cast<int*>(scratch + 64);
    __syncthreads();
    if (lane == 31) wtot[warp] = incl;
    __syncthreads();
    int add = 0;
    for (int k = 0; k < warp; ++k) add += wtot[k];
    base += add;
  }
  const long long n = 64LL * nw;
  long long H = n * base + (long long)s1;
  long long H2 = n * base * base + 2LL * base * (long long)s1 + (long long)s2;
#pragma unroll
  for (int d = SEG / 2; d >= 1; d >>= 1) {
    H += __shfl_down_sync(0xFFFFFFFFu, H, d, SEG);
    H2 += __shfl_down_sync(0xFFFFFFFFu, H2, d, SEG);
  }
  if (SINGLE_WARP) {
    if (pos == 0 && writer) {
      *out_h = H;
      *out_h2 = H2;
    }
  } else {
    const int warp = threadIdx.x >> 5;
    if (lane == 0) {
      scratch[warp] = H;
      scratch[32 + warp] = H2;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
      long long a = 0, b = 0;
      for (int k = 0; k < NTHREADS / 32; ++k) {
        a += scratch[k];
        b += scratch[32 + k];
      }
      *out_h = a;
      *out_h2 = b;
    }
  }
}

// Offsets of the 32 passes of the 16 MCS starting at (m & ~15): lane l draws (mcs = base + l/2, pass = l & 1) and a
// ballot packs them: bit 2k+pass of the result = offset of pass `pass` of MCS base+k.
__device__ __forceinline__ uint32_t draw_offsets16(const PhiloxKeys& K, uint32_t gs, long long m) {
  const int lane = threadIdx.x & 31;
  const unsigned long long mb = ((unsigned long long)m & ~15ull) + (unsigned)(lane >> 1);
  const uint4 w = philox4x32_10(0u, gs, (uint32_t)mb, ctr3(TAG_OFFSET, lane & 1, 0, (uint32_t)(mb >> 32)), K);
  return __ballot_sync(0xFFFFFFFFu, w.x & 1u);
}

struct Ctx {
  uint32_t P[NW], Q[NW];
  Tags tags;
  Unit un;
  uint32_t gs;   // global sample index (Philox counter c1)
  uint32_t G;    // supergroup index of this thread's first unit (Philox counter c0)
  int parity;
  uint32_t offbits;
  uint32_t frame;  // frame P is in between MCS (branch-free sweep: the offset of the last pass; else 0)
};

// MCS m: draw the planes of MCS m+1 into Rn, then apply MCS m with the planes Rc drawn one step earlier.  Both sit
// in one basic block per offset combination, so the scheduler overlaps the Philox rounds with the pair logic.
__device__ __forceinline__ void mcs_step(Ctx& c, const Planes& Rc, Planes& Rn, const PhiloxKeys& K, long long m,
                                         uint32_t* halo) {
  const uint32_t tlo = (uint32_t)m, thi = (uint32_t)((unsigned long long)m >> 32);
  if (K1J_OFFSET_MODE == 1 && !GENERAL) {
    if (K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
    mcs_logic<0, 1>(c.P, c.Q, c.tags, Rc, c.un, halo, c.parity);
  } else if (K1J_VARIANT == 1 || GENERAL || SPW > 1) {
    const uint32_t code = K1J_OFFSET_MODE == 1 ? 2u : (c.offbits >> (2 * ((int)m & 15))) & 3u;  // o0 | o1 << 1
    if (K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
    if (K1J_REFRAME && SPW == 1) {  // one exchange per frame change, the frame is carried across MCS
      reframe(c.P, c.un, c.frame, code & 1u, halo, c.parity);
      pass_branchfree(c.P, c.Q, c.tags, Rc.r[0], c.un, code & 1u, halo, c.parity, K, c.G, c.gs, tlo,
                      ctr3(TAG_PAIR, 0u, 0u, thi));
      reframe(c.P, c.un, code & 1u, code >> 1, halo, c.parity);
      pass_branchfree(c.P, c.Q, c.tags, Rc.r[1], c.un, code >> 1, halo, c.parity, K, c.G, c.gs, tlo,
                      ctr3(TAG_PAIR, 1u, 0u, thi));
      c.frame = code >> 1;
    } else {  // frame 0 around every pass: shift up by o, pass, shift down by o
      frame_up(c.P, c.un, halo, c.parity, code & 1u);
      pass_branchfree(c.P, c.Q, c.tags, Rc.r[0], c.un, code & 1u, halo, c.parity, K, c.G, c.gs, tlo,
                      ctr3(TAG_PAIR, 0u, 0u, thi));
      frame_down(c.P, c.un, halo, c.parity, code & 1u);
      frame_up(c.P, c.un, halo, c.parity, code >> 1);
      pass_branchfree(c.P, c.Q, c.tags, Rc.r[1], c.un, code >> 1, halo, c.parity, K, c.G, c.gs, tlo,
                      ctr3(TAG_PAIR, 1u, 0u, thi));
      frame_down(c.P, c.un, halo, c.parity, code >> 1);
    }
  } else {
    const uint32_t code = (c.offbits >> (2 * ((int)m & 15))) & 3u;  // o0 | o1 << 1
    constexpr bool INSIDE = K1J_VARIANT == 0;  // variant 0: the Philox rounds are repeated inside every code path;
    if (!INSIDE && K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);  // variant 2: drawn once, before the switch
    switch (code) {
      case 0:
        if (INSIDE && K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
        mcs_logic<0, 0>(c.P, c.Q, c.tags, Rc, c.un, halo, c.parity);
        break;
      case 1:
        if (INSIDE && K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
        mcs_logic<1, 0>(c.P, c.Q, c.tags, Rc, c.un, halo, c.parity);
        break;
      case 2:
        if (INSIDE && K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
        mcs_logic<0, 1>(c.P, c.Q, c.tags, Rc, c.un, halo, c.parity);
        break;
      default:
        if (INSIDE && K1J_AHEAD) draw_planes(Rn, K, c.G, c.gs, m + 1);
        mcs_logic<1, 1>(c.P, c.Q, c.tags, Rc, c.un, halo, c.parity);
        break;
    }
  }
}

}  // namespace k1j
}  // namespace kpz

#if defined(K1J_STREAM)
// ---- K3 pass kernel, specialised: one launch = one sub-lattice pass of a ring streamed through HBM (north_star (2)) --
// Thread = one unit: 128-bit loads of its 4+4 words from the input buffer, the frame change (if this pass's offset
// differs from the stored frame) with ONE extra word of the unmodified input (the halo), the same
// folded pair logic as K1, 128-bit stores to the ping-pong partner.  The frame of the stored ring follows the offsets.
extern "C" __global__ void __launch_bounds__(256)
kpz_k3_pass_jit(const __grid_constant__ kpz::KpzDev D, const __grid_constant__ kpz::K3Pass A) {
  using namespace kpz;
  using namespace kpz::k1j;
#if K1J_PDL
  // Programmatic dependent launch (the host sets the launch attribute): the NEXT pass may start to launch while this
  // one runs; its threads draw their planes - which depend on nothing in memory - and only then wait for this pass to
  // be complete and visible.  Hides the launch gap between two passes.
  asm volatile("griddepcontrol.launch_dependents;" ::: "memory");
#endif
  const unsigned long long gid = (unsigned long long)blockIdx.x * 256ull + threadIdx.x;
  if (gid >= (unsigned long long)D.S * U) return;
  const int s = (int)(gid / U);
  const int u = (int)(gid % U);
  const int nw = PARTIAL ? min(4, PW - 4 * u) : 4;
  const unsigned long long srow = (unsigned long long)s * PWp;
  const unsigned long long row = srow + 4ull * u;
  const uint32_t gs = (uint32_t)(D.first_sample + s);
  const uint32_t tlo = (uint32_t)A.m, thi = (uint32_t)((unsigned long long)A.m >> 32);
  uint32_t r[NPSA][4];
  if (A.fo) {  // a kernel parameter: no memory is read before the wait below
    uint32_t keep = 0u;
#pragma unroll
    for (int pl = 0; pl < NEAG; ++pl) {
      const uint4 v = philox4x32_10((uint32_t)u, gs, tlo, ctr3(TAG_PAIR, (uint32_t)A.pass, (uint32_t)pl, thi), D.keys);
      r[pl][0] = v.x; r[pl][1] = v.y; r[pl][2] = v.z; r[pl][3] = v.w;
      keep ^= v.x ^ v.y ^ v.z ^ v.w;
    }
#if K1J_PDL
    asm volatile("" ::"r"(keep));  // the planes are computed BEFORE the wait
#endif
    (void)keep;
  }
#if K1J_PDL
  asm volatile("griddepcontrol.wait;" ::: "memory");
#endif
  const uint32_t fin = A.fin[s];
  const uint32_t o = A.fo ? A.fo[s] : 0u;
  uint32_t P[4], Q[4];
  {
    const uint4 e = *reinterpret_cast<const uint4*>(A.Ein + row);
    const uint4 q = *reinterpret_cast<const uint4*>(A.Oin + row);
    P[0] = e.x; P[1] = e.y; P[2] = e.z; P[3] = e.w;
    Q[0] = q.x; Q[1] = q.y; Q[2] = q.z; Q[3] = q.w;
  }
  const int nxt = (u + 1 >= U) ? 0 : u + 1;
  if (fin != o) {
    if (o) {
      shift_up_words(P, nw, A.Ein[srow + 4ull * nxt], 1u);
    } else {
      const int prv = (u == 0) ? U - 1 : u - 1;
      const int nwp = PARTIAL ? min(4, PW - 4 * prv) : 4;
      shift_down_words(P, nw, A.Ein[srow + 4ull * prv + nwp - 1], 1u);
    }
  }
  if (A.fo) {
    uint32_t spa[4] = {0, 0, 0, 0}, sqb[4] = {0, 0, 0, 0};
    if (DIS >= 1) {
      const uint4 x = *reinterpret_cast<const uint4*>((o ? D.SPO : D.SPE) + row);
      spa[0] = x.x; spa[1] = x.y; spa[2] = x.z; spa[3] = x.w;
    }
    if (DIS >= 2) {
      const uint4 x = *reinterpret_cast<const uint4*>((o ? D.SQE : D.SQO) + row);
      sqb[0] = x.x; sqb[1] = x.y; sqb[2] = x.z; sqb[3] = x.w;
      if (o) shift_up_words(sqb, nw, D.SQE[srow + 4ull * nxt], 1u);
    }
    const uint32_t M = 0u - o;
    if constexpr (!GENERAL) {
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        const uint32_t a = lop3<0xCA>(M, Q[w], P[w]);
        const uint32_t sel = select_word(a, spa[w], sqb[w], r, w);
        const uint32_t np = lop3<0xD8>(P[w], Q[w], sel);
        const uint32_t nq = lop3<0xE4>(P[w], Q[w], sel);
        P[w] = np;
        Q[w] = nq;
      }
    } else {
      uint32_t a[4], x[4], lt[4];
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        a[w] = lop3<0xCA>(M, Q[w], P[w]);
        x[w] = P[w] ^ Q[w];
      }
      general_flips(lt, x, a, spa, sqb, r, D.keys, (uint32_t)u, gs, tlo, ctr3(TAG_PAIR, (uint32_t)A.pass, 0u, thi));
#pragma unroll
      for (int w = 0; w < 4; ++w) {
        P[w] ^= lt[w];
        Q[w] ^= lt[w];
      }
    }
  }
  *reinterpret_cast<uint4*>(A.Eout + row) = make_uint4(P[0], P[1], P[2], P[3]);
  *reinterpret_cast<uint4*>(A.Oout + row) = make_uint4(Q[0], Q[1], Q[2], Q[3]);
}
#elif !defined(K1J_TILE)
// grid = S samples (ceil(S / SPW) warps for small rings), block = NTHREADS; thread u = units UPT u .. UPT u + UPT - 1
// (idle when u >= UT, but it joins every barrier / shuffle).
extern "C" __global__ void __launch_bounds__(kpz::k1j::NTHREADS)
kpz_k1_sweep_jit(const __grid_constant__ kpz::KpzDev D, const __grid_constant__ kpz::KpzRunArgs A) {
  using namespace kpz;
  using namespace kpz::k1j;
  __shared__ uint32_t halo[SINGLE_WARP ? 1 : HALO_WORDS];
  __shared__ long long scratch[SINGLE_WARP ? 1 : 96];
  __shared__ uint32_t lut[256];
  for (int i = threadIdx.x; i < 256; i += NTHREADS) lut[i] = height_lut_entry(i);
#if K1J_HALOCHECK
  if (threadIdx.x == 0) g_halo_check = A.check;  // every CTA writes the same pointer
#endif
  __syncthreads();

  // SPW == 1: CTA = sample, thread = UPT units.  SPW > 1: CTA = one warp = SPW samples, lane = (sample, units).
  // run_sample: MCS [ta, tb) of the sample(s) of block index sblk
  auto run_sample = [&](const int sblk, const long long ta, const long long tb) {
  int sub = 0, s = sblk, u = (int)threadIdx.x, lane0 = 0;  // lane0 = first lane of this sample
  bool active = u < UT;
  if constexpr (SPW > 1) {
    sub = (int)threadIdx.x / UT;
    s = sblk * SPW + sub;
    u = (int)threadIdx.x % UT;
    lane0 = sub * UT;
    active = s < D.S;
  }
  Ctx c;
  c.un.nw = !active ? 0 : (PARTIAL ? min(4, PW - 4 * u) : NW);
  c.un.nxt = lane0 + ((u + 1 >= UT) ? 0 : u + 1);
  c.un.prv = lane0 + ((u == 0) ? UT - 1 : u - 1);
  if (!SINGLE_WARP) asm volatile("" : "+r"(c.un.nxt), "+r"(c.un.prv));  // measured: +3.5 % on 2-warp rings, -5 % on 1-warp
  c.gs = (uint32_t)(D.first_sample + s);
  c.G = (uint32_t)(UPT * u);
  c.parity = 0;
  c.offbits = 0;
  c.frame = 0;
  const unsigned long long row = (unsigned long long)s * PWp + (unsigned long long)NW * (active ? u : 0);
#pragma unroll
  for (int w = 0; w < NW; ++w) {
    c.P[w] = c.Q[w] = 0u;
    c.tags.spa0[w] = c.tags.spa1[w] = c.tags.sqb0[w] = c.tags.sqb1[w] = 0u;
  }
  auto load_words = [&](uint32_t(&dst)[NW], const uint32_t* src) {
#pragma unroll
    for (int j = 0; j < UPT; ++j) {
      // (K1J_QUEUE: the ring may have been parked by another SM a moment ago: read it past L1)
      const uint4 v = K1J_QUEUE ? __ldcg(reinterpret_cast<const uint4*>(src + row + 4 * j))
                                : *reinterpret_cast<const uint4*>(src + row + 4 * j);
      dst[4 * j + 0] = v.x; dst[4 * j + 1] = v.y; dst[4 * j + 2] = v.z; dst[4 * j + 3] = v.w;
    }
  };
  if (active) {
    load_words(c.P, D.E);
    load_words(c.Q, D.O);
    if (DIS >= 1) {
      load_words(c.tags.spa0, D.SPE);
      load_words(c.tags.spa1, D.SPO);
    }
    if (DIS >= 2) {
      load_words(c.tags.sqb0, D.SQO);
      load_words(c.tags.sqb1, D.SQE);
    }
  }
  if (DIS >= 2) frame_up(c.tags.sqb1, c.un, halo, c.parity);  // b side of frame 1 = the NEXT even site

  int ri = A.rec_begin;
  while (K1J_QUEUE && ri < A.nt && A.rec_t[ri] <= ta) ++ri;  // records of earlier chunks
  long long next_rec = ri < A.nt ? A.rec_t[ri] : -1;
  const long long t_end = tb;
  long long m = ta;
  auto draw_offsets = [&]() {
    if constexpr (SPW == 1) {
      c.offbits = draw_offsets16(D.keys, c.gs, m);
    } else {
#pragma unroll 1
      for (int k = 0; k < SPW; ++k) {  // one ballot per sample of this warp; each lane keeps its own sample's
        const uint32_t b = draw_offsets16(D.keys, (uint32_t)(D.first_sample + sblk * SPW + k), m);
        if (k == sub) c.offbits = b;
      }
    }
  };
  if (K1J_OFFSET_MODE == 0) draw_offsets();

  Planes RA, RB;
  draw_planes(RA, D.keys, c.G, c.gs, m);

  auto to_frame0 = [&]() {
    if (c.frame) {  // warp- and CTA-uniform
      reframe(c.P, c.un, c.frame, 0u, halo, c.parity);
      c.frame = 0;
    }
  };
  auto after_mcs = [&]() {  // m has been advanced: t = m
    if (m == next_rec) {
      to_frame0();
      record_sums(c.P, c.Q, c.un.nw, lut, scratch, A.rec_sum_h + (size_t)ri * D.S + s,
                  A.rec_sum_h2 + (size_t)ri * D.S + s, active);
      ++ri;
      next_rec = ri < A.nt ? A.rec_t[ri] : -1;
    }
    if (K1J_OFFSET_MODE == 0 && ((int)m & 15) == 0) draw_offsets();
  };

  while (m < t_end) {
    mcs_step(c, RA, RB, D.keys, m, halo);
    ++m;
    after_mcs();
    if (m >= t_end) break;
    mcs_step(c, RB, RA, D.keys, m, halo);
    ++m;
    after_mcs();
  }
  to_frame0();

  if (active) {
#pragma unroll
    for (int j = 0; j < UPT; ++j) {
      *reinterpret_cast<uint4*>(D.E + row + 4 * j) = make_uint4(c.P[4 * j], c.P[4 * j + 1], c.P[4 * j + 2], c.P[4 * j + 3]);
      *reinterpret_cast<uint4*>(D.O + row + 4 * j) = make_uint4(c.Q[4 * j], c.Q[4 * j + 1], c.Q[4 * j + 2], c.Q[4 * j + 3]);
    }
  }
  };  // run_sample
#if K1J_QUEUE
  static_assert(SPW == 1, "K1J_QUEUE: one sample per CTA");
  __shared__ unsigned int s_item;
  const long long nchunks = (A.n_mcs + K1J_QUEUE - 1) / K1J_QUEUE;
  const unsigned long long nitems = (unsigned long long)nchunks * (unsigned long long)D.S;
  for (;;) {
    if (threadIdx.x == 0) s_item = atomicAdd(A.queue, 1u);
    __syncthreads();
    const unsigned long long item = s_item;
    __syncthreads();
    if (item >= nitems) break;
    const int smp = (int)(item % (unsigned)D.S);
    const long long ch = (long long)(item / (unsigned)D.S);
    if (ch > 0) {  // the previous chunk of this ring was handed out D.S items ago: wait until it is parked
      if (threadIdx.x == 0) {
        unsigned int done;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(done) : "l"(A.queue + 1 + smp) : "memory");
          if (done < (unsigned)ch) __nanosleep(128);
        } while (done < (unsigned)ch);
      }
      __syncthreads();
    }
    const long long ta = A.t0 + ch * K1J_QUEUE;
    run_sample(smp, ta, ta + K1J_QUEUE < A.t0 + A.n_mcs ? ta + K1J_QUEUE : A.t0 + A.n_mcs);
    __threadfence();
    __syncthreads();
    if (threadIdx.x == 0)
      asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(A.queue + 1 + smp), "r"((unsigned)(ch + 1)) : "memory");
  }
#else
  run_sample((int)blockIdx.x, A.t0, A.t0 + A.n_mcs);
#endif
}
#else  // K1J_TILE
// ---- K3T: temporally blocked sweep of rings beyond on-chip memory (north_star (2)) --------------------
// The ring streams through HBM once per CHUNK of up to 32 MCS instead of once per pass.  A warp loads a window of 32
// consecutive units (lane l holds unit tile*30 - 1 + l mod U), sweeps it exactly like K1 with the neighbour words of
// the window's two ends left undefined, and stores the 30 interior units to the ping-pong buffer.  A pass moves
// information by one site, so after k passes only the outer k+1 sites of the window are contaminated: the two end
// units (256 sites each) absorb up to 127 MCS.  The random numbers are counter-based - keyed by the GLOBAL unit index
// - so the halo units a neighbouring warp recomputes are bit-identical, and the result equals the pass-by-pass sweep.
#ifndef K1J_TILE_MINB  // CTAs per SM this kernel is compiled for (0: left to the compiler, which takes 114 registers; 4: 120
#define K1J_TILE_MINB 4  // registers and a slightly better schedule: config 4 +1.7 %; 5 ... 8 CTAs: no further gain, measured)
#endif
#if K1J_TILE_MINB > 0
extern "C" __global__ void __launch_bounds__(128, K1J_TILE_MINB)
#else
extern "C" __global__ void __launch_bounds__(128)
#endif
kpz_k3t_sweep_jit(const __grid_constant__ kpz::KpzDev D, const __grid_constant__ kpz::K3TArgs A) {
  using namespace kpz;
  using namespace kpz::k1j;
  constexpr int TI = 30;  // interior units per window
  constexpr int NT = (U + TI - 1) / TI;
  const int lane = threadIdx.x & 31;
  const long long wid = (long long)blockIdx.x * 4 + (threadIdx.x >> 5);
  if (wid >= (long long)D.S * NT) return;  // whole warps leave; the kernel has no block-wide barrier
  const int s = (int)(wid / NT), tile = (int)(wid % NT);
  int g = (tile * TI - 1 + lane) % U;
  if (g < 0) g += U;
  Ctx c;
  c.un.nw = PARTIAL ? min(4, PW - 4 * g) : 4;
  c.un.nxt = lane < 31 ? lane + 1 : 31;
  c.un.prv = lane > 0 ? lane - 1 : 0;
  c.gs = (uint32_t)(D.first_sample + s);
  c.G = (uint32_t)g;
  c.parity = 0;
  c.offbits = 0;
  c.frame = 0;
  const unsigned long long row = (unsigned long long)s * PWp + 4ull * g;
  {
    const uint4 e = *reinterpret_cast<const uint4*>(D.E + row);
    const uint4 o = *reinterpret_cast<const uint4*>(D.O + row);
    c.P[0] = e.x; c.P[1] = e.y; c.P[2] = e.z; c.P[3] = e.w;
    c.Q[0] = o.x; c.Q[1] = o.y; c.Q[2] = o.z; c.Q[3] = o.w;
  }
#pragma unroll
  for (int w = 0; w < 4; ++w) c.tags.spa0[w] = c.tags.spa1[w] = c.tags.sqb0[w] = c.tags.sqb1[w] = 0u;
  if (DIS >= 1) {
    const uint4 x = *reinterpret_cast<const uint4*>(D.SPE + row);
    const uint4 y = *reinterpret_cast<const uint4*>(D.SPO + row);
    c.tags.spa0[0] = x.x; c.tags.spa0[1] = x.y; c.tags.spa0[2] = x.z; c.tags.spa0[3] = x.w;
    c.tags.spa1[0] = y.x; c.tags.spa1[1] = y.y; c.tags.spa1[2] = y.z; c.tags.spa1[3] = y.w;
  }
  if (DIS >= 2) {
    const uint4 x = *reinterpret_cast<const uint4*>(D.SQO + row);
    const uint4 y = *reinterpret_cast<const uint4*>(D.SQE + row);
    c.tags.sqb0[0] = x.x; c.tags.sqb0[1] = x.y; c.tags.sqb0[2] = x.z; c.tags.sqb0[3] = x.w;
    c.tags.sqb1[0] = y.x; c.tags.sqb1[1] = y.y; c.tags.sqb1[2] = y.z; c.tags.sqb1[3] = y.w;
    frame_up(c.tags.sqb1, c.un, nullptr, c.parity);  // lane 31's incoming word is undefined: it is a halo unit
  }
  const long long t_end = A.t0 + A.n_mcs;
  long long m = A.t0;
  if (K1J_OFFSET_MODE == 0) c.offbits = draw_offsets16(D.keys, c.gs, m);
  if (K1J_AHEAD) {
    Planes RA, RB;
    draw_planes(RA, D.keys, c.G, c.gs, m);
    while (m < t_end) {
      mcs_step(c, RA, RB, D.keys, m, nullptr);
      ++m;
      if (K1J_OFFSET_MODE == 0 && ((int)m & 15) == 0) c.offbits = draw_offsets16(D.keys, c.gs, m);
      if (m >= t_end) break;
      mcs_step(c, RB, RA, D.keys, m, nullptr);
      ++m;
      if (K1J_OFFSET_MODE == 0 && ((int)m & 15) == 0) c.offbits = draw_offsets16(D.keys, c.gs, m);
    }
  } else {
    Planes RA;
#pragma unroll 1
    while (m < t_end) {
      draw_planes(RA, D.keys, c.G, c.gs, m);
      mcs_step(c, RA, RA, D.keys, m, nullptr);
      ++m;
      if (K1J_OFFSET_MODE == 0 && ((int)m & 15) == 0) c.offbits = draw_offsets16(D.keys, c.gs, m);
    }
  }
  if (c.frame) reframe(c.P, c.un, c.frame, 0u, nullptr, c.parity);
  if (lane >= 1 && lane <= TI && tile * TI + lane - 1 < U) {
    *reinterpret_cast<uint4*>(A.Eout + row) = make_uint4(c.P[0], c.P[1], c.P[2], c.P[3]);
    *reinterpret_cast<uint4*>(A.Oout + row) = make_uint4(c.Q[0], c.Q[1], c.Q[2], c.Q[3]);
  }
}
#endif  // K1J_TILE
