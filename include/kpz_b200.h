/*
 * include/kpz_b200.h — C ABI of libkpz_b200.so: the B200 (sm_100a) hot path of arxiv/paper_1012_0385.
 *
 * What the library computes (citations: PAPER.md:<line> = /root/reference/PAPER.md; DESIGN §R<n> = the numbered
 * readings in DESIGN.md §1):
 *   - the two-sub-lattice Monte-Carlo sweep of the 1+1D RSOS/KPZ model in ASEP lattice-gas form on periodic
 *     rings, site-dependent rates p_i, q_i with quenched bimodal disorder (PAPER.md:151-155,
 *     Eq. 8), randomness from counter-based Philox4x32-10;
 *   - heights h_x and the exact integer sums behind the width W of Eq. 3 at listed record
 *     times, W^2 averaged over samples;
 *   - the two-lane opposite-direction model with turning points.
 *
 * Conventions
 *   - Every function returns 0 (KPZ_OK) or a negative error code; no exception or abort crosses the ABI.
 *     kpz_last_error() returns a thread-local text for the last failing call.
 *   - Pointers named d_* are DEVICE pointers, all others are HOST pointers.  The caller (PyTorch) allocates
 *     all device memory — the workspace handed to *_create and every d_* output — and owns the CUDA stream;
 *     the handle borrows them and they must outlive it.  The library performs no device allocation.
 *   - All work is enqueued on the stream given at create time; only the calls documented "syncs" wait for it.
 *   - Lattice / mask words use the NATURAL layout: bit (i & 31) of word (i >> 5) is site i; a sample occupies
 *     L/32 consecutive uint32 words; samples are consecutive.  (Internally rings are kept de-interleaved.)
 *   - L must be a multiple of 64, L >= 64.  Handles are not thread-safe; distinct handles are independent.
 */
#ifndef KPZ_B200_H
#define KPZ_B200_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define KPZ_OK 0
#define KPZ_EINVAL (-1)       /* NULL pointer, L odd or < 4, probability outside [0,1], nsamples < 1, bad record times */
#define KPZ_EUNSUPPORTED (-2) /* L not a multiple of 64, size beyond a path's limit, sum-of-squares overflow guard */
#define KPZ_ENOMEM (-3)       /* workspace / output capacity too small */
#define KPZ_ECUDA (-4)        /* CUDA launch or runtime error; text in kpz_last_error() */

typedef struct kpz_sim kpz_sim;     /* opaque */
typedef struct lanes_sim lanes_sim; /* opaque */

/* Eq. 8: a site is "slow" with probability prob_slow_*, independently per site and sample
 * (DESIGN §R8); slow sites use p_slow / q_slow instead of p / q. */
typedef struct {
  double prob_slow_p;
  double p_slow;
  double prob_slow_q;
  double q_slow;
} kpz_disorder;

typedef struct {
  int32_t first_sample; /* global index of sample 0 of this handle (part of the RNG key); default 0 */
  int32_t offset_mode;  /* 0 = sub-lattice offset drawn per pass, 1 = alternating 0,1 */
  int32_t path;         /* 0 auto, 1 on-chip per-sample kernel (K1), 2 streamed pass by pass (K3), 3 streamed in
                           temporally blocked chunks (K3T); auto = 1 up to 262144 sites per ring, else 3 */
} kpz_options;

#define KPZ_PATH_AUTO 0
#define KPZ_PATH_ONCHIP 1
#define KPZ_PATH_STREAM 2
#define KPZ_PATH_BLOCKED 3
#define KPZ2D_PATH_CLUSTER 3 /* kpz2d_* only: a sample on chip, spread over a thread-block cluster (K5C) */

/* ---- KPZ / ASEP ring ensemble ----------------------------------------------------------------------------- */

/* Bytes of device workspace kpz_create needs for these sizes (max_records = capacity of the record list). */
int kpz_workspace_bytes(int64_t L, int32_t nsamples, const kpz_disorder* disorder, const kpz_options* opt,
                        int32_t max_records, size_t* bytes);

/* Create an ensemble of nsamples rings of L sites: flat start n_i = i & 1, rates p (forward) and
 * q (backward), optional disorder (NULL = none), Philox key = seed.  d_workspace: device memory of at least
 * kpz_workspace_bytes(...) bytes, 256-byte aligned.  cuda_stream: a cudaStream_t (NULL = default stream).
 * Enqueues the initialisation kernels; does not sync. */
int kpz_create(kpz_sim** out, int64_t L, int32_t nsamples, double p, double q, const kpz_disorder* disorder,
               uint64_t seed, const kpz_options* opt, int32_t max_records, void* d_workspace, size_t workspace_bytes,
               void* cuda_stream);

/* Record times (host array): strictly increasing absolute MCS counts, t[0] > current time, nt <= max_records
 * (DESIGN §R7).  Replaces the list and clears captured records. */
int kpz_set_record_times(kpz_sim*, const int64_t* t, int32_t nt);

/* Advance every sample by n_mcs Monte-Carlo steps (one MCS = two sub-lattice passes), capturing
 * (sum h, sum h^2) per sample at every record time passed.  Asynchronous on the stream.
 * run(a); run(b) is bit-identical to run(a+b). */
int kpz_run(kpz_sim*, int64_t n_mcs);

/* MCS done so far: "when all sites are updated once the time (t) is incremented by one Monte Carlo step"
 * (DESIGN §R10).  Host value; no sync. */
int kpz_time(const kpz_sim*, int64_t* t);

/* Checkpoint restore: continue from MCS count t (0 <= t < 2^54).  Every random number is a function of (seed,
 * sample, MCS index, ...) (§R10), so the lattice (kpz_set_lattice), the disorder tags and t are the whole
 * state.  Drops the record-time list and the captured records; host-side only (no sync). */
int kpz_set_time(kpz_sim*, int64_t t);

/* Back to the state right after kpz_create: flat lattice, disorder tags regenerated from the seed, t = 0,
 * captured records dropped (the record-time list is kept).  Enqueues the initialisation kernels; async. */
int kpz_reset(kpz_sim*);

/* Copy the occupation bits out / in (device buffers, natural layout, nsamples * L/32 words).  Async.
 * The overflow guard of the exact sums (|h| <= 1 + 8 t from the flat start) cannot know how rough a lattice
 * handed in here is: on rings long enough for sum h^2 to leave int64 (L^3 >= 9e18) kpz_set_lattice also measures
 * max |h| on the device, and the next kpz_set_record_times / kpz_run reads it back (one 4-byte copy, syncs once) and
 * refuses record times with KPZ_EUNSUPPORTED as it would after kpz_create. */
int kpz_lattice(kpz_sim*, uint32_t* d_words);
int kpz_set_lattice(kpz_sim*, const uint32_t* d_words);
/* Quenched disorder tags, same layout; either pointer may be NULL.  Async. */
int kpz_disorder_masks(kpz_sim*, uint32_t* d_slow_p, uint32_t* d_slow_q);
int kpz_set_disorder_masks(kpz_sim*, const uint32_t* d_slow_p, const uint32_t* d_slow_q);

/* Heights of one sample: d_h[x] = sum_{i<=x} (2 n_i - 1), x = 0..L-1, L int32 values
 * on the device.  Async. */
int kpz_heights(kpz_sim*, int32_t sample, int32_t* d_h);

/* Records captured so far (host outputs; SYNCS the stream).  nt: in = capacity of the arrays, out = count.
 * t[nt]; sum_h, sum_h2 [nt][nsamples] exact int64 (Eq. 3 sums); w2_mean[nt] = mean over samples of
 * (L*sum_h2 - sum_h^2)/L^2.  Any output pointer may be NULL. */
int kpz_roughness(kpz_sim*, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean);

/* The exact sums behind the width W of Eq. 3 of rings handed in by the caller, WITHOUT any
 * allocation: no handle, no workspace, no cudaMalloc / cudaFree / allocating library call - for callers that cannot
 * allocate (CUDA graph capture, serving loops, harnesses that forbid it).  d_words: nsamples * L/32 device words, natural
 * layout, 16-byte aligned (as kpz_lattice writes them); d_sum_h, d_sum_h2: nsamples device int64 each, overwritten with
 * sum_x h_x and sum_x h_x^2, h_x = sum_{i<=x} (2 n_i - 1) - the values kpz_roughness reports for the same lattice.  They
 * are exact modulo 2^64, hence exact whenever L * max|h|^2 < 2^63 (any lattice with L < 2^21; rougher, longer rings are the
 * caller's to bound, cf. the guard of kpz_set_lattice).  Asynchronous on cuda_stream (a cudaStream_t of the CURRENT device).
 * The tile scratch of the reduction (one int per 65536 sites) is a static device array of KPZ_NOALLOC_MAX_TILES ints
 * (256 KiB per GPU that loads the library, until exit): nsamples * ceil(L / 65536) beyond that, L beyond 2^30 or not a
 * multiple of 64 -> KPZ_EUNSUPPORTED with the reason in kpz_last_error().  ALL calls share that array: two calls that
 * overlap on the GPU (different streams or host threads without an ordering between them) race; calls on one stream
 * are safe back to back. */
#define KPZ_NOALLOC_MAX_TILES 65536
int kpz_noalloc_height_sums(const uint32_t* d_words, int64_t L, int32_t nsamples, int64_t* d_sum_h, int64_t* d_sum_h2,
                            void* cuda_stream);

/* Frees the host-side handle only ("device memory is touched at the start and the end of a time loop", PAPER.md:91:
 * the state lives in the caller's workspace, which the caller frees).  Pending work on the stream is not waited for. */
int kpz_destroy(kpz_sim*);

/* ---- two-lane opposite-direction model -------------------------------------------------- */

int lanes_workspace_bytes(int64_t L, int32_t nsamples, int32_t max_records, size_t* bytes);

/* Two rings of L sites per sample; lane A hops right with p_a, lane B hops left with p_b under the same
 * sub-lattice schedule; initial occupation Bernoulli(rho0) per site per lane; each site is a turning point with
 * probability turn_prob, redrawn every turn_period MCS (0 = never); at a turning point a particle changes lane
 * with probability omega if the target site is empty. */
int lanes_create(lanes_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0, double turn_prob,
                 int64_t turn_period, double omega, uint64_t seed, const kpz_options* opt, int32_t max_records,
                 void* d_workspace, size_t workspace_bytes, void* cuda_stream);
/* The paper's own two-lane model: EVERY site can be crossed - with probability
 * w_flagged where the site's flag is set and w_unflagged elsewhere (the paper: flags set with probability 1/2, crossing
 * "reduced from 0.8 to 0.2" at flagged sites, in-lane p = 0.5, half filling).  independent = 1: the A->B crossings read
 * the flags u_i, the B->A crossings their own set v_i; 0: one set for both.  Flags are redrawn every turn_period MCS
 * (0 = quenched).  lanes_create is the case {turn_prob, omega, 0, 0}.  Runs on the run-time specialised kernel
 * (L <= 131072); lanes_run returns KPZ_EUNSUPPORTED otherwise. */
typedef struct {
  double prob_flag;
  double w_flagged;
  double w_unflagged;
  int32_t independent;
} lanes_crossing;
int lanes_create_crossing(lanes_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                          const lanes_crossing* crossing, int64_t turn_period, uint64_t seed, const kpz_options* opt,
                          int32_t max_records, void* d_workspace, size_t workspace_bytes, void* cuda_stream);
/* Flag sets u (A->B) and v (B->A) of the current epoch (device, natural layout; NULL = skip; v = u unless
 * independent, and lanes_set_flags then takes the one set as d_u).  Async. */
int lanes_flags(lanes_sim*, uint32_t* d_u, uint32_t* d_v);
int lanes_set_flags(lanes_sim*, const uint32_t* d_u, const uint32_t* d_v);
/* Record times of the currents, "sampling ... done in the same way as in case of ASEP simulations (7)" (PAPER.md:275,
 * 134): as kpz_set_record_times. */
int lanes_set_record_times(lanes_sim*, const int64_t* t, int32_t nt);
/* Advance by n_mcs sweeps of the five-part sequence of PAPER.md:259-265: in-lane pass of both lanes,
 * A->B changes, second in-lane pass with the ring closure, B->A changes; hop counters, records and the
 * epoch-end profile (§R16) are updated in the kernel.  Asynchronous; run(a); run(b) == run(a+b). */
int lanes_run(lanes_sim*, int64_t n_mcs);
int lanes_time(const lanes_sim*, int64_t* t); /* sweeps done so far; host value */
/* As kpz_set_time; restore lanes and turning-point mask with lanes_set_state.  Hop counters and profile keep going. */
int lanes_set_time(lanes_sim*, int64_t t);
int lanes_reset(lanes_sim*); /* as kpz_reset: initial occupations, epoch-0 turning points, zero counters; async */
/* Occupations of lanes A, B and the current turning-point mask (device, natural layout, any may be NULL). Async. */
int lanes_state(lanes_sim*, uint32_t* d_a, uint32_t* d_b, uint32_t* d_turn);
int lanes_set_state(lanes_sim*, const uint32_t* d_a, const uint32_t* d_b, const uint32_t* d_turn);
/* Hop counts J_A, J_B and lane populations at the record times (host; SYNCS). */
int lanes_currents(lanes_sim*, int32_t* nt, int64_t* t, int64_t* j_a, int64_t* j_b, int64_t* n_a, int64_t* n_b);
/* Epoch-end occupancy counts [nsamples][L] per lane (device, uint32) and the snapshot count. SYNCS. */
int lanes_profile(lanes_sim*, uint32_t* d_occ_a, uint32_t* d_occ_b, int64_t* nsnap);
int lanes_destroy(lanes_sim*); /* as kpz_destroy: host-side handle only */

/* ---- 2+1D generalisation ------------------------------------- */
/* "We used two-sub-lattice updates, which can be generalized to checker-board lattice decomposition in two dimensions"
 * (PAPER.md:289), towards the 2+1D simulations of refs. [7, 28]: the dimer / octahedron move on a periodic
 * Lx x Ly lattice.  Slopes as bits, sx[y][x] = 1 iff h(x,y) - h(x-1,y) = +1, sy[y][x] = 1 iff h(x,y) - h(x,y-1) = +1; site
 * (x,y) moves forward with probability p when its x-pair (sx[y][x], sx[y][x+1]) and its y-pair (sy[y][x], sy[y+1][x]) are
 * both (1,0) - both become (0,1) - and backward with q when both are (0,1).  One MCS = two colour passes of the
 * checkerboard, sites with (x + y + o) even, o drawn per pass as in the 1+1D sweep (or o = pass with offset_mode 1); the
 * j-th active site of row y draws element y * Lx/2 + j of stream PAIR.  Flat start h = (x + y) & 1.
 * Layout of every slope buffer (device): [nsamples][Ly][Lx/32] uint32, bit (x & 31) of word x >> 5 of row y.
 * Lx a multiple of 64, Ly even, Lx, Ly <= 32768, Lx * Ly <= 2^30.  Ownership, streams and error codes as above. */
typedef struct kpz2d_sim kpz2d_sim;
int kpz2d_workspace_bytes(int32_t Lx, int32_t Ly, int32_t nsamples, int32_t max_records, size_t* bytes);
int kpz2d_create(kpz2d_sim** out, int32_t Lx, int32_t Ly, int32_t nsamples, double p, double q, uint64_t seed,
                 const kpz_options* opt /* first_sample, offset_mode, path: see kpz2d_path */, int32_t max_records, void* d_workspace,
                 size_t workspace_bytes, void* cuda_stream);
int kpz2d_set_record_times(kpz2d_sim*, const int64_t* t, int32_t nt); /* as kpz_set_record_times */
/* n_mcs checkerboard sweeps (see kpz2d_path); captures (sum h, sum h^2) over the Lx * Ly heights
 * h(x,0) = sum_{i<=x} (2 sx[0][i] - 1), h(x,y) = h(x,y-1) + 2 sy[y][x] - 1 at the record times.  Asynchronous. */
int kpz2d_run(kpz2d_sim*, int64_t n_mcs);
int kpz2d_time(const kpz2d_sim*, int64_t* t);
/* 1 = a whole sample in the shared memory of one CTA, one persistent launch per kpz2d_run (auto up to 96 KiB of slopes
 * per sample, e.g. 512 x 512; options.path = 1 forces it up to 200 KiB); 3 (KPZ2D_PATH_CLUSTER) = a sample spread over
 * the shared memories of a thread-block cluster of 2, 4, 8 or 16 CTAs, neighbour rows through distributed shared memory,
 * one persistent launch (auto beyond 96 KiB when Lx is a multiple of 256 and the rows divide, up to 1600 KiB per sample,
 * e.g. 1024 x 1024 on 8 CTAs, 2048 x 2048 on 16 - the non-portable cluster size, used when the device says it can hold
 * one; run-time specialised kernels only); 2 = one in-place launch per colour pass (everything else), consecutive passes
 * launched with programmatic dependent launch. */
int kpz2d_path(const kpz2d_sim*, int32_t* path);
int kpz2d_reset(kpz2d_sim*);                                          /* flat surface, t = 0, records dropped; async */
int kpz2d_slopes(kpz2d_sim*, uint32_t* d_sx, uint32_t* d_sy);        /* copy out (either may be NULL); async */
/* Copy in.  The two fields must describe a single-valued surface (every plaquette curl-free: sx[y][x] + sy[y+1][x] =
 * sx[y+1][x] + sy[y+1][x-1], both ways round a plaquette give the same height), as every state reached from the flat start
 * does: the sums captured at record times integrate the heights row by row, kpz2d_heights column by column, and the
 * two agree exactly on such surfaces only. */
int kpz2d_set_slopes(kpz2d_sim*, const uint32_t* d_sx, const uint32_t* d_sy);
int kpz2d_heights(kpz2d_sim*, int32_t sample, int32_t* d_h /* [Ly][Lx] int32, device */);
/* As kpz_roughness: W^2 over the Lx * Ly sites of a sample (Eq. 3), mean over samples.  SYNCS. */
int kpz2d_roughness(kpz2d_sim*, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean);
int kpz2d_destroy(kpz2d_sim*);

/* ---- diagnostics ------------------------------------------------------------------------------------------ */
/* Text of an error code.  The paper's programs report nothing of the kind; this serves the "no exception or abort
 * crosses the ABI" rule of SURVEY §8(b). */
const char* kpz_strerror(int code);
const char* kpz_last_error(void);        /* thread-local detail of the last failing call */
int64_t kpz_kernel_launches(void);       /* kernels launched by this library in this process so far */
/* Which kernel family a handle's kpz_run uses: 1 = on-chip per-sample (K1), 2 = streamed (K3), 3 = blocked (K3T). */
int kpz_path(const kpz_sim*, int32_t* path);

/* Test and tuning hook, not part of the paper's problem statement: a ';'-separated list of NAME=VALUE items that
 * replaces the process-wide debug configuration (NULL or "" restores the defaults).  "jit=0" selects the statically
 * compiled generic kernels instead of the run-time specialised ones; "K1J_<X>=v" / "K4J_<X>=v" / "K5J_<X>=v" are appended
 * as definitions to every later run-time compilation of the KPZ / two-lane / 2+1D sweep kernels (the knobs documented at
 * the top of csrc/k1_sweep_jit.cuh and csrc/k4_lanes_jit.cuh; 2+1D: K5J_RIW=0 no shuffles, K5J_PIPE=0 no software
 * pipeline in the on-chip kernel, K5J_CS=2|4|8|16 cluster size, K5J_NBR=1 neighbour-only barriers, K5J_DUAL=1 two samples per cluster, K5J_PDL=0 no programmatic dependent launch of the streamed passes, K5J_XRALL=1 every warp
 * through shared::cluster addresses in the cluster kernel).  Every setting computes the same results (tests/ check that);
 * kpz_run / lanes_run read no environment variable.  KPZ_EINVAL for anything else. */
int kpz_debug_config(const char* spec);
/* Writes every kernel image compiled by this process so far (kpz_run, lanes_run, *_jit_check) to
 * <dir>/<entry>_<n>.cubin with its definition list in <dir>/<entry>_<n>.txt, for `cuobjdump -sass` (the instruction
 * census behind DESIGN §6.1).  count (may be NULL) receives the number of images.  Host-side only. */
int kpz_debug_dump_cubins(const char* dir, int32_t* count);

/* The on-chip sweep kernel is specialised at run time (NVRTC) on the ring size and the acceptance thresholds
 * (DESIGN §5); kpz_debug_config("jit=0") selects the statically compiled generic kernels instead.
 * kpz_jit_check compiles - without loading, so it needs no GPU - the kernel kpz_run would use for these parameters
 * and returns the size of its sm_100a cubin (0 when that configuration runs on a statically compiled kernel). */
int kpz_jit_check(int64_t L, double p, double q, const kpz_disorder* disorder, const kpz_options* opt,
                  size_t* cubin_bytes);
int lanes_jit_check(int64_t L, double p_a, double p_b, double turn_prob, int64_t turn_period, double omega,
                    const kpz_options* opt, size_t* cubin_bytes); /* same for the two-lane kernel */
int lanes_crossing_jit_check(int64_t L, double p_a, double p_b, const lanes_crossing* crossing, int64_t turn_period,
                             const kpz_options* opt, size_t* cubin_bytes);
/* Same for the 2+1D kernels (K5 / K5S / K5C, specialised on Lx, Ly and the thresholds of p, q): the kernel kpz2d_run would use
 * for these parameters and options.path. */
int kpz2d_jit_check(int32_t Lx, int32_t Ly, double p, double q, const kpz_options* opt, size_t* cubin_bytes);

#ifdef __cplusplus
}
#endif
#endif
