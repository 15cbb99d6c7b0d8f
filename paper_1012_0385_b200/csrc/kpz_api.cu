// kpz_api.cu — host side of the KPZ/ASEP ring ensemble: the kpz_* entry points of include/kpz_b200.h.
// Validation, workspace carving, kernel dispatch.  Every step of the path runs in the kernels; this file only
// launches them.  There is no CPU fallback: without a CUDA device every call that needs one fails with KPZ_ECUDA.
#include <algorithm>
#include <atomic>
#include <cstdlib>
#include <cstring>
#include <string>
#include <new>
#include <vector>

#include "common.cuh"
#include "jit.h"
#include "kpz_k1.cuh"
#include "kpz_k3.cuh"
#include "kpz_util.cuh"

namespace kpz {

// ---- error plumbing ------------------------------------------------------------------------------------
static thread_local char g_err[512] = "";
static std::atomic<long long> g_launches{0};

void set_error(const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
}
int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}
void count_launch(int n) { g_launches += n; }

static int grid_for(size_t n, int block = 256) {
  size_t g = (n + block - 1) / block;
  return (int)std::min<size_t>(std::max<size_t>(g, 1), 148 * 16);
}

}  // namespace kpz

using namespace kpz;

struct kpz_sim {
  int64_t L = 0;
  int32_t S = 0;
  int32_t max_records = 0;
  int32_t path = 0;  // 1 = K1, 2 = K3
  bool has_disorder = false, has_sp = false, has_sq = false;
  bool has_sp0 = false, has_sq0 = false;  // as created (kpz_reset restores them)
  kpz_disorder dis{};
  KpzDev dev{};
  cudaStream_t stream = nullptr;
  // workspace carve-up (device)
  uint32_t *E = nullptr, *O = nullptr, *E2 = nullptr, *O2 = nullptr;
  uint32_t *SPE = nullptr, *SPO = nullptr, *SQE = nullptr, *SQO = nullptr;
  long long *rec_t = nullptr, *rec_sum_h = nullptr, *rec_sum_h2 = nullptr;
  int* scratch = nullptr;
  size_t scratch_ints = 0;
  unsigned char* k3off = nullptr;  // [(chunk+1)][S] offsets of a chunk of passes; row 0 = frame of the stored lattice
  int* tiles = nullptr;            // [S][ntiles]
  int ntiles = 0;
  // host state
  int64_t t = 0;
  int frame = 0;  // K3: frame of the stored lattice (always 0 between calls)
  std::vector<int64_t> rec_times;
  int32_t nrec = 0;  // records captured (times <= t)
  // overflow guard of the exact sums: |h| <= min(L, h0 + 8 (t - t_h0)); flat start: h0 = 1, t_h0 = 0
  int64_t h0 = 1, t_h0 = 0;
  bool h0_pending = false;  // h0 is being measured on the device (kpz_set_lattice on a ring long enough to overflow)
  bool guard_checked = true;  // the current record-time list has been checked against the current (h0, t_h0)
};

namespace {

constexpr int kK3ChunkPasses = 4096;  // offsets are drawn for this many passes at a time

struct Layout {
  size_t off_E, off_O, off_E2, off_O2, off_SPE, off_SPO, off_SQE, off_SQO, off_rec_t, off_h, off_h2, off_scratch, total;
  size_t off_k3off, off_tiles;
  int PW, PWp, U, ntiles;
  size_t scratch_ints;
};

int choose_path(int64_t L, const kpz_options* opt, int* path) {
  const int64_t U = (L / 64 + 3) / 4;
  int want = opt ? opt->path : KPZ_PATH_AUTO;
  if (want == KPZ_PATH_AUTO) want = (U <= 1024) ? KPZ_PATH_ONCHIP : (jit_enabled() ? KPZ_PATH_BLOCKED : KPZ_PATH_STREAM);
  if (want == KPZ_PATH_ONCHIP && U > 1024)
    return fail(KPZ_EUNSUPPORTED, "on-chip path holds at most 262144 sites per sample (L=%lld)", (long long)L);
  if (want != KPZ_PATH_ONCHIP && want != KPZ_PATH_STREAM && want != KPZ_PATH_BLOCKED)
    return fail(KPZ_EINVAL, "options.path must be 0, 1, 2 or 3");
  if (want == KPZ_PATH_BLOCKED && !jit_enabled())
    return fail(KPZ_EUNSUPPORTED, "the blocked streamed path is compiled at run time (kpz_debug_config(\"jit=0\") disables it)");
  *path = want;
  return KPZ_OK;
}

int validate_sizes(int64_t L, int32_t S, int32_t max_records) {
  if (L < 4 || (L & 1) || S < 1 || max_records < 0) return fail(KPZ_EINVAL, "need even L >= 4, nsamples >= 1, max_records >= 0");
  if (L % 64 != 0) return fail(KPZ_EUNSUPPORTED, "the CUDA path needs L to be a multiple of 64 (L=%lld)", (long long)L);
  if (L > ((int64_t)1 << 36)) return fail(KPZ_EUNSUPPORTED, "L too large");
  if ((L / 64) * (int64_t)S > ((int64_t)1 << 31) - 8) return fail(KPZ_EUNSUPPORTED, "nsamples * L too large");
  return KPZ_OK;
}

Layout make_layout(int64_t L, int32_t S, bool disorder, int path, int32_t max_records) {
  Layout y{};
  y.PW = (int)(L / 64);
  y.PWp = (y.PW + 3) / 4 * 4;
  y.U = y.PWp / 4;
  const size_t plane = align_up((size_t)S * y.PWp * 4, 256);
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off += align_up(bytes, 256);
    return o;
  };
  y.off_E = take(plane);
  y.off_O = take(plane);
  y.off_E2 = y.off_O2 = 0;
  if (path == KPZ_PATH_STREAM || path == KPZ_PATH_BLOCKED) {
    y.off_E2 = take(plane);
    y.off_O2 = take(plane);
  }
  y.off_SPE = y.off_SPO = y.off_SQE = y.off_SQO = 0;
  if (disorder) {
    y.off_SPE = take(plane);
    y.off_SPO = take(plane);
    y.off_SQE = take(plane);
    y.off_SQO = take(plane);
  }
  y.off_rec_t = take((size_t)std::max(max_records, 1) * 8);
  y.off_h = take((size_t)std::max(max_records, 1) * S * 8);
  y.off_h2 = take((size_t)std::max(max_records, 1) * S * 8);
  y.scratch_ints = (size_t)y.PW + 8192;
  y.off_scratch = take(y.scratch_ints * 4);
  y.ntiles = (y.U + 255) / 256;
  y.off_k3off = y.off_tiles = 0;
  if (path == KPZ_PATH_STREAM || path == KPZ_PATH_BLOCKED) {
    y.off_k3off = take((size_t)(kK3ChunkPasses + 1) * S);
    y.off_tiles = take((size_t)S * y.ntiles * 4);
  }
  y.total = off;
  return y;
}

// ---- K1 dispatch ---------------------------------------------------------------------------------------
using K1Fn = void (*)(const KpzDev, const KpzRunArgs);

template <bool SW, bool PARTIAL, int DIS>
K1Fn k1_pick_nps(int nps) {
  if (PARTIAL) return kpz_k1_kernel<SW, PARTIAL, DIS, -1>;
  switch (nps) {
    case 0: return kpz_k1_kernel<SW, false, DIS, 0>;
    case 1: return kpz_k1_kernel<SW, false, DIS, 1>;
    case 2: return kpz_k1_kernel<SW, false, DIS, 2>;
    default: return kpz_k1_kernel<SW, false, DIS, -1>;
  }
}
template <bool SW, bool PARTIAL>
K1Fn k1_pick_dis(int dis, int nps) {
  switch (dis) {
    case 0: return k1_pick_nps<SW, PARTIAL, 0>(nps);
    case 1: return k1_pick_nps<SW, PARTIAL, 1>(nps);
    default: return k1_pick_nps<SW, PARTIAL, 2>(nps);
  }
}
K1Fn k1_pick(bool single_warp, bool partial, int dis, int nps) {
  if (single_warp) return partial ? k1_pick_dis<true, true>(dis, nps) : k1_pick_dis<true, false>(dis, nps);
  return partial ? k1_pick_dis<false, true>(dis, nps) : k1_pick_dis<false, false>(dis, nps);
}

// ---- K1 v2: the sweep specialised at run time on (L, thresholds, tags, offset mode) — k1_sweep_jit.cuh ----------
// Every threshold set runs on it: up to three selection inputs fold into one LOP3, anything else (tags + planes,
// non-dyadic rates) takes its GENERAL path with eagerly drawn leading planes and a lazy tail.
std::vector<std::string> k1_jit_defines(const KpzDev& D, int dis) {
  auto T = [&](int c) -> unsigned long long {
    return D.thr[c].always ? (1ull << 32) : (unsigned long long)D.thr[c].value;
  };
  char buf[64];
  std::vector<std::string> d;
  snprintf(buf, sizeof buf, "K1J_PW=%d", D.PW);
  d.push_back(buf);
  for (int c = 0; c < 4; ++c) {
    // classes a kernel variant never reads are normalised so that equal kernels share one cache entry
    unsigned long long t = T(c);
    if ((c == 1 && dis < 1) || (c == 3 && dis < 2)) t = 0;
    snprintf(buf, sizeof buf, "K1J_T%d=0x%llxull", c, t);
    d.push_back(buf);
  }
  snprintf(buf, sizeof buf, "K1J_DIS=%d", dis);
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K1J_OFFSET_MODE=%d", D.offset_mode);
  d.push_back(buf);
  debug_defines("K1J_", &d);  // kpz_debug_config: tests and tuning only (the run reads no environment)
  return d;
}

bool k1_use_jit(const KpzDev&) { return jit_enabled(); }

// The streamed kernels keep one unit per thread whatever the debug configuration says.
void drop_define(std::vector<std::string>* defs, const char* name) {
  const std::string key = std::string(name) + "=";
  defs->erase(std::remove_if(defs->begin(), defs->end(),
                             [&](const std::string& d) { return d.compare(0, key.size(), key) == 0; }),
              defs->end());
}

// Launch shape of the per-sample kernel (k1_sweep_jit.cuh): definitions, block size, samples per warp.
struct K1Shape {
  std::vector<std::string> defs;
  int block = 32, spw = 1, upt = 1;
  int queue = 0;  // K1J_QUEUE: MCS per work item (0 = one CTA per sample for the whole run)
  int grid = 1;
};
constexpr int kQueueMaxSamples = 8000;  // the done flags live in the scratch area behind the group totals

K1Shape k1_shape(const KpzDev& D, int S, int dis, long long n_mcs = 1LL << 40) {
  static int smsp = 0;
  if (!smsp) {
    int dev = 0, sms = 148;
    if (cudaGetDevice(&dev) == cudaSuccess) cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
    smsp = 4 * sms;
  }
  K1Shape sh;
  const bool partial = (D.PW % 4) != 0;
  // units per thread (K1J_UPT, k1_sweep_jit.cuh): 2 gives a ring of 64 units to ONE warp - no barrier, two independent
  // chains of pair logic per thread.  Measured (profiles/r02_k1_upt.md): no gain at BASELINE's 512 rings of 16384
  // sites (a lone warp per SMSP stays latency-bound), +8 % with K1J_VARIANT=2 once 1184 rings fill the chip, and a loss
  // on the lazily evaluated path (twice the registers, same trips) - so the default stays 1; the knob is kept for tests.
  sh.upt = debug_int("K1J_UPT", 1);
  if (sh.upt < 1 || sh.upt > 2 || partial || D.U % sh.upt != 0) sh.upt = 1;
  const int UT = D.U / sh.upt;
  sh.block = (UT + 31) / 32 * 32;
  // small rings (SPW): UT <= 16 threads, a power of two, no ragged unit -> 32/UT samples per warp
  // (measured: packing never loses - a 30-ring launch runs at the same 17 GSU/s packed or one ring per warp)
  const bool pack = UT <= 16 && (UT & (UT - 1)) == 0 && !partial;
  sh.spw = pack ? 32 / UT : 1;
  sh.defs = k1_jit_defines(D, dis);
  char buf[32];
  drop_define(&sh.defs, "K1J_UPT");  // the value clamped above, not the raw debug setting
  snprintf(buf, sizeof buf, "K1J_UPT=%d", sh.upt);
  sh.defs.push_back(buf);
  if (!pack) sh.defs.push_back("K1J_PACK=0");
  if (!debug_has("K1J_VARIANT")) {
    // code shape by occupancy (k1_sweep_jit.cuh, K1J_VARIANT): with >= 4 resident warps per SMSP the other warps
    // hide the latency, so the shape with the fewest alu slots wins (measured: +12..16 % on 16384-site rings)
    const long long warps = (long long)((S + sh.spw - 1) / sh.spw) * (sh.block / 32);
    if (warps >= 4LL * smsp) sh.defs.push_back("K1J_VARIANT=2");
  }
  // Work queue (K1J_QUEUE = MCS per item, K1J_QGRID = CTAs in percent of the rings; k1_sweep_jit.cuh): chunks pulled from a
  // counter let CTAs on emptier SMSPs run more of them.  Measured (profiles/r02_summary.md 3): config 2 -12 % (rings are
  // chains, so a CTA that runs ahead ends up waiting for the chunk in front of it), config 3 +2 ... +4 % with chunks of
  // 1024 MCS and 16 % spare CTAs: inside the run-to-run spread, so the default is off; the knob is kept for tests.
  const long long warps = (long long)((S + sh.spw - 1) / sh.spw) * (sh.block / 32);
  (void)warps;
  (void)n_mcs;
  int q = 0;
  q = debug_int("K1J_QUEUE", q);
  if (sh.spw != 1 || S > kQueueMaxSamples || q < 0) q = 0;
  sh.queue = q;
  drop_define(&sh.defs, "K1J_QUEUE");
  drop_define(&sh.defs, "K1J_QGRID");
  snprintf(buf, sizeof buf, "K1J_QUEUE=%d", q);
  sh.defs.push_back(buf);
  const int nblocks = (S + sh.spw - 1) / sh.spw;
  sh.grid = nblocks;
  if (q > 0) sh.grid = std::max(1, std::min(2 * nblocks, (int)((long long)nblocks * debug_int("K1J_QGRID", 100) / 100)));
  return sh;
}

void refresh_planes(kpz_sim* sim) {
  int np = std::max(planes_needed(sim->dev.thr[0]), planes_needed(sim->dev.thr[2]));
  if (sim->has_sp) np = std::max(np, planes_needed(sim->dev.thr[1]));
  if (sim->has_sq) np = std::max(np, planes_needed(sim->dev.thr[3]));
  sim->dev.nplanes = np;
  sim->dev.SPE = sim->has_sp || sim->has_sq ? sim->SPE : nullptr;
  sim->dev.SPO = sim->has_sp || sim->has_sq ? sim->SPO : nullptr;
  sim->dev.SQE = sim->has_sq ? sim->SQE : nullptr;
  sim->dev.SQO = sim->has_sq ? sim->SQO : nullptr;
}


// a1: flat start and the quenched disorder tags (Eq. 8) — the kernels kpz_create and kpz_reset enqueue.
int init_state(kpz_sim* sim) {
  const KpzDev& D = sim->dev;
  const size_t nwords = (size_t)D.S * D.PWp;
  k_init_flat<<<grid_for(nwords), 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.PW, D.PWp);
  KPZ_LAUNCH_CHECK("k_init_flat");
  if (sim->has_disorder) {
    const size_t ng = (size_t)D.S * ((D.PW + 1) / 2);
    if (D.PWp != D.PW) {  // pad words of the mask rows must be zero
      for (uint32_t* m : {sim->SPE, sim->SPO, sim->SQE, sim->SQO}) {
        k_zero_words<<<grid_for(nwords), 256, 0, sim->stream>>>(m, nwords);
        KPZ_LAUNCH_CHECK("k_zero_words");
      }
    }
    k_site_mask_eo<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_SLOW_P, make_thresh(sim->dis.prob_slow_p),
                                                              D.first_sample, D.S, D.PW, D.PWp, sim->SPE, sim->SPO);
    KPZ_LAUNCH_CHECK("k_site_mask_eo");
    k_site_mask_eo<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_SLOW_Q, make_thresh(sim->dis.prob_slow_q),
                                                              D.first_sample, D.S, D.PW, D.PWp, sim->SQE, sim->SQO);
    KPZ_LAUNCH_CHECK("k_site_mask_eo");
  }
  return KPZ_OK;
}

// ---- K3 dispatch and driver ------------------------------------------------------------------------------
using K3Fn = void (*)(const KpzDev, const K3Pass);

template <bool PARTIAL, int DIS>
K3Fn k3_pick_nps(int nps) {
  if (PARTIAL) return k3_pass_kernel<PARTIAL, DIS, -1>;
  switch (nps) {
    case 0: return k3_pass_kernel<false, DIS, 0>;
    case 1: return k3_pass_kernel<false, DIS, 1>;
    case 2: return k3_pass_kernel<false, DIS, 2>;
    default: return k3_pass_kernel<false, DIS, -1>;
  }
}
template <bool PARTIAL>
K3Fn k3_pick_dis(int dis, int nps) {
  switch (dis) {
    case 0: return k3_pick_nps<PARTIAL, 0>(nps);
    case 1: return k3_pick_nps<PARTIAL, 1>(nps);
    default: return k3_pick_nps<PARTIAL, 2>(nps);
  }
}

// "K1J_PDL=0" (kpz_debug_config) launches consecutive passes of the streamed kernel without programmatic dependent launch
bool k3_pdl() { return debug_int("K1J_PDL", 1) != 0; }

int k3_launch_pass(kpz_sim* sim, K3Fn fn, void* jitfn, const unsigned char* fin, const unsigned char* fo, long long m,
                   int pass) {
  KpzDev D = sim->dev;
  K3Pass A{};
  A.Ein = sim->E;
  A.Oin = sim->O;
  A.Eout = sim->E2;
  A.Oout = sim->O2;
  A.fin = fin;
  A.fo = fo;
  A.m = m;
  A.pass = pass;
  const size_t nunits = (size_t)D.S * D.U;
  if (jitfn) {
    void* args[] = {(void*)&D, (void*)&A};
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = dim3((unsigned)((nunits + 255) / 256));
    cfg.blockDim = dim3(256);
    cfg.stream = sim->stream;
    cudaLaunchAttribute at{};
    at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at.val.programmaticStreamSerializationAllowed = 1;  // the next pass may start to launch while this one runs (K1J_PDL)
    cfg.attrs = &at;
    cfg.numAttrs = k3_pdl() ? 1 : 0;
    KPZ_CUDA_CHECK(cudaLaunchKernelExC(&cfg, jitfn, args));
  } else {
    fn<<<(unsigned)((nunits + 255) / 256), 256, 0, sim->stream>>>(D, A);
  }
  KPZ_LAUNCH_CHECK("k3_pass_kernel");
  std::swap(sim->E, sim->E2);
  std::swap(sim->O, sim->O2);
  sim->dev.E = sim->E;
  sim->dev.O = sim->O;
  return KPZ_OK;
}

int k3_record(kpz_sim* sim, int ri) {
  const KpzDev& D = sim->dev;
  const bool partial = (D.PW % 4) != 0;
  const int nt = sim->ntiles;
  unsigned long long* oh = (unsigned long long*)(sim->rec_sum_h + (size_t)ri * D.S);
  unsigned long long* oh2 = (unsigned long long*)(sim->rec_sum_h2 + (size_t)ri * D.S);
  KPZ_CUDA_CHECK(cudaMemsetAsync(oh, 0, (size_t)D.S * 8, sim->stream));
  KPZ_CUDA_CHECK(cudaMemsetAsync(oh2, 0, (size_t)D.S * 8, sim->stream));
  if (partial) k3_tile_totals<true><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles);
  else k3_tile_totals<false><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles);
  KPZ_LAUNCH_CHECK("k3_tile_totals");
  k3_scan_tiles<<<D.S, 1024, 0, sim->stream>>>(sim->tiles, nt);
  KPZ_LAUNCH_CHECK("k3_scan_tiles");
  if (partial) k3_tile_sums<true><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles, oh, oh2);
  else k3_tile_sums<false><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles, oh, oh2);
  KPZ_LAUNCH_CHECK("k3_tile_sums");
  return KPZ_OK;
}

// The stored lattice is in frame 0 on entry and on exit.  Inside, the frame of each sample follows its offsets;
// row r of k3off holds the offsets of pass (chunk start + r - 1), row 0 the frame the chunk starts in.
int k3_run(kpz_sim* sim, int64_t n_mcs) {
  const KpzDev& D0 = sim->dev;
  const int S = D0.S;
  const bool partial = (D0.PW % 4) != 0;
  const int dis = sim->has_sq ? 2 : sim->has_sp ? 1 : 0;
  K3Fn fn = partial ? k3_pick_dis<true>(dis, D0.nplanes) : k3_pick_dis<false>(dis, D0.nplanes);
  void* jitfn = nullptr;  // the same pass specialised on (L, thresholds) when run-time compilation is enabled
  if (jit_enabled()) {
    std::vector<std::string> defs = k1_jit_defines(D0, dis);
    drop_define(&defs, "K1J_UPT");
    drop_define(&defs, "K1J_PDL");
    defs.push_back("K1J_STREAM=1");
    defs.push_back(k3_pdl() ? "K1J_PDL=1" : "K1J_PDL=0");
    int rcj = jit_get("k1_sweep_jit.cuh", "kpz_k3_pass_jit", defs, &jitfn);
    if (rcj) return rcj;
  }
  const int nt = (int)sim->rec_times.size();
  int ri = sim->nrec;
  const long long pass_begin = 2 * (long long)sim->t, pass_end = 2 * (long long)(sim->t + n_mcs);
  bool frame_dirty = false;  // some sample may be in frame 1
  const unsigned char* prev_row = nullptr;  // device row with the current frames (nullptr = all zero)
  for (long long c0 = pass_begin; c0 < pass_end; c0 += kK3ChunkPasses) {
    const int np = (int)std::min<long long>(kK3ChunkPasses, pass_end - c0);
    // row 0 := current frames, rows 1..np := offsets
    k3_copy_row<<<grid_for(S), 256, 0, sim->stream>>>(sim->k3off, frame_dirty ? prev_row : nullptr, S);
    KPZ_LAUNCH_CHECK("k3_copy_row");
    k3_offsets<<<grid_for((size_t)np * S), 256, 0, sim->stream>>>(D0.keys, D0.first_sample, S, c0, np, D0.offset_mode,
                                                                 sim->k3off);
    KPZ_LAUNCH_CHECK("k3_offsets");
    // the copy above read prev_row (= last row of this same buffer) before k3_offsets overwrites it only if
    // np rows do not reach it; keep it safe by staging through row 0 first (stream order guarantees it).
    int fin_row = 0;
    for (int k = 0; k < np; ++k) {
      const long long gp = c0 + k;
      const long long m = gp >> 1;
      const int pass = (int)(gp & 1);
      int rc = k3_launch_pass(sim, fn, jitfn, sim->k3off + (size_t)fin_row * S, sim->k3off + (size_t)(k + 1) * S, m, pass);
      if (rc) return rc;
      fin_row = k + 1;
      frame_dirty = true;
      if (pass == 1 && ri < nt && sim->rec_times[ri] == m + 1) {
        // bring every sample to frame 0 (no update), then reduce
        rc = k3_launch_pass(sim, fn, jitfn, sim->k3off + (size_t)fin_row * S, nullptr, m, pass);
        if (rc) return rc;
        // from now on the stored frame is 0: point fin at a zero row (row 0 rewritten to zero)
        k3_copy_row<<<grid_for(S), 256, 0, sim->stream>>>(sim->k3off, nullptr, S);
        KPZ_LAUNCH_CHECK("k3_copy_row");
        fin_row = 0;
        frame_dirty = false;
        rc = k3_record(sim, ri);
        if (rc) return rc;
        ++ri;
      }
    }
    prev_row = sim->k3off + (size_t)fin_row * S;
    if (fin_row == 0) frame_dirty = false;
  }
  if (frame_dirty) {
    int rc = k3_launch_pass(sim, fn, jitfn, prev_row, nullptr, 0, 0);
    if (rc) return rc;
  }
  return KPZ_OK;
}

// ---- K3T: temporally blocked streamed sweep (k1_sweep_jit.cuh, K1J_TILE) --------------------------------------------
// One launch per chunk of up to kK3TChunk MCS (chunks end at record times); the lattice is in frame 0 between launches.
constexpr long long kK3TChunk = 32;

int k3t_run(kpz_sim* sim, int64_t n_mcs) {
  const int dis = sim->has_sq ? 2 : sim->has_sp ? 1 : 0;
  std::vector<std::string> defs = k1_jit_defines(sim->dev, dis);
  drop_define(&defs, "K1J_UPT");
  defs.push_back("K1J_TILE=1");
  void* kfn = nullptr;
  int rc = jit_get("k1_sweep_jit.cuh", "kpz_k3t_sweep_jit", defs, &kfn);
  if (rc) return rc;
  const int nt = (int)sim->rec_times.size();
  int ri = sim->nrec;
  long long t = sim->t;
  const long long t_end = sim->t + n_mcs;
  const long long ntiles = ((long long)sim->dev.U + 29) / 30;
  const long long nwarps = ntiles * sim->S;
  while (t < t_end) {
    long long n = std::min<long long>(kK3TChunk, t_end - t);
    if (ri < nt && sim->rec_times[ri] - t < n) n = sim->rec_times[ri] - t;
    KpzDev D = sim->dev;
    K3TArgs A{};
    A.Eout = sim->E2;
    A.Oout = sim->O2;
    A.t0 = t;
    A.n_mcs = n;
    void* args[] = {(void*)&D, (void*)&A};
    KPZ_CUDA_CHECK(cudaLaunchKernel(kfn, dim3((unsigned)((nwarps + 3) / 4)), dim3(128), args, 0, sim->stream));
    KPZ_LAUNCH_CHECK("kpz_k3t_sweep_jit");
    std::swap(sim->E, sim->E2);
    std::swap(sim->O, sim->O2);
    sim->dev.E = sim->E;
    sim->dev.O = sim->O;
    t += n;
    if (ri < nt && sim->rec_times[ri] == t) {
      rc = k3_record(sim, ri);
      if (rc) return rc;
      ++ri;
    }
  }
  return KPZ_OK;
}

// ---- overflow guard ------------------------------------------------------------------------------
// A pass moves h_x by at most 2 through its own pair and 2 more through the closing pair: |h| grows by <= 8 per MCS.
int guard_record_times(kpz_sim* sim, const int64_t* t, int32_t nt) {
  if (sim->h0_pending) {  // measured by kpz_set_lattice: max |height in front of a unit| + 256
    int v = 0;
    KPZ_CUDA_CHECK(cudaMemcpyAsync(&v, sim->scratch + sim->dev.PW + 16, sizeof(int), cudaMemcpyDeviceToHost, sim->stream));
    KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
    sim->h0 = (int64_t)v + 256;
    sim->h0_pending = false;
  }
  for (int32_t k = 0; k < nt; ++k) {
    if (t[k] <= sim->t) continue;  // already captured
    const long double bound = std::min<long double>((long double)sim->L,
                                                    (long double)sim->h0 + 8.0L * (long double)(t[k] - sim->t_h0));
    if ((long double)sim->L * bound * bound >= 9.0e18L)
      return fail(KPZ_EUNSUPPORTED, "sum of h^2 could overflow int64 at t=%lld for L=%lld", (long long)t[k], (long long)sim->L);
    if (sim->path != KPZ_PATH_ONCHIP && bound >= 2147483647.0L)
      return fail(KPZ_EUNSUPPORTED, "heights could overflow int32 at t=%lld", (long long)t[k]);
  }
  sim->guard_checked = true;
  return KPZ_OK;
}

// A lattice handed in by the caller can be as rough as |h| = L/2: measure it when that could matter.
int measure_h0(kpz_sim* sim) {
  const KpzDev& D = sim->dev;
  sim->t_h0 = sim->t;
  sim->guard_checked = false;
  const long double Lh = (long double)sim->L;
  if (Lh * Lh * Lh < 9.0e18L && (sim->path == KPZ_PATH_ONCHIP || Lh < 2147483647.0L)) {
    sim->h0 = sim->L;  // the trivial bound |h| <= L never overflows on this ring
    sim->h0_pending = false;
    return KPZ_OK;
  }
  // streamed / blocked rings only reach this point (an on-chip ring has L <= 262144): their tile scan gives the height
  // in front of every 256-site unit
  int* slot = sim->scratch + D.PW + 16;  // beyond the PW ints kpz_heights uses
  const int nt = sim->ntiles;
  const bool partial = (D.PW % 4) != 0;
  KPZ_CUDA_CHECK(cudaMemsetAsync(slot, 0, sizeof(int), sim->stream));
  if (partial) k3_tile_totals<true><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles);
  else k3_tile_totals<false><<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.U, D.PW, D.PWp, nt, sim->tiles);
  KPZ_LAUNCH_CHECK("k3_tile_totals");
  k3_scan_tiles<<<D.S, 1024, 0, sim->stream>>>(sim->tiles, nt);
  KPZ_LAUNCH_CHECK("k3_scan_tiles");
  k3_tile_absmax<<<D.S * nt, 256, 0, sim->stream>>>(sim->E, sim->O, D.U, D.PW, D.PWp, nt, sim->tiles, slot);
  KPZ_LAUNCH_CHECK("k3_tile_absmax");
  sim->h0_pending = true;
  return KPZ_OK;
}

}  // namespace

extern "C" {

const char* kpz_strerror(int code) {
  switch (code) {
    case KPZ_OK: return "ok";
    case KPZ_EINVAL: return "invalid argument";
    case KPZ_EUNSUPPORTED: return "unsupported size or configuration";
    case KPZ_ENOMEM: return "workspace or output capacity too small";
    case KPZ_ECUDA: return "CUDA error";
    default: return "unknown error";
  }
}
const char* kpz_last_error(void) { return kpz::g_err; }
int64_t kpz_kernel_launches(void) { return (int64_t)kpz::g_launches.load(); }

int kpz_debug_config(const char* spec) { return kpz::debug_config(spec); }
int kpz_debug_dump_cubins(const char* dir, int32_t* count) {
  int n = 0;
  const int rc = kpz::dump_cubins(dir, &n);
  if (count) *count = n;
  return rc;
}

int kpz_workspace_bytes(int64_t L, int32_t nsamples, const kpz_disorder* disorder, const kpz_options* opt,
                        int32_t max_records, size_t* bytes) {
  if (!bytes) return fail(KPZ_EINVAL, "bytes is NULL");
  int rc = validate_sizes(L, nsamples, max_records);
  if (rc) return rc;
  int path;
  rc = choose_path(L, opt, &path);
  if (rc) return rc;
  *bytes = make_layout(L, nsamples, disorder != nullptr, path, max_records).total;
  return KPZ_OK;
}

int kpz_create(kpz_sim** out, int64_t L, int32_t nsamples, double p, double q, const kpz_disorder* disorder,
               uint64_t seed, const kpz_options* opt, int32_t max_records, void* d_workspace, size_t workspace_bytes,
               void* cuda_stream) {
  if (!out) return fail(KPZ_EINVAL, "out is NULL");
  *out = nullptr;
  int rc = validate_sizes(L, nsamples, max_records);
  if (rc) return rc;
  if (!valid_prob(p) || !valid_prob(q)) return fail(KPZ_EINVAL, "p and q must lie in [0,1]");
  kpz_disorder d{0.0, p, 0.0, q};
  if (disorder) {
    d = *disorder;
    if (!valid_prob(d.prob_slow_p) || !valid_prob(d.p_slow) || !valid_prob(d.prob_slow_q) || !valid_prob(d.q_slow))
      return fail(KPZ_EINVAL, "disorder probabilities must lie in [0,1]");
  }
  kpz_options o{0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1))
    return fail(KPZ_EINVAL, "options: first_sample >= 0, offset_mode in {0,1}");
  int path;
  rc = choose_path(L, &o, &path);
  if (rc) return rc;
  if (!d_workspace) return fail(KPZ_EINVAL, "d_workspace is NULL");
  if (((uintptr_t)d_workspace & 255) != 0) return fail(KPZ_EINVAL, "d_workspace must be 256-byte aligned");
  const Layout y = make_layout(L, nsamples, disorder != nullptr, path, max_records);
  if (workspace_bytes < y.total)
    return fail(KPZ_ENOMEM, "workspace has %zu bytes, %zu needed", workspace_bytes, y.total);

  kpz_sim* sim = new (std::nothrow) kpz_sim();
  if (!sim) return fail(KPZ_ENOMEM, "host allocation failed");
  sim->L = L;
  sim->S = nsamples;
  sim->max_records = max_records;
  sim->path = path;
  sim->has_disorder = disorder != nullptr;
  sim->has_sp = disorder && d.prob_slow_p > 0.0;
  sim->has_sq = disorder && d.prob_slow_q > 0.0;
  sim->has_sp0 = sim->has_sp;
  sim->has_sq0 = sim->has_sq;
  sim->stream = (cudaStream_t)cuda_stream;
  char* base = (char*)d_workspace;
  sim->E = (uint32_t*)(base + y.off_E);
  sim->O = (uint32_t*)(base + y.off_O);
  if (path == KPZ_PATH_STREAM || path == KPZ_PATH_BLOCKED) {
    sim->E2 = (uint32_t*)(base + y.off_E2);
    sim->O2 = (uint32_t*)(base + y.off_O2);
  }
  if (disorder) {
    sim->SPE = (uint32_t*)(base + y.off_SPE);
    sim->SPO = (uint32_t*)(base + y.off_SPO);
    sim->SQE = (uint32_t*)(base + y.off_SQE);
    sim->SQO = (uint32_t*)(base + y.off_SQO);
  }
  sim->rec_t = (long long*)(base + y.off_rec_t);
  sim->rec_sum_h = (long long*)(base + y.off_h);
  sim->rec_sum_h2 = (long long*)(base + y.off_h2);
  sim->scratch = (int*)(base + y.off_scratch);
  sim->scratch_ints = y.scratch_ints;
  sim->ntiles = y.ntiles;
  if (path == KPZ_PATH_STREAM || path == KPZ_PATH_BLOCKED) {
    sim->k3off = (unsigned char*)(base + y.off_k3off);
    sim->tiles = (int*)(base + y.off_tiles);
  }

  KpzDev& D = sim->dev;
  D.keys = make_keys(seed);
  D.thr[0] = make_thresh(p);
  D.thr[1] = make_thresh(d.p_slow);
  D.thr[2] = make_thresh(q);
  D.thr[3] = make_thresh(d.q_slow);
  D.offset_mode = o.offset_mode;
  D.first_sample = o.first_sample;
  D.S = nsamples;
  D.PW = y.PW;
  D.PWp = y.PWp;
  D.U = y.U;
  D.E = sim->E;
  D.O = sim->O;
  refresh_planes(sim);

  sim->dis = d;
  rc = init_state(sim);
  if (rc) {
    delete sim;
    return rc;
  }
  *out = sim;
  return KPZ_OK;
}

int kpz_jit_check(int64_t L, double p, double q, const kpz_disorder* disorder, const kpz_options* opt,
                  size_t* cubin_bytes) {
  if (!cubin_bytes) return fail(KPZ_EINVAL, "cubin_bytes is NULL");
  *cubin_bytes = 0;
  int rc = validate_sizes(L, 1, 0);
  if (rc) return rc;
  if (!valid_prob(p) || !valid_prob(q)) return fail(KPZ_EINVAL, "p and q must lie in [0,1]");
  kpz_disorder d{0.0, p, 0.0, q};
  if (disorder) d = *disorder;
  if (!valid_prob(d.prob_slow_p) || !valid_prob(d.p_slow) || !valid_prob(d.prob_slow_q) || !valid_prob(d.q_slow))
    return fail(KPZ_EINVAL, "disorder probabilities must lie in [0,1]");
  int path;
  rc = choose_path(L, opt, &path);
  if (rc) return rc;
  kpz_sim tmp;
  tmp.has_sp = disorder && d.prob_slow_p > 0.0;
  tmp.has_sq = disorder && d.prob_slow_q > 0.0;
  KpzDev& D = tmp.dev;
  D.thr[0] = make_thresh(p);
  D.thr[1] = make_thresh(d.p_slow);
  D.thr[2] = make_thresh(q);
  D.thr[3] = make_thresh(d.q_slow);
  D.offset_mode = opt ? opt->offset_mode : 0;
  D.PW = (int)(L / 64);
  refresh_planes(&tmp);
  if (!k1_use_jit(D)) return KPZ_OK;
  std::vector<char> cubin;
  D.PWp = (D.PW + 3) / 4 * 4;
  D.U = D.PWp / 4;
  const int dis_c = tmp.has_sq ? 2 : tmp.has_sp ? 1 : 0;
  std::vector<std::string> defs = path == KPZ_PATH_ONCHIP ? k1_shape(D, 1, dis_c).defs : k1_jit_defines(D, dis_c);
  if (path == KPZ_PATH_BLOCKED) {
    drop_define(&defs, "K1J_UPT");
    defs.push_back("K1J_TILE=1");
  } else if (path == KPZ_PATH_STREAM) {  // as k3_run asks for it
    drop_define(&defs, "K1J_UPT");
    drop_define(&defs, "K1J_PDL");
    defs.push_back("K1J_STREAM=1");
    defs.push_back(k3_pdl() ? "K1J_PDL=1" : "K1J_PDL=0");
  }
  rc = jit_compile("k1_sweep_jit.cuh",
                   path == KPZ_PATH_BLOCKED ? "kpz_k3t_sweep_jit" : path == KPZ_PATH_STREAM ? "kpz_k3_pass_jit" : "kpz_k1_sweep_jit",
                   defs, &cubin, nullptr);
  if (rc) return rc;
  *cubin_bytes = cubin.size();
  return KPZ_OK;
}

int kpz_destroy(kpz_sim* sim) {
  delete sim;
  return KPZ_OK;
}

int kpz_reset(kpz_sim* sim) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  sim->has_sp = sim->has_sp0;
  sim->has_sq = sim->has_sq0;
  refresh_planes(sim);
  int rc = init_state(sim);
  if (rc) return rc;
  sim->t = 0;
  sim->nrec = 0;
  sim->frame = 0;
  sim->h0 = 1;
  sim->t_h0 = 0;
  sim->h0_pending = false;
  sim->guard_checked = false;
  return KPZ_OK;
}

int kpz_path(const kpz_sim* sim, int32_t* path) {
  if (!sim || !path) return fail(KPZ_EINVAL, "NULL argument");
  *path = sim->path;
  return KPZ_OK;
}

int kpz_time(const kpz_sim* sim, int64_t* t) {
  if (!sim || !t) return fail(KPZ_EINVAL, "NULL argument");
  *t = sim->t;
  return KPZ_OK;
}

int kpz_set_time(kpz_sim* sim, int64_t t) {
  if (!sim || t < 0 || ((uint64_t)t >> 54) != 0) return fail(KPZ_EINVAL, "need 0 <= t < 2^54");
  if (!sim->h0_pending) {  // the lattice is as rough as it was a moment ago; only the clock moves
    sim->h0 = std::min<int64_t>(sim->L, sim->h0 + 8 * std::max<int64_t>(sim->t - sim->t_h0, 0));
  }
  sim->t_h0 = t;
  sim->t = t;
  sim->rec_times.clear();
  sim->nrec = 0;
  return KPZ_OK;
}

int kpz_set_record_times(kpz_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return fail(KPZ_EINVAL, "bad record-time list");
  if (nt > sim->max_records) return fail(KPZ_ENOMEM, "%d record times but max_records=%d", nt, sim->max_records);
  for (int32_t k = 0; k < nt; ++k) {
    if (t[k] < 1 || (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1]))
      return fail(KPZ_EINVAL, "record times must be strictly increasing and later than the current time");
  }
  // |h| <= min(L, h0 + 8 (t - t0)); refuse when L * bound^2 could overflow int64
  if (int rc = guard_record_times(sim, t, nt)) return rc;
  sim->rec_times.assign(t, t + nt);
  sim->nrec = 0;
  if (nt > 0) {
    // stream-ordered copy from a staging vector that outlives the call: use a synchronous-safe pageable copy
    KPZ_CUDA_CHECK(cudaMemcpyAsync(sim->rec_t, sim->rec_times.data(), (size_t)nt * 8, cudaMemcpyHostToDevice, sim->stream));
    KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  }
  return KPZ_OK;
}

int kpz_run(kpz_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return fail(KPZ_EINVAL, "bad arguments");
  if (n_mcs == 0) return KPZ_OK;
  if (((uint64_t)(sim->t + n_mcs) >> 54) != 0) return fail(KPZ_EUNSUPPORTED, "time beyond 2^54 MCS");
  const int32_t nt = (int32_t)sim->rec_times.size();
  int rc = KPZ_OK;
  if (!sim->guard_checked) {  // the lattice was replaced after the record times were listed
    rc = guard_record_times(sim, sim->rec_times.data(), nt);
    if (rc) return rc;
  }
  if (sim->path == KPZ_PATH_ONCHIP) {
    KpzRunArgs A{};
    A.t0 = sim->t;
    A.n_mcs = n_mcs;
    A.rec_t = sim->rec_t;
    A.rec_begin = sim->nrec;
    A.nt = nt;
    A.rec_sum_h = sim->rec_sum_h;
    A.rec_sum_h2 = sim->rec_sum_h2;
    const KpzDev& D = sim->dev;
    const bool single = D.U <= 32;
    const bool partial = (D.PW % 4) != 0;
    const int dis = sim->has_sq ? 2 : sim->has_sp ? 1 : 0;
    const int block = (D.U + 31) / 32 * 32;
    if (k1_use_jit(D)) {
      K1Shape sh = k1_shape(D, sim->S, dis, n_mcs);
      void* kfn = nullptr;
      rc = jit_get("k1_sweep_jit.cuh", "kpz_k1_sweep_jit", sh.defs, &kfn);
      if (rc) return rc;
      // debug (kpz_debug_config "K1J_HALOCHECK=1"): sequence numbers on the shared-memory halo slots, counted here
      const bool halocheck = debug_int("K1J_HALOCHECK", 0) != 0;
      unsigned int* check = (unsigned int*)(sim->scratch + D.PW + 32);
      if (halocheck) {
        KPZ_CUDA_CHECK(cudaMemsetAsync(check, 0, sizeof(unsigned int), sim->stream));
        A.check = check;
      }
      if (sh.queue > 0) {  // work counter and per-sample chunk counters: scratch ints [PW + 64, PW + 64 + S]
        A.queue = (unsigned int*)(sim->scratch + D.PW + 64);
        KPZ_CUDA_CHECK(cudaMemsetAsync(A.queue, 0, ((size_t)sim->S + 1) * sizeof(unsigned int), sim->stream));
      }
      void* args[] = {(void*)&D, (void*)&A};
      KPZ_CUDA_CHECK(cudaLaunchKernel(kfn, dim3(sh.grid), dim3(sh.block), args, 0, sim->stream));
      KPZ_LAUNCH_CHECK("kpz_k1_sweep_jit");
      if (halocheck) {
        unsigned int bad = 0;
        KPZ_CUDA_CHECK(cudaMemcpyAsync(&bad, check, sizeof bad, cudaMemcpyDeviceToHost, sim->stream));
        KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
        if (bad) return fail(KPZ_ECUDA, "halo sequence check: %u reads of a slot of another exchange", bad);
      }
    } else {
      K1Fn fn = k1_pick(single, partial, dis, D.nplanes);
      fn<<<sim->S, block, 0, sim->stream>>>(D, A);
      KPZ_LAUNCH_CHECK("kpz_k1_kernel");
    }
  } else if (sim->path == KPZ_PATH_BLOCKED) {
    rc = k3t_run(sim, n_mcs);
    if (rc) return rc;
  } else {
    rc = k3_run(sim, n_mcs);
    if (rc) return rc;
  }
  sim->t += n_mcs;
  while (sim->nrec < nt && sim->rec_times[sim->nrec] <= sim->t) sim->nrec++;
  return KPZ_OK;
}

int kpz_lattice(kpz_sim* sim, uint32_t* d_words) {
  if (!sim || !d_words) return fail(KPZ_EINVAL, "NULL argument");
  const KpzDev& D = sim->dev;
  k_eo_to_nat<<<grid_for((size_t)D.S * D.PW), 256, 0, sim->stream>>>(sim->E, sim->O, D.S, D.PW, D.PWp, d_words);
  KPZ_LAUNCH_CHECK("k_eo_to_nat");
  return KPZ_OK;
}

int kpz_set_lattice(kpz_sim* sim, const uint32_t* d_words) {
  if (!sim || !d_words) return fail(KPZ_EINVAL, "NULL argument");
  const KpzDev& D = sim->dev;
  k_nat_to_eo<<<grid_for((size_t)D.S * D.PW), 256, 0, sim->stream>>>(d_words, D.S, D.PW, D.PWp, sim->E, sim->O);
  KPZ_LAUNCH_CHECK("k_nat_to_eo");
  return measure_h0(sim);
}

int kpz_disorder_masks(kpz_sim* sim, uint32_t* d_slow_p, uint32_t* d_slow_q) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const KpzDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.PW;
  if (d_slow_p) {
    if (sim->has_disorder) k_eo_to_nat<<<grid_for(n), 256, 0, sim->stream>>>(sim->SPE, sim->SPO, D.S, D.PW, D.PWp, d_slow_p);
    else k_zero_words<<<grid_for(2 * n), 256, 0, sim->stream>>>(d_slow_p, 2 * n);
    KPZ_LAUNCH_CHECK("disorder_masks(p)");
  }
  if (d_slow_q) {
    if (sim->has_disorder) k_eo_to_nat<<<grid_for(n), 256, 0, sim->stream>>>(sim->SQE, sim->SQO, D.S, D.PW, D.PWp, d_slow_q);
    else k_zero_words<<<grid_for(2 * n), 256, 0, sim->stream>>>(d_slow_q, 2 * n);
    KPZ_LAUNCH_CHECK("disorder_masks(q)");
  }
  return KPZ_OK;
}

int kpz_set_disorder_masks(kpz_sim* sim, const uint32_t* d_slow_p, const uint32_t* d_slow_q) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  if (!sim->has_disorder) return fail(KPZ_EINVAL, "handle was created without a disorder description");
  const KpzDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.PW;
  if (d_slow_p) {
    k_nat_to_eo<<<grid_for(n), 256, 0, sim->stream>>>(d_slow_p, D.S, D.PW, D.PWp, sim->SPE, sim->SPO);
    KPZ_LAUNCH_CHECK("set_disorder_masks(p)");
    sim->has_sp = true;
  }
  if (d_slow_q) {
    k_nat_to_eo<<<grid_for(n), 256, 0, sim->stream>>>(d_slow_q, D.S, D.PW, D.PWp, sim->SQE, sim->SQO);
    KPZ_LAUNCH_CHECK("set_disorder_masks(q)");
    sim->has_sq = true;
  }
  refresh_planes(sim);
  return KPZ_OK;
}

int kpz_heights(kpz_sim* sim, int32_t sample, int32_t* d_h) {
  if (!sim || !d_h || sample < 0 || sample >= sim->S) return fail(KPZ_EINVAL, "bad arguments");
  if (sim->L > 0x7FFFFFFF) return fail(KPZ_EUNSUPPORTED, "heights need L < 2^31");
  const KpzDev& D = sim->dev;
  const uint32_t* E = sim->E + (size_t)sample * D.PWp;
  const uint32_t* O = sim->O + (size_t)sample * D.PWp;
  k_group_totals<<<grid_for(D.PW), 256, 0, sim->stream>>>(E, O, D.PW, sim->scratch);
  KPZ_LAUNCH_CHECK("k_group_totals");
  k_exclusive_scan_1block<<<1, 1024, 0, sim->stream>>>(sim->scratch, D.PW);
  KPZ_LAUNCH_CHECK("k_exclusive_scan_1block");
  k_heights_expand<<<grid_for(D.PW, 128), 128, 0, sim->stream>>>(E, O, sim->scratch, D.PW, d_h);
  KPZ_LAUNCH_CHECK("k_heights_expand");
  return KPZ_OK;
}

int kpz_roughness(kpz_sim* sim, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean) {
  if (!sim || !nt) return fail(KPZ_EINVAL, "NULL argument");
  if (*nt < sim->nrec) return fail(KPZ_ENOMEM, "capacity %d < %d records", *nt, sim->nrec);
  const int32_t n = sim->nrec;
  const size_t cells = (size_t)n * sim->S;
  std::vector<int64_t> h, h2;
  int64_t* ph = sum_h;
  int64_t* ph2 = sum_h2;
  if (n > 0) {
    if (!ph) {
      h.resize(cells);
      ph = h.data();
    }
    if (!ph2) {
      h2.resize(cells);
      ph2 = h2.data();
    }
    KPZ_CUDA_CHECK(cudaMemcpyAsync(ph, sim->rec_sum_h, cells * 8, cudaMemcpyDeviceToHost, sim->stream));
    KPZ_CUDA_CHECK(cudaMemcpyAsync(ph2, sim->rec_sum_h2, cells * 8, cudaMemcpyDeviceToHost, sim->stream));
  }
  KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  for (int32_t k = 0; k < n; ++k) {
    if (t) t[k] = sim->rec_times[k];
    if (w2_mean) {
      // Eq. 3 squared per sample, averaged over samples
      double acc = 0.0;
      for (int32_t s = 0; s < sim->S; ++s) {
        const __int128 s1 = ph[(size_t)k * sim->S + s], s2 = ph2[(size_t)k * sim->S + s];
        const __int128 num = (__int128)sim->L * s2 - s1 * s1;
        acc += (double)num / ((double)sim->L * (double)sim->L);
      }
      w2_mean[k] = acc / (double)sim->S;
    }
  }
  *nt = n;
  return KPZ_OK;
}

}  // extern "C"
