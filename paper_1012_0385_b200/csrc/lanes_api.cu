// lanes_api.cu — host side of the two-lane model: the lanes_* entry points of include/kpz_b200.h.
#include <algorithm>
#include <cstdlib>
#include <new>
#include <string>
#include <vector>

#include "common.cuh"
#include "jit.h"
#include "lanes_k4.cuh"

using namespace kpz;

struct lanes_sim {
  int64_t L = 0;
  int32_t S = 0;
  int32_t max_records = 0;
  LanesDev dev{};
  cudaStream_t stream = nullptr;
  long long* rec_t = nullptr;
  long long* rec = nullptr;  // [4][max_records][S] (plane stride = nt * S of the current list)
  int64_t t = 0;
  int64_t nsnap = 0;  // profile snapshots taken (epoch ends passed by lanes_run)
  std::vector<int64_t> rec_times;
  int32_t nrec = 0;
  unsigned int* check = nullptr;  // debug counter (K4J_HALOCHECK)
  char* base = nullptr;   // workspace start
  size_t zero_bytes = 0;  // lattices (incl. pad words), counters and profile sit in [base, base + zero_bytes)
  Thresh t_rho{};
};

namespace {

struct LLayout {
  size_t off_A, off_B, off_T, off_V, off_JA, off_JB, off_occA, off_occB, off_rec_t, off_rec, off_check, total;
  int W, Wp, U;
};

int lanes_validate(int64_t L, int32_t S, int32_t max_records) {
  if (L < 4 || (L & 1) || S < 1 || max_records < 0) return fail(KPZ_EINVAL, "need even L >= 4, nsamples >= 1, max_records >= 0");
  if (L % 64 != 0) return fail(KPZ_EUNSUPPORTED, "the CUDA path needs L to be a multiple of 64 (L=%lld)", (long long)L);
  if (L > 262144) return fail(KPZ_EUNSUPPORTED, "the two-lane kernel holds at most 262144 sites per lane on chip (L=%lld)", (long long)L);
  if ((int64_t)S * L > ((int64_t)1 << 33)) return fail(KPZ_EUNSUPPORTED, "nsamples * L too large");
  return KPZ_OK;
}

LLayout lanes_layout(int64_t L, int32_t S, int32_t max_records) {
  LLayout y{};
  y.W = (int)(L / 32);
  y.Wp = (y.W + 7) / 8 * 8;
  y.U = y.Wp / 8;
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off += align_up(bytes, 256);
    return o;
  };
  const size_t plane = (size_t)S * y.Wp * 4;
  y.off_A = take(plane);
  y.off_B = take(plane);
  y.off_T = take(plane);
  y.off_V = take(plane);
  y.off_JA = take((size_t)S * 8);
  y.off_JB = take((size_t)S * 8);
  y.off_occA = take((size_t)S * L * 4);
  y.off_occB = take((size_t)S * L * 4);
  y.off_rec_t = take((size_t)std::max(max_records, 1) * 8);
  y.off_rec = take((size_t)4 * std::max(max_records, 1) * S * 8);
  y.off_check = take(256);  // debug counter (K4J_HALOCHECK)
  y.total = off;
  return y;
}

// ---- K4 v2: kernel specialised at run time on (L, thresholds, offset mode) — k4_lanes_jit.cuh ---------------------
bool k4_use_jit(const LanesDev& D) { return jit_enabled() && (D.W + 3) / 4 <= 1024; }

// Launch shape of the run-time specialised two-lane kernel (k4_lanes_jit.cuh): which of its code shapes, how many MCS
// per precomputed chunk, block size, dynamic shared memory - the same numbers go to the compiler as definitions.
struct K4Shape {
  int pre = 1, chunk = 1, vprof = 0, block = 32;
  size_t smem = 0;
};
K4Shape k4_shape(const LanesDev& D) {
  K4Shape sh;
  const int nthreads = ((D.W + 3) / 4 + 31) / 32 * 32;
  const int nwarps = nthreads / 32;
  sh.pre = debug_int("K4J_PRE", 1) ? 1 : 0;
  sh.vprof = nthreads <= 256 ? std::max(0, std::min(12, debug_int("K4J_VPROF", 6))) : 0;
  const size_t fixed = 128 * 16 + 128 * 4 + 2 * 32 * 16;  // queue and flags of one WarpSmem
  const size_t vbytes = (size_t)2 * sh.vprof * nthreads * 16;
  // MCS per chunk: as many as keep the CTA near 100 KB (two CTAs per SM), at most 16
  const long long budget = 100 * 1024 - (long long)vbytes;
  const long long per_warp = budget / nwarps - (long long)fixed;
  int chunk = (int)std::max<long long>(1, std::min<long long>(16, per_warp / 1024));
  sh.chunk = std::max(1, std::min(256, debug_int("K4J_CHUNK", chunk)));
  sh.block = nthreads;
  sh.smem = (sh.pre ? (size_t)nwarps * ((size_t)sh.chunk * 1024 + fixed) : 0) + vbytes;
  return sh;
}

std::vector<std::string> k4_jit_defines(const LanesDev& D) {
  auto T = [](const Thresh& t) -> unsigned long long { return t.always ? (1ull << 32) : (unsigned long long)t.value; };
  char buf[64];
  std::vector<std::string> d;
  snprintf(buf, sizeof buf, "K4J_W=%d", D.W);
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_TPA=0x%llxull", T(D.t_pa));
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_TPB=0x%llxull", T(D.t_pb));
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_TOMEGA=0x%llxull", T(D.t_omega));
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_TTURN=0x%llxull", D.period > 0 ? T(D.t_turn) : 0ull);  // never redrawn without a period
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_OFFSET_MODE=%d", D.offset_mode);
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_TW0=0x%llxull", T(D.t_w0));
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_INDEP=%d", D.independent);
  d.push_back(buf);
  debug_defines("K4J_", &d);  // kpz_debug_config: tests and tuning only (the run reads no environment)
  // the launch shape as the host computed it (clamped), not the raw debug values
  const K4Shape sh = k4_shape(D);
  for (const char* name : {"K4J_PRE", "K4J_CHUNK", "K4J_VPROF"}) {
    const std::string key = std::string(name) + "=";
    d.erase(std::remove_if(d.begin(), d.end(), [&](const std::string& x) { return x.compare(0, key.size(), key) == 0; }),
            d.end());
  }
  snprintf(buf, sizeof buf, "K4J_PRE=%d", sh.pre);
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_CHUNK=%d", sh.chunk);
  d.push_back(buf);
  snprintf(buf, sizeof buf, "K4J_VPROF=%d", sh.vprof);
  d.push_back(buf);
  return d;
}

int grid_for(size_t n, int block = 256) {
  size_t g = (n + block - 1) / block;
  return (int)std::min<size_t>(std::max<size_t>(g, 1), 148 * 16);
}

// Initial occupations, epoch-0 turning points (§R13), zero counters and profile.
int lanes_init_state(lanes_sim* sim) {
  const LanesDev& D = sim->dev;
  KPZ_CUDA_CHECK(cudaMemsetAsync(sim->base, 0, sim->zero_bytes, sim->stream));
  const size_t ng = (size_t)D.S * ((D.W + 3) / 4);
  k_site_mask_nat<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_INIT_A, sim->t_rho, 0, D.first_sample, D.S, D.W, D.Wp, D.A);
  KPZ_LAUNCH_CHECK("k_site_mask_nat");
  k_site_mask_nat<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_INIT_B, sim->t_rho, 0, D.first_sample, D.S, D.W, D.Wp, D.B);
  KPZ_LAUNCH_CHECK("k_site_mask_nat");
  k_site_mask_nat<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_TURN, D.t_turn, 0, D.first_sample, D.S, D.W, D.Wp, D.T);
  KPZ_LAUNCH_CHECK("k_site_mask_nat");
  if (D.independent) {
    k_site_mask_nat<<<grid_for(ng, 128), 128, 0, sim->stream>>>(D.keys, TAG_TURN_V, D.t_turn, 0, D.first_sample, D.S, D.W, D.Wp, D.V);
    KPZ_LAUNCH_CHECK("k_site_mask_nat");
  }
  return KPZ_OK;
}

}  // namespace

extern "C" {

int lanes_reset(lanes_sim* sim) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  int rc = lanes_init_state(sim);
  if (rc) return rc;
  sim->t = 0;
  sim->nsnap = 0;
  sim->nrec = 0;
  return KPZ_OK;
}

int lanes_workspace_bytes(int64_t L, int32_t nsamples, int32_t max_records, size_t* bytes) {
  if (!bytes) return fail(KPZ_EINVAL, "bytes is NULL");
  int rc = lanes_validate(L, nsamples, max_records);
  if (rc) return rc;
  *bytes = lanes_layout(L, nsamples, max_records).total;
  return KPZ_OK;
}

int lanes_create(lanes_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0, double turn_prob,
                 int64_t turn_period, double omega, uint64_t seed, const kpz_options* opt, int32_t max_records,
                 void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  const lanes_crossing c{turn_prob, omega, 0.0, 0};  // turning-point model: no crossing at unflagged sites, one flag set
  return lanes_create_crossing(out, L, nsamples, p_a, p_b, rho0, &c, turn_period, seed, opt, max_records, d_workspace,
                               workspace_bytes, cuda_stream);
}

int lanes_create_crossing(lanes_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                          const lanes_crossing* crossing, int64_t turn_period, uint64_t seed, const kpz_options* opt,
                          int32_t max_records, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return fail(KPZ_EINVAL, "out is NULL");
  *out = nullptr;
  if (!crossing) return fail(KPZ_EINVAL, "crossing is NULL");
  const double turn_prob = crossing->prob_flag, omega = crossing->w_flagged;
  int rc = lanes_validate(L, nsamples, max_records);
  if (rc) return rc;
  if (!valid_prob(p_a) || !valid_prob(p_b) || !valid_prob(rho0) || !valid_prob(turn_prob) || !valid_prob(omega) ||
      !valid_prob(crossing->w_unflagged) || turn_period < 0 || (crossing->independent != 0 && crossing->independent != 1))
    return fail(KPZ_EINVAL, "probabilities must lie in [0,1], turn_period >= 0, independent in {0,1}");
  kpz_options o{0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1))
    return fail(KPZ_EINVAL, "options: first_sample >= 0, offset_mode in {0,1}");
  if (!d_workspace || ((uintptr_t)d_workspace & 255) != 0) return fail(KPZ_EINVAL, "d_workspace must be non-NULL and 256-byte aligned");
  const LLayout y = lanes_layout(L, nsamples, max_records);
  if (workspace_bytes < y.total) return fail(KPZ_ENOMEM, "workspace has %zu bytes, %zu needed", workspace_bytes, y.total);
  lanes_sim* sim = new (std::nothrow) lanes_sim();
  if (!sim) return fail(KPZ_ENOMEM, "host allocation failed");
  sim->L = L;
  sim->S = nsamples;
  sim->max_records = max_records;
  sim->stream = (cudaStream_t)cuda_stream;
  char* base = (char*)d_workspace;
  LanesDev& D = sim->dev;
  D.keys = make_keys(seed);
  D.t_pa = make_thresh(p_a);
  D.t_pb = make_thresh(p_b);
  D.t_turn = make_thresh(turn_prob);
  D.t_omega = make_thresh(omega);
  D.t_w0 = make_thresh(crossing->w_unflagged);
  D.independent = crossing->independent;
  D.np_a = planes_needed(D.t_pa);
  D.np_b = planes_needed(D.t_pb);
  D.np_w = planes_needed(D.t_omega);
  D.offset_mode = o.offset_mode;
  D.first_sample = o.first_sample;
  D.S = nsamples;
  D.W = y.W;
  D.Wp = y.Wp;
  D.U = y.U;
  D.period = turn_period;
  D.A = (uint32_t*)(base + y.off_A);
  D.B = (uint32_t*)(base + y.off_B);
  D.T = (uint32_t*)(base + y.off_T);
  D.V = D.independent ? (uint32_t*)(base + y.off_V) : D.T;
  D.JA = (unsigned long long*)(base + y.off_JA);
  D.JB = (unsigned long long*)(base + y.off_JB);
  D.occA = (uint32_t*)(base + y.off_occA);
  D.occB = (uint32_t*)(base + y.off_occB);
  sim->rec_t = (long long*)(base + y.off_rec_t);
  sim->rec = (long long*)(base + y.off_rec);
  sim->check = (unsigned int*)(base + y.off_check);

  sim->zero_bytes = y.off_rec_t;
  sim->base = base;
  sim->t_rho = make_thresh(rho0);
  rc = lanes_init_state(sim);
  if (rc) {
    delete sim;
    return rc;
  }
  *out = sim;
  return KPZ_OK;
}

int lanes_jit_check(int64_t L, double p_a, double p_b, double turn_prob, int64_t turn_period, double omega,
                    const kpz_options* opt, size_t* cubin_bytes) {
  const lanes_crossing c{turn_prob, omega, 0.0, 0};
  return lanes_crossing_jit_check(L, p_a, p_b, &c, turn_period, opt, cubin_bytes);
}

int lanes_crossing_jit_check(int64_t L, double p_a, double p_b, const lanes_crossing* crossing, int64_t turn_period,
                             const kpz_options* opt, size_t* cubin_bytes) {
  if (!cubin_bytes || !crossing) return fail(KPZ_EINVAL, "NULL argument");
  *cubin_bytes = 0;
  const double turn_prob = crossing->prob_flag, omega = crossing->w_flagged;
  int rc = lanes_validate(L, 1, 0);
  if (rc) return rc;
  if (!valid_prob(p_a) || !valid_prob(p_b) || !valid_prob(turn_prob) || !valid_prob(omega) ||
      !valid_prob(crossing->w_unflagged) || turn_period < 0 || (crossing->independent != 0 && crossing->independent != 1))
    return fail(KPZ_EINVAL, "probabilities must lie in [0,1], turn_period >= 0, independent in {0,1}");
  LanesDev D{};
  D.t_pa = make_thresh(p_a);
  D.t_pb = make_thresh(p_b);
  D.t_turn = make_thresh(turn_prob);
  D.t_omega = make_thresh(omega);
  D.t_w0 = make_thresh(crossing->w_unflagged);
  D.independent = crossing->independent;
  D.offset_mode = opt ? opt->offset_mode : 0;
  D.W = (int)(L / 32);
  D.period = turn_period;
  if (!k4_use_jit(D)) return KPZ_OK;
  std::vector<char> cubin;
  rc = jit_compile("k4_lanes_jit.cuh", "lanes_k4_sweep_jit", k4_jit_defines(D), &cubin, nullptr);
  if (rc) return rc;
  *cubin_bytes = cubin.size();
  return KPZ_OK;
}

int lanes_destroy(lanes_sim* sim) {
  delete sim;
  return KPZ_OK;
}

int lanes_time(const lanes_sim* sim, int64_t* t) {
  if (!sim || !t) return fail(KPZ_EINVAL, "NULL argument");
  *t = sim->t;
  return KPZ_OK;
}

int lanes_set_time(lanes_sim* sim, int64_t t) {
  if (!sim || t < 0 || ((uint64_t)t >> 54) != 0) return fail(KPZ_EINVAL, "need 0 <= t < 2^54");
  sim->t = t;
  sim->rec_times.clear();
  sim->nrec = 0;
  return KPZ_OK;
}

int lanes_set_record_times(lanes_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return fail(KPZ_EINVAL, "bad record-time list");
  if (nt > sim->max_records) return fail(KPZ_ENOMEM, "%d record times but max_records=%d", nt, sim->max_records);
  for (int32_t k = 0; k < nt; ++k)
    if (t[k] < 1 || (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1]))
      return fail(KPZ_EINVAL, "record times must be strictly increasing and later than the current time");
  sim->rec_times.assign(t, t + nt);
  sim->nrec = 0;
  if (nt > 0) {
    KPZ_CUDA_CHECK(cudaMemcpyAsync(sim->rec_t, sim->rec_times.data(), (size_t)nt * 8, cudaMemcpyHostToDevice, sim->stream));
    KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  }
  return KPZ_OK;
}

int lanes_run(lanes_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return fail(KPZ_EINVAL, "bad arguments");
  if (n_mcs == 0) return KPZ_OK;
  if (((uint64_t)(sim->t + n_mcs) >> 54) != 0) return fail(KPZ_EUNSUPPORTED, "time beyond 2^54 MCS");
  const LanesDev& D = sim->dev;
  const int32_t nt = (int32_t)sim->rec_times.size();
  LanesRunArgs A{};
  A.t0 = sim->t;
  A.n_mcs = n_mcs;
  A.rec_t = sim->rec_t;
  A.rec_begin = sim->nrec;
  A.nt = nt;
  A.rec = sim->rec;
  const bool single = D.U <= 32;
  const bool partial = (D.W % 8) != 0;
  const int block = (D.U + 31) / 32 * 32;
  if (k4_use_jit(D)) {
    void* kfn = nullptr;
    int rc = jit_get("k4_lanes_jit.cuh", "lanes_k4_sweep_jit", k4_jit_defines(D), &kfn);
    if (rc) return rc;
    void* args[] = {(void*)&D, (void*)&A};
    const int U4 = (D.W + 3) / 4;                      // one thread per 128-site supergroup
    const int block4 = (U4 + 31) / 32 * 32;
    // small rings (k4_lanes_jit.cuh, SPW): U4 <= 16 supergroups, a power of two, no ragged word -> 32/U4 samples per warp
    const bool pack = (D.W % 4) == 0 && U4 <= 16 && (U4 & (U4 - 1)) == 0;
    const int spw = pack ? 32 / U4 : 1;
    const K4Shape sh = k4_shape(D);
    (void)block4;
    const bool halocheck = debug_int("K4J_HALOCHECK", 0) != 0;  // debug: sequence numbers on the halo slots
    if (halocheck) {
      KPZ_CUDA_CHECK(cudaMemsetAsync(sim->check, 0, sizeof(unsigned int), sim->stream));
      A.check = sim->check;
      args[1] = (void*)&A;
    }
    if (sh.smem > 32 * 1024)  // static shared memory (halo, sums, pack slots) comes on top
      KPZ_CUDA_CHECK(cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sh.smem));
    KPZ_CUDA_CHECK(cudaLaunchKernel(kfn, dim3((sim->S + spw - 1) / spw), dim3(sh.block), args, sh.smem, sim->stream));
    if (halocheck) {
      unsigned int bad = 0;
      KPZ_CUDA_CHECK(cudaMemcpyAsync(&bad, sim->check, sizeof bad, cudaMemcpyDeviceToHost, sim->stream));
      KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
      if (bad) return fail(KPZ_ECUDA, "halo sequence check: %u reads of a slot of another exchange", bad);
    }
  } else if (D.independent || D.t_w0.value != 0 || D.t_w0.always) {
    return fail(KPZ_EUNSUPPORTED, "the site-wise crossing model runs on the run-time specialised kernel only "
                                  "(L <= 131072, KPZ_B200_JIT not 0)");
  } else if (single) {
    if (partial) lanes_k4_kernel<true, true><<<sim->S, block, 0, sim->stream>>>(D, A);
    else lanes_k4_kernel<true, false><<<sim->S, block, 0, sim->stream>>>(D, A);
  } else {
    if (partial) lanes_k4_kernel<false, true><<<sim->S, block, 0, sim->stream>>>(D, A);
    else lanes_k4_kernel<false, false><<<sim->S, block, 0, sim->stream>>>(D, A);
  }
  KPZ_LAUNCH_CHECK("lanes_k4_kernel");
  if (D.period > 0) sim->nsnap += (sim->t + n_mcs) / D.period - sim->t / D.period;
  sim->t += n_mcs;
  while (sim->nrec < nt && sim->rec_times[sim->nrec] <= sim->t) sim->nrec++;
  return KPZ_OK;
}

int lanes_state(lanes_sim* sim, uint32_t* d_a, uint32_t* d_b, uint32_t* d_turn) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const LanesDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.W;
  const uint32_t* src[3] = {D.A, D.B, D.T};
  uint32_t* dst[3] = {d_a, d_b, d_turn};
  for (int k = 0; k < 3; ++k)
    if (dst[k]) {
      k_copy_rows<<<grid_for(n), 256, 0, sim->stream>>>(src[k], D.S, D.W, D.Wp, D.W, dst[k]);
      KPZ_LAUNCH_CHECK("k_copy_rows");
    }
  return KPZ_OK;
}

int lanes_set_state(lanes_sim* sim, const uint32_t* d_a, const uint32_t* d_b, const uint32_t* d_turn) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const LanesDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.W;
  const uint32_t* src[3] = {d_a, d_b, d_turn};
  uint32_t* dst[3] = {D.A, D.B, D.T};
  for (int k = 0; k < 3; ++k)
    if (src[k]) {
      k_copy_rows<<<grid_for(n), 256, 0, sim->stream>>>(src[k], D.S, D.W, D.W, D.Wp, dst[k]);
      KPZ_LAUNCH_CHECK("k_copy_rows");
    }
  return KPZ_OK;
}

int lanes_flags(lanes_sim* sim, uint32_t* d_u, uint32_t* d_v) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const LanesDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.W;
  const uint32_t* src[2] = {D.T, D.V};
  uint32_t* dst[2] = {d_u, d_v};
  for (int k = 0; k < 2; ++k)
    if (dst[k]) {
      k_copy_rows<<<grid_for(n), 256, 0, sim->stream>>>(src[k], D.S, D.W, D.Wp, D.W, dst[k]);
      KPZ_LAUNCH_CHECK("k_copy_rows");
    }
  return KPZ_OK;
}

int lanes_set_flags(lanes_sim* sim, const uint32_t* d_u, const uint32_t* d_v) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const LanesDev& D = sim->dev;
  if (d_v && !D.independent) return fail(KPZ_EINVAL, "one shared flag set: pass it as d_u");
  const size_t n = (size_t)D.S * D.W;
  const uint32_t* src[2] = {d_u, d_v};
  uint32_t* dst[2] = {D.T, D.V};
  for (int k = 0; k < 2; ++k)
    if (src[k]) {
      k_copy_rows<<<grid_for(n), 256, 0, sim->stream>>>(src[k], D.S, D.W, D.W, D.Wp, dst[k]);
      KPZ_LAUNCH_CHECK("k_copy_rows");
    }
  return KPZ_OK;
}

int lanes_currents(lanes_sim* sim, int32_t* nt, int64_t* t, int64_t* j_a, int64_t* j_b, int64_t* n_a, int64_t* n_b) {
  if (!sim || !nt) return fail(KPZ_EINVAL, "NULL argument");
  if (*nt < sim->nrec) return fail(KPZ_ENOMEM, "capacity %d < %d records", *nt, sim->nrec);
  const int32_t n = sim->nrec;
  const size_t cells = (size_t)n * sim->S;
  const size_t plane = sim->rec_times.size() * (size_t)sim->S;
  int64_t* dst[4] = {j_a, j_b, n_a, n_b};
  if (n > 0)
    for (int k = 0; k < 4; ++k)
      if (dst[k])
        KPZ_CUDA_CHECK(cudaMemcpyAsync(dst[k], sim->rec + k * plane, cells * 8, cudaMemcpyDeviceToHost, sim->stream));
  KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  for (int32_t k = 0; k < n; ++k)
    if (t) t[k] = sim->rec_times[k];
  *nt = n;
  return KPZ_OK;
}

int lanes_profile(lanes_sim* sim, uint32_t* d_occ_a, uint32_t* d_occ_b, int64_t* nsnap) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const size_t bytes = (size_t)sim->S * sim->L * 4;
  if (d_occ_a) KPZ_CUDA_CHECK(cudaMemcpyAsync(d_occ_a, sim->dev.occA, bytes, cudaMemcpyDeviceToDevice, sim->stream));
  if (d_occ_b) KPZ_CUDA_CHECK(cudaMemcpyAsync(d_occ_b, sim->dev.occB, bytes, cudaMemcpyDeviceToDevice, sim->stream));
  KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  if (nsnap) *nsnap = sim->nsnap;
  return KPZ_OK;
}

}  // extern "C"
