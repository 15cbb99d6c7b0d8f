// kpz2d_api.cu — host side of the 2+1D generalisation: the kpz2d_* entry
// points of include/kpz_b200.h.  Validation, workspace carving, kernel launches; every step of the path runs in the
// kernels of kpz2d_k5.cuh.  No CPU fallback.
#include <algorithm>
#include <new>
#include <string>
#include <vector>

#include "common.cuh"
#include "jit.h"
#include "kpz2d_util.cuh"

using namespace kpz;

struct kpz2d_sim {
  Kpz2dDev dev{};
  int path = KPZ_PATH_STREAM;  // KPZ_PATH_ONCHIP: K5S (a sample per CTA), KPZ2D_PATH_CLUSTER: K5C, else K5 (a launch per pass)
  int32_t max_records = 0;
  cudaStream_t stream = nullptr;
  long long *rec_t = nullptr, *rec_h = nullptr, *rec_h2 = nullptr;
  unsigned char* off = nullptr;  // [kChunkPasses][S] colour offsets of a chunk of passes
  int64_t t = 0;
  std::vector<int64_t> rec_times;
  int32_t nrec = 0;
};

namespace {

constexpr int kChunkPasses = 1024;
constexpr size_t kOnchipBytes = 96 * 1024;  // both slope fields of a sample in shared memory, two CTAs per SM

size_t onchip_bytes(int32_t Lx, int32_t Ly) { return (size_t)4 * Ly * (Lx / 64) * 4; }  // 4 parity planes of Ly * Lx/64 words

// K5C: a sample spread over a cluster of cs CTAs (kpz2d_k5.cuh): one supergroup per thread and row parity.
struct ClusterShape {
  int cs = 0, threads = 0, minb = 1;
  size_t smem = 0;  // dynamic shared memory per CTA
  int dual = 0;     // 1: two samples per cluster, swept alternately (cluster_body_dual)
};
constexpr int KPZ2D_CLUSTER = KPZ2D_PATH_CLUSTER;

// A cluster of 2, 4, 8 or 16 CTAs ("K5J_CS=n" forces one; 16 is beyond the portable cluster size and needs the kernel's
// consent: cudaFuncAttributeNonPortableClusterSizeAllowed) whose CTAs hold their rows in at most 100 KiB (two CTAs per
// SM) with at most max_nh supergroups per row parity (= threads per CTA); the smallest such cluster.  False when there
// is none.
bool cluster_shape_upto(int32_t Lx, int32_t Ly, int forced, int max_nh, ClusterShape* out) {
  for (int cs : {2, 4, 8, 16}) {
    if (forced && cs != forced) continue;
    if (Ly % (2 * cs) != 0) continue;
    const size_t smem = onchip_bytes(Lx, Ly) / cs;
    const int nh = Lx / 256 * (Ly / cs) / 2;
    if (nh > max_nh || smem > 100 * 1024) continue;
    ClusterShape c;
    c.cs = cs;
    c.smem = smem;
    c.threads = std::max(32, (nh + 31) / 32 * 32);
    const int by_regs = 1024 / c.threads;  // 64 registers per thread
    const int by_smem = (int)((227 * 1024) / (smem + 3 * 1024));
    c.minb = std::max(1, std::min({by_regs, by_smem, 16}));
    *out = c;
    return true;
  }
  return false;
}

// Measured (profiles/r02_summary.md §6): CTAs of at most 256 threads run best, so that size is looked for first.
bool cluster_shape(int32_t Lx, int32_t Ly, ClusterShape* out) {
  if (Lx % 256 != 0) return false;
  const int forced = debug_int("K5J_CS", 0);
  bool ok = !forced && cluster_shape_upto(Lx, Ly, 0, 256, out);
  if (!ok) ok = cluster_shape_upto(Lx, Ly, forced, 512, out);
  if (ok && debug_int("K5J_DUAL", 0) != 0 && 2 * out->smem <= 200 * 1024) {  // two samples per cluster
    out->dual = 1;
    out->smem *= 2;
    out->minb = std::max(1, std::min({1024 / out->threads, (int)((227 * 1024) / (out->smem + 3 * 1024)), 16}));
  }
  return ok;
}

// options.path: 0 auto, 1 on chip (K5S: a sample in the shared memory of one CTA), 2 streamed (K5: one launch per colour
// pass), 3 on chip over a thread-block cluster (K5C).  auto: K5S when the sample fits 96 KiB, else K5C when a cluster
// shape exists (and run-time specialisation is on), else K5.
int choose_path2d(int32_t Lx, int32_t Ly, const kpz_options* opt, int* path) {
  const size_t bytes = onchip_bytes(Lx, Ly);
  int want = opt ? opt->path : KPZ_PATH_AUTO;
  ClusterShape cshape;
  const bool can_cluster = jit_enabled() && cluster_shape(Lx, Ly, &cshape);
  if (want == KPZ_PATH_AUTO) want = bytes <= kOnchipBytes ? KPZ_PATH_ONCHIP : (can_cluster ? KPZ2D_CLUSTER : KPZ_PATH_STREAM);
  if (want == KPZ_PATH_ONCHIP && bytes > 200 * 1024)
    return fail(KPZ_EUNSUPPORTED, "the on-chip 2+1D path holds at most 200 KiB of slopes per sample (%zu needed)", bytes);
  if (want == KPZ2D_CLUSTER && !can_cluster)
    return fail(KPZ_EUNSUPPORTED, "no thread-block cluster shape for %d x %d (needs Lx %% 256 == 0, Ly %% 4 == 0, at most 1600 KiB of "
                                  "slopes per sample, run-time specialisation on)", Lx, Ly);
  if (want != KPZ_PATH_ONCHIP && want != KPZ_PATH_STREAM && want != KPZ2D_CLUSTER)
    return fail(KPZ_EINVAL, "options.path must be 0, 1, 2 or 3 here");
  *path = want;
  return KPZ_OK;
}

int grid_for2(size_t n, int block = 256) {
  size_t g = (n + block - 1) / block;
  return (int)std::min<size_t>(std::max<size_t>(g, 1), 148 * 16);
}

struct Layout2d {
  size_t off_EX, off_OX, off_EY, off_OY, off_rec_t, off_h, off_h2, off_off, total;
  int RH;
};

int validate2d(int32_t Lx, int32_t Ly, int32_t S, int32_t max_records) {
  if (Lx < 2 || Ly < 2 || (Lx & 1) || (Ly & 1) || S < 1 || max_records < 0)
    return fail(KPZ_EINVAL, "need even Lx, Ly >= 2, nsamples >= 1, max_records >= 0");
  if (Lx % 64 != 0) return fail(KPZ_EUNSUPPORTED, "the CUDA path needs Lx to be a multiple of 64 (Lx=%d)", Lx);
  if (Lx > 32768 || Ly > 32768 || (int64_t)Lx * Ly > ((int64_t)1 << 30))
    return fail(KPZ_EUNSUPPORTED, "lattice too large (Lx, Ly <= 32768, Lx * Ly <= 2^30)");
  if ((int64_t)S * Lx * Ly / 64 > ((int64_t)1 << 31) - 8) return fail(KPZ_EUNSUPPORTED, "nsamples * Lx * Ly too large");
  return KPZ_OK;
}

Layout2d layout2d(int32_t Lx, int32_t Ly, int32_t S, int32_t max_records) {
  Layout2d y{};
  y.RH = Lx / 64;
  size_t off = 0;
  auto take = [&](size_t bytes) {
    size_t o = off;
    off += align_up(bytes, 256);
    return o;
  };
  const size_t plane = (size_t)S * Ly * y.RH * 4;  // one parity plane of one slope field
  y.off_EX = take(plane);
  y.off_OX = take(plane);
  y.off_EY = take(plane);
  y.off_OY = take(plane);
  y.off_rec_t = take((size_t)std::max(max_records, 1) * 8);
  y.off_h = take((size_t)std::max(max_records, 1) * S * 8);
  y.off_h2 = take((size_t)std::max(max_records, 1) * S * 8);
  y.off_off = take((size_t)kChunkPasses * S);
  y.total = off;
  return y;
}

// both thresholds depend on their two leading bit-planes at most (p = 0.75, 0.5, 0.25, 0, 1 ...): the kernels then draw
// those two planes unconditionally
bool two_planes(const Kpz2dDev& D) { return planes_needed(D.t_p) <= 2 && planes_needed(D.t_q) <= 2; }

// Definitions of the run-time specialised kernels (kpz2d_k5.cuh under NVRTC): shape, thresholds, launch shape.
// entry: 1 kpz2d_k5s_jit (smem = its dynamic shared memory), 2 kpz2d_k5c_jit (cl), 3 kpz2d_k5_pass_jit.
std::vector<std::string> k5_jit_defines(const Kpz2dDev& D, int entry, size_t smem, const ClusterShape* cl = nullptr) {
  char buf[64];
  std::vector<std::string> d;
  auto add = [&](const char* name, long long v) {
    snprintf(buf, sizeof buf, "%s=%lld", name, v);
    d.push_back(buf);
  };
  add("K5J_ENTRY", entry);
  add("K5J_LX", D.Lx);
  add("K5J_LY", D.Ly);
  snprintf(buf, sizeof buf, "K5J_TP=0x%xu", D.t_p.value);
  d.push_back(buf);
  add("K5J_TP_ALWAYS", D.t_p.always);
  snprintf(buf, sizeof buf, "K5J_TQ=0x%xu", D.t_q.value);
  d.push_back(buf);
  add("K5J_TQ_ALWAYS", D.t_q.always);
  add("K5J_TWO", two_planes(D) ? 1 : 0);
  // CTAs per SM the on-chip kernel is compiled for: two when two samples fit the shared memory of an SM
  add("K5J_MINB", debug_int("K5J_MINB", cl ? cl->minb : (smem != 0 && 2 * (smem + 1024) <= 227 * 1024 ? 2 : 1)));
  add("K5J_CS", cl ? cl->cs : 1);
  add("K5J_THREADS", cl ? cl->threads : 512);
  add("K5J_DUAL", cl ? cl->dual : 0);
  add("K5J_RIW", debug_int("K5J_RIW", 1));
  add("K5J_PIPE", debug_int("K5J_PIPE", 1));
  add("K5J_PDL", debug_int("K5J_PDL", 1));  // streamed kernel: programmatic dependent launch of consecutive passes
  add("K5J_NBR", debug_int("K5J_NBR", 0));  // neighbour-only mbarriers: measured slower than barrier.cluster (r02_summary §6)
  if (debug_has("K5J_XRALL")) add("K5J_XRALL", debug_int("K5J_XRALL", 0));
  return d;
}

// The specialised K5C kernel for this handle, ready to launch (attributes set).  KPZ_EUNSUPPORTED when the device cannot
// hold one cluster of that shape at all (clusters of 16 on a partitioned GPU, say).
int k5c_kernel(const Kpz2dDev& D, const ClusterShape& cl, void** kfn) {
  int rc = jit_get("kpz2d_k5.cuh", "kpz2d_k5c_jit", k5_jit_defines(D, 2, cl.smem, &cl), kfn);
  if (rc) return rc;
  KPZ_CUDA_CHECK(cudaFuncSetAttribute(*kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)cl.smem));
  if (cl.cs > 8) KPZ_CUDA_CHECK(cudaFuncSetAttribute(*kfn, cudaFuncAttributeNonPortableClusterSizeAllowed, 1));
  cudaLaunchConfig_t cfg{};
  cfg.gridDim = dim3(cl.cs);
  cfg.blockDim = dim3(cl.threads);
  cfg.dynamicSmemBytes = cl.smem;
  cudaLaunchAttribute at{};
  at.id = cudaLaunchAttributeClusterDimension;
  at.val.clusterDim.x = cl.cs;
  at.val.clusterDim.y = at.val.clusterDim.z = 1;
  cfg.attrs = &at;
  cfg.numAttrs = 1;
  int nclusters = 0;
  KPZ_CUDA_CHECK(cudaOccupancyMaxActiveClusters(&nclusters, *kfn, &cfg));
  if (nclusters < 1)
    return fail(KPZ_EUNSUPPORTED, "this device cannot hold a cluster of %d CTAs of %d threads with %zu bytes of shared memory",
                cl.cs, cl.threads, cl.smem);
  return KPZ_OK;
}

int record2d(kpz2d_sim* sim, int ri) {
  const Kpz2dDev& D = sim->dev;
  unsigned long long* oh = (unsigned long long*)(sim->rec_h + (size_t)ri * D.S);
  unsigned long long* oh2 = (unsigned long long*)(sim->rec_h2 + (size_t)ri * D.S);
  KPZ_CUDA_CHECK(cudaMemsetAsync(oh, 0, (size_t)D.S * 8, sim->stream));
  KPZ_CUDA_CHECK(cudaMemsetAsync(oh2, 0, (size_t)D.S * 8, sim->stream));
  const int nyb = (D.Ly + 255) / 256;
  k2d_row_sums<<<D.S * nyb, 256, 0, sim->stream>>>(D.EX, D.OX, D.EY, D.Lx, D.Ly, D.RH, nyb, oh, oh2);
  KPZ_LAUNCH_CHECK("k2d_row_sums");
  return KPZ_OK;
}

}  // namespace

extern "C" {

int kpz2d_workspace_bytes(int32_t Lx, int32_t Ly, int32_t nsamples, int32_t max_records, size_t* bytes) {
  if (!bytes) return fail(KPZ_EINVAL, "bytes is NULL");
  int rc = validate2d(Lx, Ly, nsamples, max_records);
  if (rc) return rc;
  *bytes = layout2d(Lx, Ly, nsamples, max_records).total;
  return KPZ_OK;
}

int kpz2d_reset(kpz2d_sim* sim) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const Kpz2dDev& D = sim->dev;
  k2d_init_flat<<<grid_for2((size_t)D.S * D.Ly * D.RH), 256, 0, sim->stream>>>(D.EX, D.OX, D.EY, D.OY, D.S, D.Ly, D.RH);
  KPZ_LAUNCH_CHECK("k2d_init_flat");
  sim->t = 0;
  sim->nrec = 0;
  return KPZ_OK;
}

int kpz2d_create(kpz2d_sim** out, int32_t Lx, int32_t Ly, int32_t nsamples, double p, double q, uint64_t seed,
                 const kpz_options* opt, int32_t max_records, void* d_workspace, size_t workspace_bytes, void* cuda_stream) {
  if (!out) return fail(KPZ_EINVAL, "out is NULL");
  *out = nullptr;
  int rc = validate2d(Lx, Ly, nsamples, max_records);
  if (rc) return rc;
  if (!valid_prob(p) || !valid_prob(q)) return fail(KPZ_EINVAL, "p and q must lie in [0,1]");
  kpz_options o{0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1))
    return fail(KPZ_EINVAL, "options: first_sample >= 0, offset_mode in {0,1}");
  int path;
  rc = choose_path2d(Lx, Ly, &o, &path);
  if (rc) return rc;
  if (!d_workspace || ((uintptr_t)d_workspace & 255) != 0) return fail(KPZ_EINVAL, "d_workspace must be non-NULL and 256-byte aligned");
  const Layout2d y = layout2d(Lx, Ly, nsamples, max_records);
  if (workspace_bytes < y.total) return fail(KPZ_ENOMEM, "workspace has %zu bytes, %zu needed", workspace_bytes, y.total);
  kpz2d_sim* sim = new (std::nothrow) kpz2d_sim();
  if (!sim) return fail(KPZ_ENOMEM, "host allocation failed");
  char* base = (char*)d_workspace;
  Kpz2dDev& D = sim->dev;
  D.keys = make_keys(seed);
  D.t_p = make_thresh(p);
  D.t_q = make_thresh(q);
  D.offset_mode = o.offset_mode;
  D.first_sample = o.first_sample;
  D.S = nsamples;
  D.Lx = Lx;
  D.Ly = Ly;
  D.RH = y.RH;
  D.n_ew = (int32_t)((int64_t)Lx * Ly / 64);
  D.n_sg = (D.n_ew + 3) / 4;
  D.EX = (uint32_t*)(base + y.off_EX);
  D.OX = (uint32_t*)(base + y.off_OX);
  D.EY = (uint32_t*)(base + y.off_EY);
  D.OY = (uint32_t*)(base + y.off_OY);
  if (path == KPZ2D_CLUSTER) {  // a cluster of 16 CTAs is beyond the portable size: ask the device before promising it
    ClusterShape cl;
    void* kfn = nullptr;
    if (cluster_shape(Lx, Ly, &cl) && cl.cs > 8 && k5c_kernel(D, cl, &kfn) != KPZ_OK) {
      if (o.path != KPZ_PATH_AUTO) {
        delete sim;
        return KPZ_EUNSUPPORTED;  // text set by k5c_kernel
      }
      path = KPZ_PATH_STREAM;
    }
  }
  sim->max_records = max_records;
  sim->path = path;
  sim->stream = (cudaStream_t)cuda_stream;
  sim->rec_t = (long long*)(base + y.off_rec_t);
  sim->rec_h = (long long*)(base + y.off_h);
  sim->rec_h2 = (long long*)(base + y.off_h2);
  sim->off = (unsigned char*)(base + y.off_off);
  rc = kpz2d_reset(sim);
  if (rc) {
    delete sim;
    return rc;
  }
  *out = sim;
  return KPZ_OK;
}

int kpz2d_jit_check(int32_t Lx, int32_t Ly, double p, double q, const kpz_options* opt, size_t* cubin_bytes) {
  if (!cubin_bytes) return fail(KPZ_EINVAL, "cubin_bytes is NULL");
  *cubin_bytes = 0;
  int rc = validate2d(Lx, Ly, 1, 0);
  if (rc) return rc;
  if (!valid_prob(p) || !valid_prob(q)) return fail(KPZ_EINVAL, "p and q must lie in [0,1]");
  int path;
  rc = choose_path2d(Lx, Ly, opt, &path);
  if (rc) return rc;
  if (!jit_enabled()) return KPZ_OK;
  Kpz2dDev D{};
  D.t_p = make_thresh(p);
  D.t_q = make_thresh(q);
  D.Lx = Lx;
  D.Ly = Ly;
  std::vector<char> cubin;
  const bool onchip = path == KPZ_PATH_ONCHIP;
  if (path == KPZ2D_CLUSTER) {
    ClusterShape cl;
    cluster_shape(Lx, Ly, &cl);
    rc = jit_compile("kpz2d_k5.cuh", "kpz2d_k5c_jit", k5_jit_defines(D, 2, cl.smem, &cl), &cubin, nullptr);
  } else {
    rc = jit_compile("kpz2d_k5.cuh", onchip ? "kpz2d_k5s_jit" : "kpz2d_k5_pass_jit",
                     k5_jit_defines(D, onchip ? 1 : 3, onchip ? onchip_bytes(Lx, Ly) : 0), &cubin, nullptr);
  }
  if (rc) return rc;
  *cubin_bytes = cubin.size();
  return KPZ_OK;
}

int kpz2d_destroy(kpz2d_sim* sim) {
  delete sim;
  return KPZ_OK;
}

int kpz2d_time(const kpz2d_sim* sim, int64_t* t) {
  if (!sim || !t) return fail(KPZ_EINVAL, "NULL argument");
  *t = sim->t;
  return KPZ_OK;
}

int kpz2d_set_record_times(kpz2d_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return fail(KPZ_EINVAL, "bad record-time list");
  if (nt > sim->max_records) return fail(KPZ_ENOMEM, "%d record times but max_records=%d", nt, sim->max_records);
  for (int32_t k = 0; k < nt; ++k)
    if (t[k] < 1 || (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1]))
      return fail(KPZ_EINVAL, "record times must be strictly increasing and later than the current time");
  // no overflow guard is needed: |h| <= (Lx + Ly) / 2 + 1 <= 32769 and Lx * Ly <= 2^30, so sum h^2 < 2^61
  sim->rec_times.assign(t, t + nt);
  sim->nrec = 0;
  if (nt > 0) {
    KPZ_CUDA_CHECK(cudaMemcpyAsync(sim->rec_t, sim->rec_times.data(), (size_t)nt * 8, cudaMemcpyHostToDevice, sim->stream));
    KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  }
  return KPZ_OK;
}

int kpz2d_path(const kpz2d_sim* sim, int32_t* path) {
  if (!sim || !path) return fail(KPZ_EINVAL, "NULL argument");
  *path = sim->path;
  return KPZ_OK;
}

int kpz2d_run(kpz2d_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return fail(KPZ_EINVAL, "bad arguments");
  if (((uint64_t)(sim->t + n_mcs) >> 54) != 0) return fail(KPZ_EUNSUPPORTED, "time beyond 2^54 MCS");
  const Kpz2dDev D = sim->dev;
  const int nt = (int)sim->rec_times.size();
  int ri = sim->nrec;
  if (n_mcs == 0) return KPZ_OK;
  if (sim->path == KPZ_PATH_ONCHIP || sim->path == KPZ2D_CLUSTER) {
    Kpz2dRun A{};
    A.t0 = sim->t;
    A.n_mcs = n_mcs;
    A.rec_t = sim->rec_t;
    A.rec_begin = ri;
    A.nt = nt;
    A.rec_h = sim->rec_h;
    A.rec_h2 = sim->rec_h2;
    const size_t smem = onchip_bytes(D.Lx, D.Ly);
    if (sim->path == KPZ2D_CLUSTER) {  // K5C: the CTAs of a cluster add their rows' sums into the records
      ClusterShape cl;
      if (!jit_enabled() || !cluster_shape(D.Lx, D.Ly, &cl))
        return fail(KPZ_EUNSUPPORTED, "the cluster path needs run-time specialisation (kpz_debug_config jit=0 is set)");
      if (ri < nt) {
        const size_t off = (size_t)ri * D.S * 8, len = (size_t)(nt - ri) * D.S * 8;
        KPZ_CUDA_CHECK(cudaMemsetAsync((char*)sim->rec_h + off, 0, len, sim->stream));
        KPZ_CUDA_CHECK(cudaMemsetAsync((char*)sim->rec_h2 + off, 0, len, sim->stream));
      }
      void* kfn = nullptr;
      int rc = k5c_kernel(D, cl, &kfn);
      if (rc) return rc;
      void* args[] = {(void*)&D, (void*)&A};
      const int nclusters = cl.dual ? (D.S + 1) / 2 : D.S;
      KPZ_CUDA_CHECK(cudaLaunchKernel(kfn, dim3(nclusters * cl.cs), dim3(cl.threads), args, cl.smem, sim->stream));
      count_launch();
    } else if (jit_enabled()) {  // specialised on the shape and the thresholds (NVRTC)
      void* kfn = nullptr;
      int rc = jit_get("kpz2d_k5.cuh", "kpz2d_k5s_jit", k5_jit_defines(D, 1, smem), &kfn);
      if (rc) return rc;
      void* args[] = {(void*)&D, (void*)&A};
      KPZ_CUDA_CHECK(cudaFuncSetAttribute(kfn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      KPZ_CUDA_CHECK(cudaLaunchKernel(kfn, dim3(D.S), dim3(kK5SThreads), args, smem, sim->stream));
      count_launch();
    } else {
      using OnchipFn = void (*)(const Kpz2dDev, const Kpz2dRun);
      const OnchipFn fn = D.RH % 4 == 0 ? (two_planes(D) ? k2d_onchip<true, true> : k2d_onchip<true, false>)
                                        : (two_planes(D) ? k2d_onchip<false, true> : k2d_onchip<false, false>);
      KPZ_CUDA_CHECK(cudaFuncSetAttribute(fn, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem));
      fn<<<D.S, kK5SThreads, smem, sim->stream>>>(D, A);
      KPZ_LAUNCH_CHECK("k2d_onchip");
    }
    sim->t += n_mcs;
    while (sim->nrec < nt && sim->rec_times[sim->nrec] <= sim->t) sim->nrec++;
    return KPZ_OK;
  }
  using PassFn = void (*)(const Kpz2dDev, const unsigned char*, long long, int);
  const PassFn pass_fn = D.RH % 4 == 0 ? (two_planes(D) ? k2d_pass<true, true> : k2d_pass<true, false>)
                                       : (two_planes(D) ? k2d_pass<false, true> : k2d_pass<false, false>);
  void* pass_jit = nullptr;
  const bool pdl = debug_int("K5J_PDL", 1) != 0;
  if (jit_enabled()) {
    int rc = jit_get("kpz2d_k5.cuh", "kpz2d_k5_pass_jit", k5_jit_defines(D, 3, 0), &pass_jit);
    if (rc) return rc;
  }
  const long long p_begin = 2 * (long long)sim->t, p_end = 2 * (long long)(sim->t + n_mcs);
  const long long nthreads = (long long)D.S * D.n_sg;
  const unsigned nblocks = (unsigned)((nthreads + 127) / 128);
  for (long long c0 = p_begin; c0 < p_end; c0 += kChunkPasses) {
    const int np = (int)std::min<long long>(kChunkPasses, p_end - c0);
    k2d_offsets<<<grid_for2((size_t)np * D.S), 256, 0, sim->stream>>>(D.keys, D.first_sample, D.S, c0, np, D.offset_mode,
                                                                    sim->off);
    KPZ_LAUNCH_CHECK("k2d_offsets");
    for (int k = 0; k < np; ++k) {
      const long long gp = c0 + k;
      const long long m = gp >> 1;
      const int ps = (int)(gp & 1);
      if (pass_jit) {
        const unsigned char* off_k = sim->off + (size_t)k * D.S;
        long long m_arg = m;
        int ps_arg = ps;
        void* args[] = {(void*)&D, (void*)&off_k, (void*)&m_arg, (void*)&ps_arg};
        cudaLaunchConfig_t cfg{};
        cfg.gridDim = dim3(nblocks);
        cfg.blockDim = dim3(128);
        cfg.stream = sim->stream;
        cudaLaunchAttribute at{};
        at.id = cudaLaunchAttributeProgrammaticStreamSerialization;
        at.val.programmaticStreamSerializationAllowed = 1;  // the next pass may start to launch while this one runs
        cfg.attrs = &at;
        cfg.numAttrs = pdl ? 1 : 0;
        KPZ_CUDA_CHECK(cudaLaunchKernelExC(&cfg, pass_jit, args));
        count_launch();
      } else {
        pass_fn<<<nblocks, 128, 0, sim->stream>>>(D, sim->off + (size_t)k * D.S, m, ps);
        KPZ_LAUNCH_CHECK("k2d_pass");
      }
      if (ps == 1 && ri < nt && sim->rec_times[ri] == m + 1) {
        int rc = record2d(sim, ri);
        if (rc) return rc;
        ++ri;
      }
    }
  }
  sim->t += n_mcs;
  sim->nrec = ri;
  return KPZ_OK;
}

int kpz2d_slopes(kpz2d_sim* sim, uint32_t* d_sx, uint32_t* d_sy) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const Kpz2dDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.Ly * D.RH;
  if (d_sx) {
    k2d_eo_to_nat<<<grid_for2(n), 256, 0, sim->stream>>>(D.EX, D.OX, n, d_sx);
    KPZ_LAUNCH_CHECK("k2d_eo_to_nat");
  }
  if (d_sy) {
    k2d_eo_to_nat<<<grid_for2(n), 256, 0, sim->stream>>>(D.EY, D.OY, n, d_sy);
    KPZ_LAUNCH_CHECK("k2d_eo_to_nat");
  }
  return KPZ_OK;
}

int kpz2d_set_slopes(kpz2d_sim* sim, const uint32_t* d_sx, const uint32_t* d_sy) {
  if (!sim) return fail(KPZ_EINVAL, "NULL handle");
  const Kpz2dDev& D = sim->dev;
  const size_t n = (size_t)D.S * D.Ly * D.RH;
  if (d_sx) {
    k2d_nat_to_eo<<<grid_for2(n), 256, 0, sim->stream>>>(d_sx, n, D.EX, D.OX);
    KPZ_LAUNCH_CHECK("k2d_nat_to_eo");
  }
  if (d_sy) {
    k2d_nat_to_eo<<<grid_for2(n), 256, 0, sim->stream>>>(d_sy, n, D.EY, D.OY);
    KPZ_LAUNCH_CHECK("k2d_nat_to_eo");
  }
  return KPZ_OK;
}

int kpz2d_heights(kpz2d_sim* sim, int32_t sample, int32_t* d_h) {
  if (!sim || !d_h || sample < 0 || sample >= sim->dev.S) return fail(KPZ_EINVAL, "bad arguments");
  const Kpz2dDev& D = sim->dev;
  const int nxb = (D.Lx + 255) / 256;
  const size_t row0 = (size_t)sample * D.Ly * D.RH;
  k2d_heights<<<nxb, 256, 0, sim->stream>>>(D.EX + row0, D.OX + row0, D.EY + row0, D.OY + row0, D.Lx, D.Ly, D.RH, d_h);
  KPZ_LAUNCH_CHECK("k2d_heights");
  return KPZ_OK;
}

int kpz2d_roughness(kpz2d_sim* sim, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean) {
  if (!sim || !nt) return fail(KPZ_EINVAL, "NULL argument");
  if (*nt < sim->nrec) return fail(KPZ_ENOMEM, "capacity %d < %d records", *nt, sim->nrec);
  const int32_t n = sim->nrec, S = sim->dev.S;
  const size_t cells = (size_t)n * S;
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
    KPZ_CUDA_CHECK(cudaMemcpyAsync(ph, sim->rec_h, cells * 8, cudaMemcpyDeviceToHost, sim->stream));
    KPZ_CUDA_CHECK(cudaMemcpyAsync(ph2, sim->rec_h2, cells * 8, cudaMemcpyDeviceToHost, sim->stream));
  }
  KPZ_CUDA_CHECK(cudaStreamSynchronize(sim->stream));
  const double N = (double)sim->dev.Lx * (double)sim->dev.Ly;
  for (int32_t k = 0; k < n; ++k) {
    if (t) t[k] = sim->rec_times[k];
    if (w2_mean) {
      double acc = 0.0;  // Eq. 3 squared per sample over the Lx * Ly sites, averaged over samples
      for (int32_t s = 0; s < S; ++s) {
        const __int128 s1 = ph[(size_t)k * S + s], s2 = ph2[(size_t)k * S + s];
        const __int128 num = (__int128)((int64_t)sim->dev.Lx * sim->dev.Ly) * s2 - s1 * s1;
        acc += (double)num / (N * N);
      }
      w2_mean[k] = acc / (double)S;
    }
  }
  *nt = n;
  return KPZ_OK;
}

}  // extern "C"
