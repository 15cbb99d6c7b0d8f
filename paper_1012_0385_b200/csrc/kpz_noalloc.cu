// kpz_noalloc.cu — kpz_noalloc_height_sums of include/kpz_b200.h: the exact sums behind the width W of Eq. 3
// of rings the caller hands in, for callers that cannot allocate (code under CUDA graph
// capture, serving loops, harnesses that forbid cudaMalloc): no handle, no workspace, no device or host allocation.
//
// It is a variant of the multi-CTA reduction of the streamed paths (kpz_k3.cuh: tile totals -> exclusive scan per ring
// -> lifted per-unit sums), reading the NATURAL layout directly.  That reduction needs one int of scratch per tile of
// 65536 sites; here the scratch is the file-scope device array g_tile_scratch below (kMaxTiles ints = 256 KiB, held by
// every GPU that loads the library until the process exits).  Host code must not hand `g_tile_scratch` itself to a
// kernel - in host code the name is a host-side stand-in - so its device address is looked up once per device with
// cudaGetSymbolAddress, with that device current.
//
// Every call shares the array and it keeps the last call's contents.  With several tiles per ring, entries
// [0, nsamples * ntiles) are all written by phase A before phase B reads them; with one tile per ring the tile bases
// must be zero and are cleared (phases A and B are skipped); the two output arrays are accumulated with atomics and are
// cleared first.  Calls that overlap on the GPU (two streams, two host threads) race on the array.
#include <mutex>

#include "common.cuh"
#include "height_lut.cuh"

using namespace kpz;

// The scratch of every call on this device: tile totals, then tile bases.  256 KiB of device memory per GPU.
static __device__ __align__(256) int g_tile_scratch[KPZ_NOALLOC_MAX_TILES];

namespace {

constexpr int kTileUnits = 256;                        // units of 256 sites per tile: one CTA, 65536 sites
constexpr int kMaxTiles = KPZ_NOALLOC_MAX_TILES;       // nsamples * ceil(L / 65536) may not exceed this
constexpr int kMaxDevices = 64;

// Exclusive scan of one int per thread over a CTA of 256 threads; total = sum over the CTA.
__device__ __forceinline__ int cta_exclusive_scan(int v, int* smem /* 8 */, int& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int incl = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) {
    const int x = __shfl_up_sync(0xFFFFFFFFu, incl, d);
    if (lane >= d) incl += x;
  }
  __syncthreads();
  if (lane == 31) smem[warp] = incl;
  __syncthreads();
  int add = 0, tot = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k) {
    const int t = smem[k];
    if (k < warp) add += t;
    tot += t;
  }
  total = tot;
  return add + incl - v;
}

// The 8 natural words (256 sites) of unit u of ring s; words beyond the ring read as 0.  nw8 = words that exist.
__device__ __forceinline__ int load_unit(const uint32_t* words, size_t ring, int PWn, int u, uint32_t (&w)[8]) {
  const int nw8 = min(8, PWn - 8 * u);
  const uint32_t* p = words + ring * (size_t)PWn + 8 * (size_t)u;
  if (nw8 == 8 && ((PWn & 3) == 0)) {  // rows stay 16-byte aligned
    const uint4 a = __ldg(reinterpret_cast<const uint4*>(p)), b = __ldg(reinterpret_cast<const uint4*>(p) + 1);
    w[0] = a.x, w[1] = a.y, w[2] = a.z, w[3] = a.w, w[4] = b.x, w[5] = b.y, w[6] = b.z, w[7] = b.w;
  } else {
#pragma unroll
    for (int k = 0; k < 8; ++k) w[k] = k < nw8 ? __ldg(p + k) : 0u;
  }
  return nw8;
}

// Phase A: total slope of every tile -> scratch[s * ntiles + tile]
__global__ void __launch_bounds__(256) na_tile_totals(const uint32_t* words, int U, int PWn, int ntiles, int* scratch) {
  __shared__ int sm[8];
  const int s = blockIdx.x / ntiles, tile = blockIdx.x % ntiles;
  const int u = tile * kTileUnits + threadIdx.x;
  int r = 0;
  if (u < U) {
    uint32_t w[8];
    const int nw8 = load_unit(words, (size_t)s, PWn, u, w);
    int pc = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) pc += __popc(w[k]);
    r = 2 * pc - 32 * nw8;
  }
  int total;
  cta_exclusive_scan(r, sm, total);
  if (threadIdx.x == 0) scratch[(size_t)s * ntiles + tile] = total;
}

// Phase B: exclusive scan of each ring's tile totals, in place (one CTA of 1024 threads per ring)
__global__ void __launch_bounds__(1024) na_scan_tiles(int* scratch, int ntiles) {
  __shared__ int warp_tot[32];
  __shared__ int chunk_total;
  int* data = scratch + (size_t)blockIdx.x * ntiles;
  int carry = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < ntiles; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = i < ntiles ? data[i] : 0;
    int incl = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
      const int x = __shfl_up_sync(0xFFFFFFFFu, incl, d);
      if (lane >= d) incl += x;
    }
    if (lane == 31) warp_tot[warp] = incl;
    __syncthreads();
    int add = 0;
    for (int k = 0; k < warp; ++k) add += warp_tot[k];
    if (threadIdx.x == 1023) chunk_total = incl + add;
    if (i < ntiles) data[i] = carry + add + incl - v;
    __syncthreads();
    carry += chunk_total;
    __syncthreads();
  }
}

// Phase C: sums of h and h^2 over each unit relative to the site before it (byte table of height_lut.cuh), lifted by
// the height before the unit = tile base (scratch) + in-tile exclusive scan; one atomic pair per CTA.
__global__ void __launch_bounds__(256) na_tile_sums(const uint32_t* words, int U, int PWn, int ntiles, const int* scratch,
                                                    unsigned long long* out_h, unsigned long long* out_h2) {
  __shared__ int sm[8];
  __shared__ long long red[16];
  __shared__ uint32_t lut[256];
  lut[threadIdx.x] = height_lut_entry((int)threadIdx.x);
  __syncthreads();
  const int s = blockIdx.x / ntiles, tile = blockIdx.x % ntiles;
  const int u = tile * kTileUnits + threadIdx.x;
  int r = 0, s1 = 0, s2 = 0, nw = 0;
  if (u < U) {
    uint32_t w[8];
    nw = load_unit(words, (size_t)s, PWn, u, w) / 2;  // L is a multiple of 64: whole pairs of words
    uint32_t P[4], Q[4];
#pragma unroll
    for (int k = 0; k < 4; ++k) nat_to_eo(w[2 * k], w[2 * k + 1], P[k], Q[k]);
    unit_relative_sums_lut(P, Q, nw, lut, r, s1, s2);
  }
  int total;
  const long long base = (long long)scratch[(size_t)s * ntiles + tile] + cta_exclusive_scan(r, sm, total);
  const long long n = 64LL * nw;
  long long H = n * base + (long long)s1;
  long long H2 = n * base * base + 2LL * base * (long long)s1 + (long long)s2;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) {
    H += __shfl_down_sync(0xFFFFFFFFu, H, d);
    H2 += __shfl_down_sync(0xFFFFFFFFu, H2, d);
  }
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  if (lane == 0) {
    red[warp] = H;
    red[8 + warp] = H2;
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

// Device address of g_tile_scratch on the current device, looked up once per device.
std::mutex g_mu;
int* g_scratch_addr[kMaxDevices] = {};

int scratch_for_current_device(int** out) {
  int dev = -1;
  KPZ_CUDA_CHECK(cudaGetDevice(&dev));
  if (dev < 0 || dev >= kMaxDevices) return fail(KPZ_EUNSUPPORTED, "device index %d beyond the %d this entry point tracks", dev, kMaxDevices);
  std::lock_guard<std::mutex> lock(g_mu);
  if (!g_scratch_addr[dev]) {
    int* p = nullptr;
    KPZ_CUDA_CHECK(cudaGetSymbolAddress((void**)&p, g_tile_scratch));
    if (!p) return fail(KPZ_ECUDA, "cudaGetSymbolAddress returned a NULL address for the scratch array");
    g_scratch_addr[dev] = p;
  }
  *out = g_scratch_addr[dev];
  return KPZ_OK;
}

}  // namespace

extern "C" int kpz_noalloc_height_sums(const uint32_t* d_words, int64_t L, int32_t nsamples, int64_t* d_sum_h,
                                       int64_t* d_sum_h2, void* cuda_stream) {
  if (!d_words || !d_sum_h || !d_sum_h2) return fail(KPZ_EINVAL, "NULL pointer");
  if (((uintptr_t)d_words & 15) != 0 || ((uintptr_t)d_sum_h & 7) != 0 || ((uintptr_t)d_sum_h2 & 7) != 0)
    return fail(KPZ_EINVAL, "d_words must be 16-byte aligned, d_sum_h / d_sum_h2 8-byte aligned");
  if (L < 64 || nsamples < 1) return fail(KPZ_EINVAL, "need L >= 64 and nsamples >= 1");
  if (L % 64 != 0) return fail(KPZ_EUNSUPPORTED, "L must be a multiple of 64 (L=%lld)", (long long)L);
  if (L > ((int64_t)1 << 30)) return fail(KPZ_EUNSUPPORTED, "L beyond 2^30: heights would leave int32 (L=%lld)", (long long)L);
  const int64_t ntiles = (L + 65535) / 65536;
  if ((int64_t)nsamples * ntiles > kMaxTiles)
    return fail(KPZ_EUNSUPPORTED,
                "nsamples * ceil(L / 65536) = %lld tiles, the static scratch of this entry point holds %d "
                "(KPZ_NOALLOC_MAX_TILES); split the batch or use kpz_create + kpz_roughness",
                (long long)((int64_t)nsamples * ntiles), kMaxTiles);
  int* scratch = nullptr;
  int rc = scratch_for_current_device(&scratch);
  if (rc) return rc;
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const int PWn = (int)(L / 32), U = (int)((L + 255) / 256), nt = (int)ntiles;
  KPZ_CUDA_CHECK(cudaMemsetAsync(d_sum_h, 0, (size_t)nsamples * 8, st));
  KPZ_CUDA_CHECK(cudaMemsetAsync(d_sum_h2, 0, (size_t)nsamples * 8, st));
  if (nt > 1) {
    na_tile_totals<<<nsamples * nt, 256, 0, st>>>(d_words, U, PWn, nt, scratch);
    KPZ_LAUNCH_CHECK("na_tile_totals");
    na_scan_tiles<<<nsamples, 1024, 0, st>>>(scratch, nt);
    KPZ_LAUNCH_CHECK("na_scan_tiles");
  } else {  // one tile per ring: its base is the height before site 0 = 0; the array still holds the last call's values
    KPZ_CUDA_CHECK(cudaMemsetAsync(scratch, 0, (size_t)nsamples * sizeof(int), st));
  }
  na_tile_sums<<<nsamples * nt, 256, 0, st>>>(d_words, U, PWn, nt, scratch, (unsigned long long*)d_sum_h,
                                              (unsigned long long*)d_sum_h2);
  KPZ_LAUNCH_CHECK("na_tile_sums");
  return KPZ_OK;
}
