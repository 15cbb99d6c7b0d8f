// kpz_k3.cuh — K3: streamed sweep for rings beyond on-chip memory (SURVEY §8(a) a4/a5 "ping-pong", north_star (2))
// and the multi-CTA exact height reduction (north_star (3)).
//
// One launch per sub-lattice pass.  The ring lives in HBM/L2 de-interleaved (even-site words E, odd-site words O),
// read with 128-bit coalesced loads (one unit = 4+4 words per thread), updated in registers with the same
// bit-plane comparator as K1, and written to the other buffer of a ping-pong pair (so the single neighbour word a
// frame change needs — the "halo", PAPER.md:128 — is always read from an unmodified buffer: no race, no extra
// pass).  The frame of the stored lattice follows the offsets: a pass with the same offset as the previous one
// touches no neighbour at all.
#pragma once
#include "height_lut.cuh"
#include "kpz_k1.cuh"

namespace kpz {

// Offsets of a chunk of passes: off[(k+1)*S + s] = o of pass k (global pass index k0+k) of sample s;
// row 0 is filled by the caller (frame of the stored lattice).
__global__ void k3_offsets(const __grid_constant__ PhiloxKeys K, int first_sample, int S, long long pass0, int npasses,
                           int offset_mode, unsigned char* off) {
  const size_t n = (size_t)npasses * S;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int k = (int)(i / S), s = (int)(i % S);
    const unsigned long long gp = (unsigned long long)pass0 + (unsigned)k;
    const unsigned long long m = gp >> 1;
    const uint32_t pass = (uint32_t)(gp & 1);
    uint32_t o = pass;
    if (offset_mode == 0) {
      const uint4 w = philox4x32_10(0u, (uint32_t)(first_sample + s), (uint32_t)m,
                                    ctr3(TAG_OFFSET, pass, 0, (uint32_t)(m >> 32)), K);
      o = w.x & 1u;
    }
    off[(size_t)(k + 1) * S + s] = (unsigned char)o;
  }
}

__global__ void k3_copy_row(unsigned char* dst, const unsigned char* src, int n) {
  for (int i = blockIdx.x * blockDim.x + threadIdx.x; i < n; i += gridDim.x * blockDim.x) dst[i] = src ? src[i] : 0;
}


template <bool PARTIAL, int DIS, int NPS>
__global__ void __launch_bounds__(256) k3_pass_kernel(const __grid_constant__ KpzDev D, const __grid_constant__ K3Pass A) {
  const size_t nunits = (size_t)D.S * D.U;
  const size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x;
  if (g >= nunits) return;
  const int s = (int)(g / D.U);
  const int u = (int)(g % D.U);
  const int nw = PARTIAL ? min(4, D.PW - 4 * u) : 4;
  const size_t srow = (size_t)s * D.PWp;
  const size_t row = srow + 4 * (size_t)u;
  const int fin = A.fin[s];
  const int o = A.fo ? A.fo[s] : 0;

  uint32_t P[4], Q[4];
  {
    const uint4 e = *reinterpret_cast<const uint4*>(A.Ein + row);
    const uint4 q = *reinterpret_cast<const uint4*>(A.Oin + row);
    P[0] = e.x; P[1] = e.y; P[2] = e.z; P[3] = e.w;
    Q[0] = q.x; Q[1] = q.y; Q[2] = q.z; Q[3] = q.w;
  }
  if (fin != o) {
    if (o) {
      const int nxt = (u + 1 >= D.U) ? 0 : u + 1;
      shift_up<PARTIAL>(P, nw, A.Ein[srow + 4 * (size_t)nxt]);
    } else {
      const int prv = (u == 0) ? D.U - 1 : u - 1;
      const int nwp = PARTIAL ? min(4, D.PW - 4 * prv) : 4;
      shift_down<PARTIAL>(P, nw, A.Ein[srow + 4 * (size_t)prv + nwp - 1]);
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
      if (o) {
        const int nxt = (u + 1 >= D.U) ? 0 : u + 1;
        shift_up<PARTIAL>(sqb, nw, D.SQE[srow + 4 * (size_t)nxt]);
      }
    }
    const uint32_t gs = (uint32_t)(D.first_sample + s);
    const uint32_t c3 = ctr3(TAG_PAIR, (uint32_t)A.pass, 0, (uint32_t)((unsigned long long)A.m >> 32));
    if (o == 0) pass_update<DIS, NPS>(P, Q, spa, sqb, D, (uint32_t)u, gs, (uint32_t)A.m, c3);
    else pass_update<DIS, NPS>(Q, P, spa, sqb, D, (uint32_t)u, gs, (uint32_t)A.m, c3);
  }
  *reinterpret_cast<uint4*>(A.Eout + row) = make_uint4(P[0], P[1], P[2], P[3]);
  *reinterpret_cast<uint4*>(A.Oout + row) = make_uint4(Q[0], Q[1], Q[2], Q[3]);
}

// ---- multi-CTA exact reduction of sum h, sum h^2 (frame-0 lattice) ---------------------------------------
// A tile = 256 units (65536 sites) = one CTA.  Phase A: tile totals; phase B: exclusive scan per sample;
// phase C: per-unit relative sums lifted by (tile base + in-tile exclusive scan), int64, one atomicAdd pair per CTA.

__device__ __forceinline__ int block_exclusive_scan_256(int v, int* smem /* >= 8 */, int& total) {
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

template <bool PARTIAL>
__global__ void __launch_bounds__(256) k3_tile_totals(const uint32_t* E, const uint32_t* O, int S, int U, int PW, int PWp,
                                                      int ntiles, int* tile_tot) {
  __shared__ int sm[8];
  const int s = blockIdx.x / ntiles, tile = blockIdx.x % ntiles;
  const int u = tile * 256 + threadIdx.x;
  int r = 0;
  if (u < U) {
    const int nw = PARTIAL ? min(4, PW - 4 * u) : 4;
    const size_t row = (size_t)s * PWp + 4 * (size_t)u;
    const uint4 e = *reinterpret_cast<const uint4*>(E + row);
    const uint4 q = *reinterpret_cast<const uint4*>(O + row);
    r = 2 * (__popc(e.x) + __popc(e.y) + __popc(e.z) + __popc(e.w) + __popc(q.x) + __popc(q.y) + __popc(q.z) + __popc(q.w)) -
        64 * nw;
  }
  int total;
  block_exclusive_scan_256(r, sm, total);
  if (threadIdx.x == 0) tile_tot[(size_t)s * ntiles + tile] = total;
  (void)S;
}

// exclusive scan of each sample's tile totals (one block of 1024 threads per sample)
__global__ void k3_scan_tiles(int* tile_tot, int ntiles) {
  __shared__ int warp_tot[32];
  __shared__ int chunk_total;
  int* data = tile_tot + (size_t)blockIdx.x * ntiles;
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

// max over the units of |height before the unit| (the overflow guard after kpz_set_lattice): inside a unit
// the height moves by at most 256 more.
__global__ void __launch_bounds__(256) k3_tile_absmax(const uint32_t* E, const uint32_t* O, int U, int PW, int PWp,
                                                      int ntiles, const int* tile_base, int* out) {
  __shared__ int sm[8];
  const int s = blockIdx.x / ntiles, tile = blockIdx.x % ntiles;
  const int u = tile * 256 + threadIdx.x;
  int r = 0;
  if (u < U) {
    const int nw = min(4, PW - 4 * u);
    const size_t row = (size_t)s * PWp + 4 * (size_t)u;
    const uint4 e = *reinterpret_cast<const uint4*>(E + row);
    const uint4 q = *reinterpret_cast<const uint4*>(O + row);
    r = 2 * (__popc(e.x) + __popc(e.y) + __popc(e.z) + __popc(e.w) + __popc(q.x) + __popc(q.y) + __popc(q.z) + __popc(q.w)) -
        64 * nw;  // pad words are zero
  }
  int total;
  const int base = tile_base[(size_t)s * ntiles + tile] + block_exclusive_scan_256(r, sm, total);
  int m = u < U ? abs(base) : 0;
#pragma unroll
  for (int d = 16; d >= 1; d >>= 1) m = max(m, __shfl_xor_sync(0xFFFFFFFFu, m, d));
  if ((threadIdx.x & 31) == 0 && m > 0) atomicMax(out, m);
}

template <bool PARTIAL>
__global__ void __launch_bounds__(256) k3_tile_sums(const uint32_t* E, const uint32_t* O, int S, int U, int PW, int PWp,
                                                    int ntiles, const int* tile_base, unsigned long long* out_h,
                                                    unsigned long long* out_h2) {
  __shared__ int sm[8];
  __shared__ long long red[16];
  __shared__ uint32_t lut[256];
  lut[threadIdx.x] = height_lut_entry((int)threadIdx.x);
  __syncthreads();
  const int s = blockIdx.x / ntiles, tile = blockIdx.x % ntiles;
  const int u = tile * 256 + threadIdx.x;
  int r = 0, s1 = 0, s2 = 0, nw = 0;
  if (u < U) {
    nw = PARTIAL ? min(4, PW - 4 * u) : 4;
    const size_t row = (size_t)s * PWp + 4 * (size_t)u;
    const uint4 e = *reinterpret_cast<const uint4*>(E + row);
    const uint4 q = *reinterpret_cast<const uint4*>(O + row);
    const uint32_t P[4] = {e.x, e.y, e.z, e.w}, Q[4] = {q.x, q.y, q.z, q.w};
    unit_relative_sums_lut(P, Q, nw, lut, r, s1, s2);
  }
  int total;
  const long long base = (long long)tile_base[(size_t)s * ntiles + tile] + block_exclusive_scan_256(r, sm, total);
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
    atomicAdd(out_h + s, (unsigned long long)a);   // exact: two's-complement wrap-around addition
    atomicAdd(out_h2 + s, (unsigned long long)b);
  }
  (void)S;
}

}  // namespace kpz
