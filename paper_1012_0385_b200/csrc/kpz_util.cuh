// kpz_util.cuh — initialisation, layout conversion and height kernels of the KPZ ensemble.
#pragma once
#include "common.cuh"

namespace kpz {

// Flat start n_i = i & 1: even sites empty, odd sites occupied; pad words are zero.
__global__ void k_init_flat(uint32_t* E, uint32_t* O, int S, int PW, int PWp) {
  const size_t n = (size_t)S * PWp;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int w = (int)(i % PWp);
    E[i] = 0u;
    O[i] = (w < PW) ? 0xFFFFFFFFu : 0u;
  }
}

// Quenched Bernoulli site mask (Eq. 8) written in de-interleaved layout.
// Thread = one supergroup of 128 sites = 2 pair-words.
__global__ void k_site_mask_eo(const __grid_constant__ PhiloxKeys K, uint32_t tag, Thresh T, int first_sample,
                               int S, int PW, int PWp, uint32_t* ME, uint32_t* MO) {
  const int ngroups = (PW + 1) / 2;
  const size_t n = (size_t)S * ngroups;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int s = (int)(i / ngroups), G = (int)(i % ngroups);
    const uint4 m = bernoulli128(K, tag, (uint32_t)(first_sample + s), 0u, 0u, (uint32_t)G, T);
    uint32_t e, o;
    nat_to_eo(m.x, m.y, e, o);
    ME[(size_t)s * PWp + 2 * G] = e;
    MO[(size_t)s * PWp + 2 * G] = o;
    if (2 * G + 1 < PW) {
      nat_to_eo(m.z, m.w, e, o);
      ME[(size_t)s * PWp + 2 * G + 1] = e;
      MO[(size_t)s * PWp + 2 * G + 1] = o;
    }
  }
}

__global__ void k_zero_words(uint32_t* p, size_t n) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) p[i] = 0u;
}

// internal (E,O)[S][PWp] -> natural words[S][2 PW]
__global__ void k_eo_to_nat(const uint32_t* E, const uint32_t* O, int S, int PW, int PWp, uint32_t* words) {
  const size_t n = (size_t)S * PW;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t s = i / PW, g = i % PW;
    uint32_t w0, w1;
    eo_to_nat(E[s * PWp + g], O[s * PWp + g], w0, w1);
    reinterpret_cast<uint2*>(words)[i] = make_uint2(w0, w1);
  }
}

__global__ void k_nat_to_eo(const uint32_t* words, int S, int PW, int PWp, uint32_t* E, uint32_t* O) {
  const size_t n = (size_t)S * PW;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const size_t s = i / PW, g = i % PW;
    const uint2 w = reinterpret_cast<const uint2*>(words)[i];
    uint32_t e, o;
    nat_to_eo(w.x, w.y, e, o);
    E[s * PWp + g] = e;
    O[s * PWp + g] = o;
  }
}

// ---- heights of one sample (kpz_heights): group totals -> exclusive scan -> expand -----------------------
__global__ void k_group_totals(const uint32_t* E, const uint32_t* O, int PW, int* tot) {
  for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < (size_t)PW; g += (size_t)gridDim.x * blockDim.x)
    tot[g] = 2 * (__popc(E[g]) + __popc(O[g])) - 64;
}

// In-place exclusive scan by ONE block of 1024 threads (carry kept in a register of every thread).
__global__ void k_exclusive_scan_1block(int* data, int n) {
  __shared__ int warp_tot[32];
  __shared__ int chunk_total;
  int carry = 0;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  for (int base = 0; base < n; base += 1024) {
    const int i = base + threadIdx.x;
    const int v = i < n ? data[i] : 0;
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
    if (i < n) data[i] = carry + add + incl - v;
    __syncthreads();
    carry += chunk_total;
    __syncthreads();
  }
}

__global__ void k_heights_expand(const uint32_t* E, const uint32_t* O, const int* base, int PW, int* h) {
  for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < (size_t)PW; g += (size_t)gridDim.x * blockDim.x) {
    int r = base[g];
    uint32_t e = E[g], o = O[g];
    int* out = h + 64 * g;
    for (int k = 0; k < 32; ++k) {
      r += 2 * (int)(e & 1u) - 1;
      out[2 * k] = r;
      r += 2 * (int)(o & 1u) - 1;
      out[2 * k + 1] = r;
      e >>= 1;
      o >>= 1;
    }
  }
}

}  // namespace kpz
