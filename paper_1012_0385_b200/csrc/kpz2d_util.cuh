// kpz2d_util.cuh — the helper kernels of the 2+1D path that only the library build needs (initialisation, layout
// conversion at the ABI, colour offsets of a chunk of passes, heights / exact sums from the planes in HBM).  The sweep
// kernels themselves are in kpz2d_k5.cuh (also compiled at run time).
#pragma once
#include "common.cuh"
#include "kpz2d_k5.cuh"

namespace kpz {

// flat start h = (x + y) & 1: sx = sy = (x + y) & 1, i.e. even sites carry y & 1, odd sites its complement
__global__ void k2d_init_flat(uint32_t* EX, uint32_t* OX, uint32_t* EY, uint32_t* OY, int S, int Ly, int RH) {
  const size_t n = (size_t)S * Ly * RH;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int y = (int)((i / RH) % Ly);
    const uint32_t e = (y & 1) ? 0xFFFFFFFFu : 0u;
    EX[i] = e;
    OX[i] = ~e;
    EY[i] = e;
    OY[i] = ~e;
  }
}

// natural words [rows][2 RH] <-> parity planes [rows][RH]
__global__ void k2d_nat_to_eo(const uint32_t* words, size_t n /* rows * RH */, uint32_t* E, uint32_t* O) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const uint2 w = reinterpret_cast<const uint2*>(words)[i];
    uint32_t e, o;
    nat_to_eo(w.x, w.y, e, o);
    E[i] = e;
    O[i] = o;
  }
}
__global__ void k2d_eo_to_nat(const uint32_t* E, const uint32_t* O, size_t n, uint32_t* words) {
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    uint32_t w0, w1;
    eo_to_nat(E[i], O[i], w0, w1);
    reinterpret_cast<uint2*>(words)[i] = make_uint2(w0, w1);
  }
}

// offsets of np passes starting at global pass index p0 (pass = 2 m + ps): out[k * S + s]
__global__ void k2d_offsets(const __grid_constant__ PhiloxKeys K, int first_sample, int S, long long p0, int np, int offset_mode,
                            unsigned char* out) {
  const size_t n = (size_t)np * S;
  for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
    const int k = (int)(i / S), s = (int)(i % S);
    const unsigned long long gp = (unsigned long long)(p0 + k);
    const unsigned long long m = gp >> 1;
    const uint32_t ps = (uint32_t)(gp & 1ull);
    uint32_t o = ps;
    if (offset_mode == 0)
      o = philox4x32_10(0u, (uint32_t)(first_sample + s), (uint32_t)m, ctr3(TAG_OFFSET, ps, 0, (uint32_t)(m >> 32)), K).x & 1u;
    out[i] = (unsigned char)o;
  }
}

// Heights of one sample, column by column - the definition of DESIGN §R19 written out (thread = column x):
// h(x,0) = 2 (occupied bonds among sx[0][0..x]) - (x + 1): even sites 0..x are bits 0..x/2 of EX[0], odd ones bits
// 0..(x-1)/2 of OX[0]; h(x,y) = h(x,y-1) + 2 sy[y][x] - 1.  (The exact sums at record times integrate row by row:
// k2d_row_sums below, row_sums_onchip in kpz2d_k5.cuh; a GPU test compares the two.)
__global__ void __launch_bounds__(256) k2d_heights(const uint32_t* __restrict__ EX, const uint32_t* __restrict__ OX,
                                                   const uint32_t* __restrict__ EY, const uint32_t* __restrict__ OY, int Lx, int Ly,
                                                   int RH, int32_t* h_out) {
  const int x = blockIdx.x * 256 + threadIdx.x;
  if (x >= Lx) return;
  const int ne = x / 2 + 1, no = (x + 1) / 2;
  int cnt = 0;
  for (int w = 0; w < (ne >> 5); ++w) cnt += __popc(EX[w]);
  if (ne & 31) cnt += __popc(EX[ne >> 5] & ((1u << (ne & 31)) - 1u));
  for (int w = 0; w < (no >> 5); ++w) cnt += __popc(OX[w]);
  if (no & 31) cnt += __popc(OX[no >> 5] & ((1u << (no & 31)) - 1u));
  int h = 2 * cnt - (x + 1);
  const uint32_t* col = (x & 1) ? OY : EY;
  const int jw = (x >> 1) >> 5, jb = (x >> 1) & 31;
  for (int y = 0; y < Ly; ++y) {
    if (y > 0) h += 2 * (int)((col[(size_t)y * RH + jw] >> jb) & 1u) - 1;
    h_out[(size_t)y * Lx + x] = h;
  }
}

// Exact sums over every sample from the planes in HBM, row by row (see row_sums_onchip): grid = S * nyb blocks of 256
// rows; a block first adds up column 0 of sy over the rows before its own (the height of its first row's site 0).
__global__ void __launch_bounds__(256) k2d_row_sums(const uint32_t* __restrict__ EX, const uint32_t* __restrict__ OX,
                                                    const uint32_t* __restrict__ EY, int Lx, int Ly, int RH, int nyb,
                                                    unsigned long long* out_h, unsigned long long* out_h2) {
  __shared__ long long red[16];
  __shared__ uint32_t lut[256];
  __shared__ int scan[8];
  lut[threadIdx.x] = height_lut_entry((int)threadIdx.x);
  const int s = blockIdx.x / nyb, y_first = (blockIdx.x % nyb) * 256;
  const size_t base = (size_t)s * Ly * RH;
  const uint32_t *ex = EX + base, *ox = OX + base, *ey = EY + base;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  auto block_total = [&](int v) {  // sum over the block, to every thread
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) v += __shfl_xor_sync(0xFFFFFFFFu, v, d);
    __syncthreads();
    if (lane == 0) scan[warp] = v;
    __syncthreads();
    int t = 0;
#pragma unroll
    for (int k = 0; k < 8; ++k) t += scan[k];
    return t;
  };
  int pre = 0;
  for (int yy = 1 + (int)threadIdx.x; yy < y_first; yy += 256) pre += 2 * (int)(ey[(size_t)yy * RH] & 1u) - 1;
  const int h_before = 2 * (int)(ex[0] & 1u) - 1 + block_total(pre);  // h(0, y_first - 1), or h(0,0) for the first block
  const int y = y_first + (int)threadIdx.x;
  const bool live = y < Ly;
  const size_t row = (size_t)(live ? y : 0) * RH;
  const int d = (live && y > 0) ? 2 * (int)(ey[row] & 1u) - 1 : 0;
  int incl = d;
#pragma unroll
  for (int k = 1; k < 32; k <<= 1) {
    const int v = __shfl_up_sync(0xFFFFFFFFu, incl, k);
    if (lane >= k) incl += v;
  }
  __syncthreads();
  if (lane == 31) scan[warp] = incl;
  __syncthreads();
  int add = 0;
#pragma unroll
  for (int k = 0; k < 8; ++k)
    if (k < warp) add += scan[k];
  long long s1 = 0, s2 = 0;
  if (live) {
    const long long B = (long long)(h_before + add + incl) - (2 * (int)(ex[row] & 1u) - 1);
    long long S1, S2;
    row_relative_sums(ex + row, ox + row, RH, lut, S1, S2);
    s1 = (long long)Lx * B + S1;
    s2 = (long long)Lx * B * B + 2 * B * S1 + S2;
  }
  block_sum2<8>(s1, s2, red);
  if (threadIdx.x == 0) {
    atomicAdd(out_h + s, (unsigned long long)s1);  // exact: two's-complement wrap-around addition
    atomicAdd(out_h2 + s, (unsigned long long)s2);
  }
}

}  // namespace kpz
