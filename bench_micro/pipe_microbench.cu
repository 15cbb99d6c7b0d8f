// pipe_microbench.cu — measures the B200 issue rates the sweep's roofline is built on.
//
// Stand-alone program (built and run by `python bench_micro/microbench.py`): for each instruction class of
// the sweep (LOP3, SHF, IMAD.WIDE, IMAD.lo, IMAD.HI, POPC, SHFL) and for mixes of IMAD.WIDE with n LOP3, every SMSP
// runs W warps with 4 independent chains per thread; it prints the cycles one "step" (NA instructions of class A + NB
// of class B) takes per SMSP.  Findings the kernels rely on: LOP3/SHF/IMAD.lo 2 clk, IMAD.WIDE 4 clk alone, and
// IMAD.WIDE + n LOP3 = max(4, 2 + 2n) clk - an IMAD.WIDE also occupies one slot of the alu pipe, so the sweep is
// bound by alu-pipe slots: 0.5 warp-instructions per clock and SMSP over {LOP3, SHF, IMAD.WIDE}.
#include <cstdint>
#include <cstdio>
#include <cuda_runtime.h>

enum { LOP3 = 0, WIDE = 1, IMADLO = 2, IMADHI = 3, SHF = 4, IADD = 5, POPC = 6, SHFL = 7 };

template <int A>
__device__ __forceinline__ void op(uint32_t& x, uint32_t& y, uint32_t s) {
  const uint32_t M0 = 0xD2511F53u;
  if (A == LOP3) asm volatile("lop3.b32 %0, %0, %1, %2, 0x96;" : "+r"(x) : "r"(y), "r"(s));
  else if (A == WIDE) {
    unsigned long long p;
    asm volatile("mul.wide.u32 %0, %1, %2;" : "=l"(p) : "r"(x), "r"(M0));
    x = (uint32_t)(p >> 32);
  } else if (A == IMADLO) asm volatile("mad.lo.u32 %0, %0, %1, %2;" : "+r"(x) : "r"(M0), "r"(y));
  else if (A == IMADHI) asm volatile("mul.hi.u32 %0, %0, %1;" : "+r"(x) : "r"(M0));
  else if (A == SHF) asm volatile("shf.r.clamp.b32 %0, %0, %1, 1;" : "+r"(x) : "r"(y));
  else if (A == IADD) asm volatile("add.u32 %0, %0, %1;" : "+r"(x) : "r"(y));
  else if (A == POPC) asm volatile("popc.b32 %0, %0;" : "+r"(x));
  else if (A == SHFL) x = __shfl_sync(0xFFFFFFFFu, x, (threadIdx.x + 1) & 31);
}

template <int A, int NA, int B, int NB>
__global__ void kern(uint32_t* out, int iters, uint32_t seed) {
  uint32_t a[4], b[4], c[4], d[4];
  for (int i = 0; i < 4; ++i) {
    a[i] = seed + threadIdx.x + i;
    b[i] = seed * 3 + i;
    c[i] = a[i] * 7;
    d[i] = b[i] + 5;
  }
  for (int it = 0; it < iters; ++it) {
#pragma unroll
    for (int r = 0; r < 8; ++r) {
#pragma unroll
      for (int i = 0; i < 4; ++i) {
#pragma unroll
        for (int k = 0; k < NA; ++k) op<A>(a[i], b[i], seed);
#pragma unroll
        for (int k = 0; k < NB; ++k) op<B>(c[i], d[i], seed);
      }
    }
  }
  uint32_t s = 0;
  for (int i = 0; i < 4; ++i) s ^= a[i] ^ b[i] ^ c[i] ^ d[i];
  if (s == 0x12345678u) out[0] = s;
}

static double g_ghz = 1.965;
static int g_sms = 148;

template <int A, int NA, int B, int NB>
void run(const char* name, uint32_t* d) {
  for (int w : {2, 4}) {
    const int iters = 20000, blocks = g_sms, tpb = 128 * w;
    kern<A, NA, B, NB><<<blocks, tpb>>>(d, 100, 1);
    cudaDeviceSynchronize();
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0);
    cudaEventCreate(&e1);
    cudaEventRecord(e0);
    kern<A, NA, B, NB><<<blocks, tpb>>>(d, iters, 1);
    cudaEventRecord(e1);
    cudaDeviceSynchronize();
    float ms;
    cudaEventElapsedTime(&ms, e0, e1);
    const double steps = (double)iters * 8 * 4 * w;  // steps issued per SMSP
    printf("%-28s warps/SMSP=%d  %.2f clk per step (%d + %d instr)\n", name, w, ms * 1e-3 * g_ghz * 1e9 / steps, NA, NB);
  }
}

int main() {
  cudaDeviceProp p;
  if (cudaGetDeviceProperties(&p, 0) != cudaSuccess) {
    printf("no CUDA device\n");
    return 1;
  }
  g_sms = p.multiProcessorCount;
  int khz = 0;
  cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, 0);
  g_ghz = khz * 1e-6;
  printf("# %s, %d SMs, clock %.3f GHz (cudaDevAttrClockRate; cycles assume the kernel runs at this clock)\n", p.name,
         g_sms, g_ghz);
  uint32_t* d;
  cudaMalloc(&d, 4);
  run<LOP3, 1, LOP3, 0>("LOP3", d);
  run<SHF, 1, LOP3, 0>("SHF", d);
  run<IADD, 1, LOP3, 0>("IADD3", d);
  run<IMADLO, 1, LOP3, 0>("IMAD.lo", d);
  run<IMADHI, 1, LOP3, 0>("IMAD.HI", d);
  run<WIDE, 1, LOP3, 0>("IMAD.WIDE", d);
  run<POPC, 1, LOP3, 0>("POPC", d);
  run<SHFL, 1, LOP3, 0>("SHFL", d);
  run<WIDE, 1, LOP3, 1>("IMAD.WIDE + 1 LOP3", d);
  run<WIDE, 1, LOP3, 2>("IMAD.WIDE + 2 LOP3", d);
  run<WIDE, 1, LOP3, 3>("IMAD.WIDE + 3 LOP3", d);
  run<WIDE, 1, SHF, 2>("IMAD.WIDE + 2 SHF", d);
  run<IMADLO, 1, LOP3, 1>("IMAD.lo + 1 LOP3", d);
  run<IMADLO, 1, LOP3, 2>("IMAD.lo + 2 LOP3", d);
  run<WIDE, 1, IMADLO, 1>("IMAD.WIDE + IMAD.lo", d);
  run<WIDE, 2, LOP3, 2>("Philox round (2 W + 2 L)", d);
  run<WIDE, 2, LOP3, 3>("Philox round + 1 LOP3", d);
  run<WIDE, 2, LOP3, 4>("Philox round + 2 LOP3", d);
  return 0;
}
