// sweep_types.cuh — plain-data kernel parameter blocks shared by the statically compiled kernels and the kernels
// specialised at run time through NVRTC (jit.cu).  No host headers: this file is also fed to NVRTC.
#pragma once
#include "philox.cuh"

namespace kpz {

// A threshold as the kernels see it: `always` (T = 2^32), else the 32-bit value (0 = never).
struct Thresh {
  uint32_t value;   // low 32 bits of T
  uint32_t always;  // 1 if T == 2^32
};

struct KpzDev {
  PhiloxKeys keys;
  Thresh thr[4];  // classes: 0 = p, 1 = p_slow, 2 = q, 3 = q_slow
  int32_t nplanes;
  int32_t offset_mode;
  int32_t first_sample;
  int32_t S;
  int32_t PW;   // 64-site groups (pair-words) per sample = L/64
  int32_t PWp;  // row stride in words, multiple of 4
  int32_t U;    // units per sample = PWp/4
  uint32_t* E;  // [S][PWp] even-site words (frame 0)
  uint32_t* O;  // [S][PWp] odd-site words
  const uint32_t* SPE;  // slow-p tags at even / odd sites, same layout (nullptr = none)
  const uint32_t* SPO;
  const uint32_t* SQE;
  const uint32_t* SQO;
};

struct KpzRunArgs {
  long long t0;      // MCS already done
  long long n_mcs;   // MCS to do
  const long long* rec_t;  // [nt] record times (device)
  int32_t rec_begin;       // first record index with time > t0
  int32_t nt;
  long long* rec_sum_h;    // [nt][S]
  long long* rec_sum_h2;   // [nt][S]
  unsigned int* check;     // debug (K1J_HALOCHECK): counter of failed halo sequence checks, else nullptr
  unsigned int* queue;     // K1J_QUEUE: [0] = next work item, [1 + s] = chunks of sample s done (zeroed before the launch)
};

// K3 (pass-by-pass streamed sweep): one launch = one sub-lattice pass from (Ein, Oin) to (Eout, Oout).
struct K3Pass {
  const uint32_t* Ein;
  const uint32_t* Oin;
  uint32_t* Eout;
  uint32_t* Oout;
  const unsigned char* fin;  // [S] frame of the input lattice
  const unsigned char* fo;   // [S] offset of this pass = frame of the output; nullptr = "bring to frame 0, no update"
  long long m;               // MCS index (time key)
  int pass;
};

// K3T (temporally blocked streamed sweep): D.E / D.O are the input ring, these the ping-pong output.
struct K3TArgs {
  uint32_t* Eout;
  uint32_t* Oout;
  long long t0;     // MCS already done
  long long n_mcs;  // MCS of this chunk (<= 64: the window's end units absorb the contaminated sites)
};

// ---- two-lane model (lanes_k4.cuh, k4_lanes_jit.cuh) ---------------------------------------------------------------
struct LanesDev {
  PhiloxKeys keys;
  Thresh t_pa, t_pb, t_turn, t_omega;
  Thresh t_w0;               // crossing threshold at unflagged sites (0 in the turning-point model)
  int32_t independent;       // 1: B->A crossings read their own flag set V
  int32_t np_a, np_b, np_w;  // planes needed by the in-lane thresholds and by omega
  int32_t offset_mode;
  int32_t first_sample;
  int32_t S;
  int32_t W;    // natural words per sample = L/32
  int32_t Wp;   // row stride, multiple of 8
  int32_t U;    // units per sample = Wp/8
  long long period;
  uint32_t* A;  // [S][Wp]
  uint32_t* B;
  uint32_t* T;  // flags of the current epoch (turning points; u_i of the A->B crossings)
  uint32_t* V;  // flags v_i of the B->A crossings (== T unless independent)
  unsigned long long* JA;  // [S] hops so far
  unsigned long long* JB;
  uint32_t* occA;  // [S][L] epoch-end occupancy counts
  uint32_t* occB;
};

struct LanesRunArgs {
  long long t0, n_mcs;
  const long long* rec_t;
  int32_t rec_begin, nt;
  long long* rec;  // [4][nt][S]: J_A, J_B, N_A, N_B
  unsigned int* check;  // debug (K4J_HALOCHECK): counter of failed halo sequence checks, else nullptr
};

}  // namespace kpz
