/*
 * oracle/kpz2d_oracle.c — CPU ORACLE of the 2+1D generalisation (test infrastructure, NOT the product).
 *
 * PAPER.md:289-291 (Sect. 4): "We used two-sub-lattice updates, which can be generalized to checker-board lattice
 * decomposition in two dimensions" and "we have made the first step towards two dimensional simulations [7, 28]" -
 * [7] is the mapping of 2+1D KPZ growth onto a driven lattice gas of dimers (the octahedron model).  The paper says no
 * more; the reading taken here is DESIGN.md §R19, restated at every step below.  Plain, slow, byte per slope, one uniform
 * per attempted site assembled from all 32 planes by kpzref_uniform (kpz_oracle.c): no batching, no bit tricks.
 *
 * parity unpinned by the paper: the model itself is this document's reading of a one-sentence outlook; what pins the
 * implementation of that reading is listed in DESIGN.md §2 (tests/test_oracle_kpz2d_pins.py).
 *
 * Model.  Periodic Lx x Ly lattice of heights h(x,y); slopes as occupation numbers, one per bond:
 *   sx[y][x] = 1 iff h(x,y) - h(x-1,y) = +1 (else -1),   sy[y][x] = 1 iff h(x,y) - h(x,y-1) = +1 (else -1).
 * Site (x,y) sits between the x-pair (sx[y][x], sx[y][x+1]) and the y-pair (sy[y][x], sy[y+1][x]) - the 1+1D pair
 * (n_a, n_b) of PAPER.md:95 in each direction.  A forward move needs BOTH pairs in state (1,0) and turns both into (0,1)
 * with probability p (h(x,y) -= 2: the octahedron move, the dimer hop of [7]); a backward move needs both in (0,1) and
 * turns both into (1,0) with probability q.  One MCS = two passes; a pass updates one colour of the checkerboard,
 * sites with (x + y + o) even, o drawn per (sample, mcs, pass) exactly as the 1+1D offset or o = pass
 * (offset_mode 1); sites of one colour share no bond, so the order inside a pass does not matter.  The uniform of the
 * j-th active site of row y (x = 2 j + ((y + o) & 1)) is element e = y * (Lx / 2) + j of stream PAIR at time key m.
 * Flat start: h(x,y) = (x + y) & 1, i.e. sx = sy = (x + y) & 1 (W^2 = 1/4 as in PAPER.md:139).
 * Heights (DESIGN §R5 carried over): h(x,0) = sum_{i<=x} (2 sx[0][i] - 1), h(x,y) = h(x,0) + sum_{1<=j<=y} (2 sy[j][x] - 1);
 * exact int64 sums over all Lx*Ly sites; W^2 per sample, mean over samples.
 */
#include "kpz2d_oracle.h"

#include <stdlib.h>
#include <string.h>

struct kpz2dref_sim {
  int32_t Lx, Ly, S, first_sample, offset_mode;
  uint64_t seed, T_p, T_q;
  uint8_t* sx; /* [S][Ly][Lx] */
  uint8_t* sy;
  int64_t t;
  int64_t *hops_fwd, *hops_bwd; /* [S] */
  int64_t* rec_t;
  int32_t nt, nrec;
  int64_t *rec_sum_h, *rec_sum_h2; /* [nt][S] */
};

static int valid_prob(double x) { return x >= 0.0 && x <= 1.0; }

int kpz2dref_create(kpz2dref_sim** out, int32_t Lx, int32_t Ly, int32_t nsamples, double p, double q, uint64_t seed,
                    const kpzref_options* opt) {
  if (!out) return KPZREF_EINVAL;
  *out = NULL;
  /* both extents even (the checkerboard must close periodically), at least 2 */
  if (Lx < 2 || Ly < 2 || (Lx & 1) || (Ly & 1) || nsamples < 1 || !valid_prob(p) || !valid_prob(q)) return KPZREF_EINVAL;
  if ((int64_t)Lx * Ly > ((int64_t)1 << 30)) return KPZREF_EUNSUPPORTED;
  kpzref_options o = {0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1)) return KPZREF_EINVAL;
  kpz2dref_sim* sim = (kpz2dref_sim*)calloc(1, sizeof(*sim));
  if (!sim) return KPZREF_ENOMEM;
  sim->Lx = Lx;
  sim->Ly = Ly;
  sim->S = nsamples;
  sim->first_sample = o.first_sample;
  sim->offset_mode = o.offset_mode;
  sim->seed = seed;
  kpzref_threshold(p, &sim->T_p);
  kpzref_threshold(q, &sim->T_q);
  const size_t cells = (size_t)nsamples * Lx * Ly;
  sim->sx = (uint8_t*)malloc(cells);
  sim->sy = (uint8_t*)malloc(cells);
  sim->hops_fwd = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  sim->hops_bwd = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  if (!sim->sx || !sim->sy || !sim->hops_fwd || !sim->hops_bwd) {
    kpz2dref_destroy(sim);
    return KPZREF_ENOMEM;
  }
  /* flat start: h(x,y) = (x + y) & 1 */
  for (int32_t s = 0; s < nsamples; ++s)
    for (int32_t y = 0; y < Ly; ++y)
      for (int32_t x = 0; x < Lx; ++x) {
        const size_t i = ((size_t)s * Ly + y) * Lx + x;
        sim->sx[i] = (uint8_t)((x + y) & 1);
        sim->sy[i] = (uint8_t)((x + y) & 1);
      }
  *out = sim;
  return KPZREF_OK;
}

int kpz2dref_destroy(kpz2dref_sim* sim) {
  if (!sim) return KPZREF_OK;
  free(sim->sx);
  free(sim->sy);
  free(sim->hops_fwd);
  free(sim->hops_bwd);
  free(sim->rec_t);
  free(sim->rec_sum_h);
  free(sim->rec_sum_h2);
  free(sim);
  return KPZREF_OK;
}

int kpz2dref_time(const kpz2dref_sim* sim, int64_t* t) {
  if (!sim || !t) return KPZREF_EINVAL;
  *t = sim->t;
  return KPZREF_OK;
}

int kpz2dref_set_record_times(kpz2dref_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return KPZREF_EINVAL;
  for (int32_t k = 0; k < nt; ++k)
    if (t[k] < 1 || (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1])) return KPZREF_EINVAL;
  free(sim->rec_t);
  free(sim->rec_sum_h);
  free(sim->rec_sum_h2);
  sim->rec_t = NULL;
  sim->rec_sum_h = sim->rec_sum_h2 = NULL;
  sim->nt = nt;
  sim->nrec = 0;
  if (nt == 0) return KPZREF_OK;
  sim->rec_t = (int64_t*)malloc((size_t)nt * sizeof(int64_t));
  sim->rec_sum_h = (int64_t*)calloc((size_t)nt * sim->S, sizeof(int64_t));
  sim->rec_sum_h2 = (int64_t*)calloc((size_t)nt * sim->S, sizeof(int64_t));
  if (!sim->rec_t || !sim->rec_sum_h || !sim->rec_sum_h2) return KPZREF_ENOMEM;
  memcpy(sim->rec_t, t, (size_t)nt * sizeof(int64_t));
  return KPZREF_OK;
}

/* h of one sample into h[Ly][Lx] (the definition in the header comment, written out). */
static void heights_of(const kpz2dref_sim* sim, int32_t s, int32_t* h) {
  const int32_t Lx = sim->Lx, Ly = sim->Ly;
  const uint8_t* sx = sim->sx + (size_t)s * Lx * Ly;
  const uint8_t* sy = sim->sy + (size_t)s * Lx * Ly;
  int32_t run = 0;
  for (int32_t x = 0; x < Lx; ++x) {
    run += 2 * (int32_t)sx[x] - 1; /* row 0 */
    h[x] = run;
  }
  for (int32_t y = 1; y < Ly; ++y)
    for (int32_t x = 0; x < Lx; ++x) h[(size_t)y * Lx + x] = h[(size_t)(y - 1) * Lx + x] + 2 * (int32_t)sy[(size_t)y * Lx + x] - 1;
}

static int record_now(kpz2dref_sim* sim) {
  const size_t n = (size_t)sim->Lx * sim->Ly;
  int32_t* h = (int32_t*)malloc(n * sizeof(int32_t));
  if (!h) return KPZREF_ENOMEM;
  for (int32_t s = 0; s < sim->S; ++s) {
    heights_of(sim, s, h);
    int64_t s1 = 0, s2 = 0;
    for (size_t i = 0; i < n; ++i) {
      s1 += h[i];
      s2 += (int64_t)h[i] * h[i];
    }
    sim->rec_sum_h[(size_t)sim->nrec * sim->S + s] = s1;
    sim->rec_sum_h2[(size_t)sim->nrec * sim->S + s] = s2;
  }
  free(h);
  sim->nrec++;
  return KPZREF_OK;
}

int kpz2dref_run(kpz2dref_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return KPZREF_EINVAL;
  const int32_t Lx = sim->Lx, Ly = sim->Ly, half = Lx / 2;
  for (int64_t step = 0; step < n_mcs; ++step) {
    const uint64_t m = (uint64_t)sim->t; /* 0-based index of the MCS being executed */
    for (int32_t s = 0; s < sim->S; ++s) {
      const uint32_t gs = (uint32_t)(sim->first_sample + s);
      uint8_t* sx = sim->sx + (size_t)s * Lx * Ly;
      uint8_t* sy = sim->sy + (size_t)s * Lx * Ly;
      for (uint32_t pass = 0; pass < 2; ++pass) {
        uint32_t o = pass;
        if (sim->offset_mode == 0) kpzref_offset(sim->seed, gs, m, pass, &o);
        for (int32_t y = 0; y < Ly; ++y) {
          const int32_t yb = (y + 1) % Ly;
          for (int32_t j = 0; j < half; ++j) {
            const int32_t x = 2 * j + (int32_t)(((uint32_t)y + o) & 1u); /* (x + y + o) even */
            const int32_t xb = (x + 1) % Lx;
            uint32_t u;
            kpzref_uniform(sim->seed, KPZREF_TAG_PAIR, gs, m, pass, (uint64_t)y * (uint64_t)half + (uint64_t)j, &u);
            uint8_t* xa_ = &sx[(size_t)y * Lx + x];
            uint8_t* xb_ = &sx[(size_t)y * Lx + xb];
            uint8_t* ya_ = &sy[(size_t)y * Lx + x];
            uint8_t* yb_ = &sy[(size_t)yb * Lx + x];
            if (*xa_ == 1 && *xb_ == 0 && *ya_ == 1 && *yb_ == 0) {
              if ((uint64_t)u < sim->T_p) {
                *xa_ = 0; *xb_ = 1; *ya_ = 0; *yb_ = 1;
                sim->hops_fwd[s]++;
              }
            } else if (*xa_ == 0 && *xb_ == 1 && *ya_ == 0 && *yb_ == 1) {
              if ((uint64_t)u < sim->T_q) {
                *xa_ = 1; *xb_ = 0; *ya_ = 1; *yb_ = 0;
                sim->hops_bwd[s]++;
              }
            }
          }
        }
      }
    }
    sim->t++;
    if (sim->nrec < sim->nt && sim->rec_t[sim->nrec] == sim->t) {
      int rc = record_now(sim);
      if (rc) return rc;
    }
  }
  return KPZREF_OK;
}

static size_t row_words(int32_t Lx) { return ((size_t)Lx + 31) / 32; }

int kpz2dref_slopes(kpz2dref_sim* sim, uint32_t* wx, uint32_t* wy) {
  if (!sim) return KPZREF_EINVAL;
  const size_t rw = row_words(sim->Lx), rows = (size_t)sim->S * sim->Ly;
  for (int k = 0; k < 2; ++k) {
    uint32_t* w = k ? wy : wx;
    const uint8_t* b = k ? sim->sy : sim->sx;
    if (!w) continue;
    memset(w, 0, rows * rw * sizeof(uint32_t));
    for (size_t r = 0; r < rows; ++r)
      for (int32_t x = 0; x < sim->Lx; ++x)
        if (b[r * sim->Lx + x]) w[r * rw + (x >> 5)] |= 1u << (x & 31);
  }
  return KPZREF_OK;
}

int kpz2dref_set_slopes(kpz2dref_sim* sim, const uint32_t* wx, const uint32_t* wy) {
  if (!sim) return KPZREF_EINVAL;
  const size_t rw = row_words(sim->Lx), rows = (size_t)sim->S * sim->Ly;
  for (int k = 0; k < 2; ++k) {
    const uint32_t* w = k ? wy : wx;
    uint8_t* b = k ? sim->sy : sim->sx;
    if (!w) continue;
    for (size_t r = 0; r < rows; ++r)
      for (int32_t x = 0; x < sim->Lx; ++x) b[r * sim->Lx + x] = (uint8_t)((w[r * rw + (x >> 5)] >> (x & 31)) & 1u);
  }
  return KPZREF_OK;
}

int kpz2dref_heights(kpz2dref_sim* sim, int32_t sample, int32_t* h) {
  if (!sim || !h || sample < 0 || sample >= sim->S) return KPZREF_EINVAL;
  heights_of(sim, sample, h);
  return KPZREF_OK;
}

int kpz2dref_roughness(kpz2dref_sim* sim, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean) {
  if (!sim || !nt) return KPZREF_EINVAL;
  if (*nt < sim->nrec) return KPZREF_ENOMEM;
  const double N = (double)sim->Lx * (double)sim->Ly;
  for (int32_t k = 0; k < sim->nrec; ++k) {
    if (t) t[k] = sim->rec_t[k];
    double acc = 0.0;
    for (int32_t s = 0; s < sim->S; ++s) {
      const int64_t s1 = sim->rec_sum_h[(size_t)k * sim->S + s], s2 = sim->rec_sum_h2[(size_t)k * sim->S + s];
      if (sum_h) sum_h[(size_t)k * sim->S + s] = s1;
      if (sum_h2) sum_h2[(size_t)k * sim->S + s] = s2;
      /* Eq. 3 squared per sample: (N * sum h^2 - (sum h)^2) / N^2, numerator exact in 128 bits */
      const __int128 num = (__int128)((int64_t)sim->Lx * sim->Ly) * s2 - (__int128)s1 * s1;
      acc += (double)num / (N * N);
    }
    if (w2_mean) w2_mean[k] = acc / (double)sim->S;
  }
  *nt = sim->nrec;
  return KPZREF_OK;
}

int kpz2dref_hops(kpz2dref_sim* sim, int64_t* fwd, int64_t* bwd) {
  if (!sim) return KPZREF_EINVAL;
  for (int32_t s = 0; s < sim->S; ++s) {
    if (fwd) fwd[s] = sim->hops_fwd[s];
    if (bwd) bwd[s] = sim->hops_bwd[s];
  }
  return KPZREF_OK;
}
