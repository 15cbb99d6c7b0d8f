/*
 * oracle/kpz_oracle.c — CPU ORACLE.  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, single-threaded, byte-per-site implementation of what the hot path of
 * arxiv/paper_1012_0385 computes, written from the paper and from the numbered readings
 * in DESIGN.md (§R1..§R17, which complete the schedule where the paper is silent).  No bit tricks,
 * no blocking, no lazy evaluation, no code shared with the CUDA path.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"):
 *   Philox4x32-10 ............ published known-answer vectors (tests/golden/philox4x32_10_kat.txt)
 *   offsets + heights + sums .. config-1 closed form (p=1,q=0 flat start: PAPER.md:124,139)
 *   acceptance rule, rate site, schedule, disorder rate .. brute-force master equation L<=12
 *   RSU mode .................. ASEP ring closed form J=(p-q)N(L-N)/(L(L-1)), E[W^2]=(L+1)/12
 *   heights/W^2 ............... flat W^2=1/4, h_{L-1}=2N-L, definition on random lattices
 *   KPZ growth ................ effective beta in [0.26,0.36]
 *   two-lane .................. brute-force two-lane master equation, conservation, A-lane == KPZ ring at omega=0
 * PARITY UNPINNED (convention only, fixed by DESIGN.md, no external source): the bit-plane layout of
 * the uniforms (§R4), the counter packing / stream tags (§R4), the drawn-offset reading (§R1) beyond
 * its master-equation statistics, two-lane step order (§R12), profile semantics (§R16), and for the site-wise
 * crossing model (§R18) the "once per run" reading of the flag redraw and the TURN_V stream tag.
 */
#include "kpz_oracle.h"

#include <math.h>
#include <stdlib.h>
#include <string.h>

/* ======================================================================================= */
/* Philox4x32-10 (Salmon et al., SC'11): multipliers, Weyl key increments.     */
/* ======================================================================================= */

void kpzref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    uint64_t prod0 = (uint64_t)0xD2511F53u * (uint64_t)c0;
    uint64_t prod1 = (uint64_t)0xCD9E8D57u * (uint64_t)c2;
    uint32_t n0 = (uint32_t)(prod1 >> 32) ^ c1 ^ k0;
    uint32_t n1 = (uint32_t)prod1;
    uint32_t n2 = (uint32_t)(prod0 >> 32) ^ c3 ^ k1;
    uint32_t n3 = (uint32_t)prod0;
    c0 = n0;
    c1 = n1;
    c2 = n2;
    c3 = n3;
  }
  out[0] = c0;
  out[1] = c1;
  out[2] = c2;
  out[3] = c3;
}

/* counter fields.
 *   c0 = supergroup G = element >> 7
 *   c1 = global sample index
 *   c2 = low 32 bits of the time key
 *   c3 = tag<<28 | pass<<27 | plane<<22 | (time key >> 32)        (time key < 2^54)
 * key = (low, high) 32 bits of the seed. */
int kpzref_philox_call(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint32_t pass,
                       uint32_t plane, uint32_t G, uint32_t out[4]) {
  if (tag > 15 || pass > 1 || plane > 31 || (timekey >> 54) != 0 || !out) return KPZREF_EINVAL;
  uint32_t ctr[4], key[2];
  ctr[0] = G;
  ctr[1] = sample;
  ctr[2] = (uint32_t)(timekey & 0xFFFFFFFFu);
  ctr[3] = (tag << 28) | (pass << 27) | (plane << 22) | (uint32_t)(timekey >> 32);
  key[0] = (uint32_t)(seed & 0xFFFFFFFFu);
  key[1] = (uint32_t)(seed >> 32);
  kpzref_philox4x32_10(ctr, key, out);
  return KPZREF_OK;
}

/* DESIGN §R4 (Appendix A-3): the 32-bit uniform of element e.  G = e>>7, word w = (e>>5)&3,
 * bit k = e&31; plane b supplies bit 31-b (plane 0 = most significant bit). */
int kpzref_uniform(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint32_t pass,
                   uint64_t element, uint32_t* u) {
  if (!u || (element >> 39) != 0) return KPZREF_EINVAL;
  uint32_t G = (uint32_t)(element >> 7);
  uint32_t w = (uint32_t)((element >> 5) & 3);
  uint32_t k = (uint32_t)(element & 31);
  uint32_t value = 0;
  for (uint32_t plane = 0; plane < 32; ++plane) {
    uint32_t words[4];
    int rc = kpzref_philox_call(seed, tag, sample, timekey, pass, plane, G, words);
    if (rc) return rc;
    uint32_t bit = (words[w] >> k) & 1u;
    value |= bit << (31 - plane);
  }
  *u = value;
  return KPZREF_OK;
}

/* The same uniforms for the first `count` (<= 128) elements of supergroup G at once: the definition
 * above evaluated for e = 128 G .. 128 G + count - 1 with the 32 Philox calls made once (tests check
 * the sweep against kpzref_uniform element by element). */
static void uniform_block128(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint32_t pass,
                             uint32_t G, int count, uint32_t u[128]) {
  memset(u, 0, 128 * sizeof(uint32_t));
  for (uint32_t plane = 0; plane < 32; ++plane) {
    uint32_t words[4];
    kpzref_philox_call(seed, tag, sample, timekey, pass, plane, G, words);
    for (int e = 0; e < count; ++e) {
      uint32_t bit = (words[e >> 5] >> (e & 31)) & 1u;
      u[e] |= bit << (31 - plane);
    }
  }
}

/* T(x) = floor(x * 2^32); x*2^32 is exact in double (power-of-two scaling). */
int kpzref_threshold(double x, uint64_t* T) {
  if (!T || !(x >= 0.0) || !(x <= 1.0)) return KPZREF_EINVAL;
  *T = (uint64_t)floor(x * 4294967296.0);
  return KPZREF_OK;
}

/* DESIGN §R1 (Appendix A-4): o = w0 & 1 of Philox(G=0, sample, time key m, tag OFFSET, pass, plane 0). */
int kpzref_offset(uint64_t seed, uint32_t sample, uint64_t mcs, uint32_t pass, uint32_t* o) {
  uint32_t words[4];
  int rc = kpzref_philox_call(seed, KPZREF_TAG_OFFSET, sample, mcs, pass, 0, 0, words);
  if (rc) return rc;
  *o = words[0] & 1u;
  return KPZREF_OK;
}

static int accept(uint32_t u, uint64_t T) { return (uint64_t)u < T; }

/* Number of elements of the 128-element block starting at `first` that exist when there are `total`. */
static int block_count(int64_t total, int64_t first) { return (total - first) < 128 ? (int)(total - first) : 128; }

/* Fill mask[i] = U(tag, time key, pass 0, i) < T for i in [0, L). */
static void bernoulli_sites(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint64_t T,
                            int64_t L, uint8_t* mask) {
  uint32_t u[128];
  for (int64_t base = 0; base < L; base += 128) {
    int count = block_count(L, base);
    uniform_block128(seed, tag, sample, timekey, 0, (uint32_t)(base >> 7), count, u);
    for (int e = 0; e < count; ++e) mask[base + e] = (uint8_t)accept(u[e], T);
  }
}

static int64_t words_per_sample(int64_t L) { return (L + 31) / 32; }

static void pack_bits(const uint8_t* sites, int64_t L, uint32_t* words) {
  int64_t nw = words_per_sample(L);
  for (int64_t w = 0; w < nw; ++w) words[w] = 0;
  for (int64_t i = 0; i < L; ++i)
    if (sites[i]) words[i >> 5] |= (uint32_t)1 << (i & 31);
}

static void unpack_bits(const uint32_t* words, int64_t L, uint8_t* sites) {
  for (int64_t i = 0; i < L; ++i) sites[i] = (uint8_t)((words[i >> 5] >> (i & 31)) & 1u);
}

/* ======================================================================================= */
/* KPZ / ASEP ring                                                                          */
/* ======================================================================================= */

struct kpzref_sim {
  int64_t L;
  int32_t S;
  int32_t first_sample;
  int32_t offset_mode;
  uint64_t seed;
  uint64_t T_p, T_p_slow, T_q, T_q_slow;
  uint8_t* n;      /* [S][L] occupation (s_i in {0,1}) */
  uint8_t* slow_p; /* [S][L] tag bits of Eq. 8 */
  uint8_t* slow_q; /* [S][L] */
  int64_t t;       /* Monte-Carlo steps done */
  int32_t nt;      /* record times */
  int64_t* rec_t;
  int32_t nrec;    /* records captured so far */
  int64_t* rec_sum_h;  /* [nt][S] */
  int64_t* rec_sum_h2; /* [nt][S] */
  int64_t* hops_fwd;   /* [S] */
  int64_t* hops_bwd;   /* [S] */
};

static int valid_prob(double x) { return x >= 0.0 && x <= 1.0; }

int kpzref_create(kpzref_sim** out, int64_t L, int32_t nsamples, double p, double q,
                  const kpzref_disorder* disorder, uint64_t seed, const kpzref_options* opt) {
  if (!out) return KPZREF_EINVAL;
  *out = NULL;
  /* any even L >= 4 (pairs must tile the ring). */
  if (L < 4 || (L & 1) || nsamples < 1 || !valid_prob(p) || !valid_prob(q)) return KPZREF_EINVAL;
  if (L >= ((int64_t)1 << 38)) return KPZREF_EUNSUPPORTED;
  kpzref_disorder d = {0.0, p, 0.0, q};
  if (disorder) d = *disorder;
  if (!valid_prob(d.prob_slow_p) || !valid_prob(d.p_slow) || !valid_prob(d.prob_slow_q) || !valid_prob(d.q_slow))
    return KPZREF_EINVAL;
  kpzref_options o = {0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1)) return KPZREF_EINVAL;

  kpzref_sim* sim = (kpzref_sim*)calloc(1, sizeof(kpzref_sim));
  if (!sim) return KPZREF_ENOMEM;
  sim->L = L;
  sim->S = nsamples;
  sim->first_sample = o.first_sample;
  sim->offset_mode = o.offset_mode;
  sim->seed = seed;
  kpzref_threshold(p, &sim->T_p);
  kpzref_threshold(q, &sim->T_q);
  kpzref_threshold(d.p_slow, &sim->T_p_slow);
  kpzref_threshold(d.q_slow, &sim->T_q_slow);
  size_t cells = (size_t)nsamples * (size_t)L;
  sim->n = (uint8_t*)malloc(cells);
  sim->slow_p = (uint8_t*)calloc(cells, 1);
  sim->slow_q = (uint8_t*)calloc(cells, 1);
  sim->hops_fwd = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  sim->hops_bwd = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  if (!sim->n || !sim->slow_p || !sim->slow_q || !sim->hops_fwd || !sim->hops_bwd) {
    kpzref_destroy(sim);
    return KPZREF_ENOMEM;
  }
  uint64_t T_prob_p, T_prob_q;
  kpzref_threshold(d.prob_slow_p, &T_prob_p);
  kpzref_threshold(d.prob_slow_q, &T_prob_q);
  for (int32_t s = 0; s < nsamples; ++s) {
    uint8_t* n = sim->n + (size_t)s * L;
    /* PAPER.md:95 "periodic, alternating 0/1 distribution, which corresponds to a flat initial surface". */
    for (int64_t i = 0; i < L; ++i) n[i] = (uint8_t)(i & 1);
    /* PAPER.md:151-155 Eq. 8; two independent Bernoulli masks per sample, fixed for the run. */
    uint32_t gs = (uint32_t)(o.first_sample + s);
    if (disorder) {
      bernoulli_sites(seed, KPZREF_TAG_SLOW_P, gs, 0, T_prob_p, L, sim->slow_p + (size_t)s * L);
      bernoulli_sites(seed, KPZREF_TAG_SLOW_Q, gs, 0, T_prob_q, L, sim->slow_q + (size_t)s * L);
    }
  }
  *out = sim;
  return KPZREF_OK;
}

int kpzref_destroy(kpzref_sim* sim) {
  if (!sim) return KPZREF_OK;
  free(sim->n);
  free(sim->slow_p);
  free(sim->slow_q);
  free(sim->rec_t);
  free(sim->rec_sum_h);
  free(sim->rec_sum_h2);
  free(sim->hops_fwd);
  free(sim->hops_bwd);
  free(sim);
  return KPZREF_OK;
}

int kpzref_set_record_times(kpzref_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return KPZREF_EINVAL;
  for (int32_t k = 0; k < nt; ++k) {
    if (t[k] < 1) return KPZREF_EINVAL;
    if (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1]) return KPZREF_EINVAL;
  }
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

/* heights from slopes, Eq. 3 sums.  DESIGN §R5: slope 2 n_i - 1, inclusive prefix,
 * x = 0..L-1, exact integer sums. */
static void heights_and_sums(const uint8_t* n, int64_t L, int32_t* h_out, int64_t* sum_h, int64_t* sum_h2) {
  int64_t h = 0, s1 = 0, s2 = 0;
  for (int64_t x = 0; x < L; ++x) {
    h += 2 * (int64_t)n[x] - 1;
    if (h_out) h_out[x] = (int32_t)h;
    s1 += h;
    s2 += h * h;
  }
  if (sum_h) *sum_h = s1;
  if (sum_h2) *sum_h2 = s2;
}

static void kpz_record_if_due(kpzref_sim* sim) {
  if (sim->nrec < sim->nt && sim->rec_t[sim->nrec] == sim->t) {
    for (int32_t s = 0; s < sim->S; ++s) {
      int64_t s1, s2;
      heights_and_sums(sim->n + (size_t)s * sim->L, sim->L, NULL, &s1, &s2);
      sim->rec_sum_h[(size_t)sim->nrec * sim->S + s] = s1;
      sim->rec_sum_h2[(size_t)sim->nrec * sim->S + s] = s2;
    }
    sim->nrec++;
  }
}

/* One sub-lattice pass of one sample (DESIGN §R1,R2,R3; Appendix A-5).
 * Pair j: a = 2j+o, b = (a+1) mod L — for o=1 the last pair (L-1,0) closes the ring. */
static void kpz_pass(kpzref_sim* sim, int32_t s, uint64_t m, uint32_t pass) {
  const int64_t L = sim->L;
  const int64_t npairs = L / 2;
  uint8_t* n = sim->n + (size_t)s * L;
  const uint8_t* slow_p = sim->slow_p + (size_t)s * L;
  const uint8_t* slow_q = sim->slow_q + (size_t)s * L;
  uint32_t gs = (uint32_t)(sim->first_sample + s);
  uint32_t o = pass;
  if (sim->offset_mode == 0) kpzref_offset(sim->seed, gs, m, pass, &o);
  uint32_t u[128];
  for (int64_t j = 0; j < npairs; ++j) {
    if ((j & 127) == 0)
      uniform_block128(sim->seed, KPZREF_TAG_PAIR, gs, m, pass, (uint32_t)(j >> 7), block_count(npairs, j), u);
    int64_t a = 2 * j + o;
    int64_t b = (a + 1) % L;
    uint32_t uj = u[j & 127];
    if (n[a] == 1 && n[b] == 0) {
      /* forward jump of the '1' at a with probability p_a (rate of the departure site, §R2) */
      uint64_t T = slow_p[a] ? sim->T_p_slow : sim->T_p;
      if (accept(uj, T)) {
        n[a] = 0;
        n[b] = 1;
        sim->hops_fwd[s]++;
      }
    } else if (n[a] == 0 && n[b] == 1) {
      /* backward jump of the '1' at b with probability q_b */
      uint64_t T = slow_q[b] ? sim->T_q_slow : sim->T_q;
      if (accept(uj, T)) {
        n[a] = 1;
        n[b] = 0;
        sim->hops_bwd[s]++;
      }
    }
  }
}

int kpzref_run(kpzref_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return KPZREF_EINVAL;
  if (((uint64_t)(sim->t + n_mcs) >> 54) != 0) return KPZREF_EUNSUPPORTED;
  for (int64_t step = 0; step < n_mcs; ++step) {
    uint64_t m = (uint64_t)sim->t; /* §R10: 0-based index of the MCS being executed */
    for (int32_t s = 0; s < sim->S; ++s)
      for (uint32_t pass = 0; pass < 2; ++pass) kpz_pass(sim, s, m, pass);
    sim->t += 1; /* PAPER.md:95 "When all sites are updated once the time (t) is incremented" */
    kpz_record_if_due(sim);
  }
  return KPZREF_OK;
}

/* Oracle-only random-sequential mode ("known results for RSU"; Appendix A-7):
 * per MCS, L bond attempts; attempt number `step` draws r0, r1 = words 0,1 of
 * Philox(G=step, sample, time key m, tag RSU, pass 0, plane 0); bond a = (r0*L)>>32, b = a+1 mod L;
 * same acceptance with u = r1. */
int kpzref_run_rsu(kpzref_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return KPZREF_EINVAL;
  if (sim->L >= ((int64_t)1 << 32)) return KPZREF_EUNSUPPORTED;
  const int64_t L = sim->L;
  for (int64_t it = 0; it < n_mcs; ++it) {
    uint64_t m = (uint64_t)sim->t;
    for (int32_t s = 0; s < sim->S; ++s) {
      uint8_t* n = sim->n + (size_t)s * L;
      const uint8_t* slow_p = sim->slow_p + (size_t)s * L;
      const uint8_t* slow_q = sim->slow_q + (size_t)s * L;
      uint32_t gs = (uint32_t)(sim->first_sample + s);
      for (int64_t step = 0; step < L; ++step) {
        uint32_t w[4];
        kpzref_philox_call(sim->seed, KPZREF_TAG_RSU, gs, m, 0, 0, (uint32_t)step, w);
        int64_t a = (int64_t)(((uint64_t)w[0] * (uint64_t)L) >> 32);
        int64_t b = (a + 1) % L;
        if (n[a] == 1 && n[b] == 0) {
          if (accept(w[1], slow_p[a] ? sim->T_p_slow : sim->T_p)) {
            n[a] = 0;
            n[b] = 1;
            sim->hops_fwd[s]++;
          }
        } else if (n[a] == 0 && n[b] == 1) {
          if (accept(w[1], slow_q[b] ? sim->T_q_slow : sim->T_q)) {
            n[a] = 1;
            n[b] = 0;
            sim->hops_bwd[s]++;
          }
        }
      }
    }
    sim->t += 1;
    kpz_record_if_due(sim);
  }
  return KPZREF_OK;
}

/* Checkpoint restore: continue from MCS count t; with the lattice (kpzref_set_lattice) this is the whole
 * state, because every random number is a function of (seed, sample, m, ...).  Drops the record list. */
int kpzref_set_time(kpzref_sim* sim, int64_t t) {
  if (!sim || t < 0 || ((uint64_t)t >> 54) != 0) return KPZREF_EINVAL;
  int rc = kpzref_set_record_times(sim, NULL, 0);
  if (rc) return rc;
  sim->t = t;
  return KPZREF_OK;
}

int kpzref_time(const kpzref_sim* sim, int64_t* t) {
  if (!sim || !t) return KPZREF_EINVAL;
  *t = sim->t;
  return KPZREF_OK;
}

int kpzref_lattice(kpzref_sim* sim, uint32_t* words) {
  if (!sim || !words) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) pack_bits(sim->n + (size_t)s * sim->L, sim->L, words + (size_t)s * nw);
  return KPZREF_OK;
}

int kpzref_set_lattice(kpzref_sim* sim, const uint32_t* words) {
  if (!sim || !words) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) unpack_bits(words + (size_t)s * nw, sim->L, sim->n + (size_t)s * sim->L);
  return KPZREF_OK;
}

int kpzref_disorder_masks(kpzref_sim* sim, uint32_t* slow_p, uint32_t* slow_q) {
  if (!sim) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) {
    if (slow_p) pack_bits(sim->slow_p + (size_t)s * sim->L, sim->L, slow_p + (size_t)s * nw);
    if (slow_q) pack_bits(sim->slow_q + (size_t)s * sim->L, sim->L, slow_q + (size_t)s * nw);
  }
  return KPZREF_OK;
}

int kpzref_set_disorder_masks(kpzref_sim* sim, const uint32_t* slow_p, const uint32_t* slow_q) {
  if (!sim) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) {
    if (slow_p) unpack_bits(slow_p + (size_t)s * nw, sim->L, sim->slow_p + (size_t)s * sim->L);
    if (slow_q) unpack_bits(slow_q + (size_t)s * nw, sim->L, sim->slow_q + (size_t)s * sim->L);
  }
  return KPZREF_OK;
}

int kpzref_heights(kpzref_sim* sim, int32_t sample, int32_t* h) {
  if (!sim || !h || sample < 0 || sample >= sim->S) return KPZREF_EINVAL;
  if (sim->L > 0x7FFFFFFF) return KPZREF_EUNSUPPORTED;
  heights_and_sums(sim->n + (size_t)sample * sim->L, sim->L, h, NULL, NULL);
  return KPZREF_OK;
}

/* PAPER.md:107 Eq. 3 squared, per sample; "the W^2(L,t) data of each sample are averaged"
 * (DESIGN §R6).  W^2 = (L*sum_h2 - sum_h^2) / L^2 with the numerator exact in 128-bit integers. */
int kpzref_roughness(kpzref_sim* sim, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean) {
  if (!sim || !nt) return KPZREF_EINVAL;
  if (*nt < sim->nrec) return KPZREF_ENOMEM;
  for (int32_t k = 0; k < sim->nrec; ++k) {
    if (t) t[k] = sim->rec_t[k];
    double acc = 0.0;
    for (int32_t s = 0; s < sim->S; ++s) {
      int64_t s1 = sim->rec_sum_h[(size_t)k * sim->S + s];
      int64_t s2 = sim->rec_sum_h2[(size_t)k * sim->S + s];
      if (sum_h) sum_h[(size_t)k * sim->S + s] = s1;
      if (sum_h2) sum_h2[(size_t)k * sim->S + s] = s2;
      __int128 num = (__int128)sim->L * (__int128)s2 - (__int128)s1 * (__int128)s1;
      acc += (double)num / ((double)sim->L * (double)sim->L);
    }
    if (w2_mean) w2_mean[k] = acc / (double)sim->S;
  }
  *nt = sim->nrec;
  return KPZREF_OK;
}

int kpzref_hops(kpzref_sim* sim, int64_t* fwd, int64_t* bwd) {
  if (!sim) return KPZREF_EINVAL;
  for (int32_t s = 0; s < sim->S; ++s) {
    if (fwd) fwd[s] = sim->hops_fwd[s];
    if (bwd) bwd[s] = sim->hops_bwd[s];
  }
  return KPZREF_OK;
}

/* ======================================================================================= */
/* Two-lane opposite-direction model (Appendix A-6)      */
/* ======================================================================================= */

struct lanesref_sim {
  int64_t L;
  int32_t S;
  int32_t first_sample;
  int32_t offset_mode;
  uint64_t seed;
  uint64_t T_pa, T_pb, T_turn, T_omega;
  uint64_t T_w0;        /* crossing threshold at sites whose flag is 0 (0 for the turning-point model, §R13) */
  int32_t independent;  /* 1: separate flags v_i for B->A, 0: one flag set for both directions */
  int64_t period;
  uint8_t* A;    /* [S][L] lane A occupation (particles hop right) */
  uint8_t* B;    /* [S][L] lane B occupation (particles hop left) */
  uint8_t* turn; /* [S][L] flags u_i of the current epoch (turning points; A->B, and B->A unless independent) */
  uint8_t* turn_v; /* [S][L] flags v_i for B->A when independent (else NULL) */
  int64_t t;
  int64_t* J_A;  /* [S] hops in lane A so far */
  int64_t* J_B;  /* [S] hops in lane B so far */
  uint32_t* occ_A; /* [S][L] epoch-end occupancy counts */
  uint32_t* occ_B;
  int64_t nsnap;
  int32_t nt;
  int64_t* rec_t;
  int32_t nrec;
  int64_t *rec_JA, *rec_JB, *rec_NA, *rec_NB; /* [nt][S] */
};

int lanesref_destroy(lanesref_sim* sim) {
  if (!sim) return KPZREF_OK;
  free(sim->A);
  free(sim->B);
  free(sim->turn);
  free(sim->turn_v);
  free(sim->J_A);
  free(sim->J_B);
  free(sim->occ_A);
  free(sim->occ_B);
  free(sim->rec_t);
  free(sim->rec_JA);
  free(sim->rec_JB);
  free(sim->rec_NA);
  free(sim->rec_NB);
  free(sim);
  return KPZREF_OK;
}

/* DESIGN §R13 (turning-point model of configs[4]): crossing probability omega at flagged sites, 0 elsewhere, one
 * flag set for both directions. */
int lanesref_create(lanesref_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                    double turn_prob, int64_t turn_period, double omega, uint64_t seed, const kpzref_options* opt) {
  return lanesref_create_crossing(out, L, nsamples, p_a, p_b, rho0, turn_prob, omega, 0.0, 0, turn_period, seed, opt);
}

/* DESIGN §R18 (the paper's own two-lane model): every site can be crossed; the crossing probability
 * is w_flagged where the site's flag is set and w_unflagged elsewhere ("the crossing probability is reduced from 0.8
 * to 0.2" at flagged sites, flags set with probability 1/2); with independent = 1 the directions A->B and B->A have
 * separate flag sets u_i (stream TURN) and v_i (stream TURN_V). */
int lanesref_create_crossing(lanesref_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                             double turn_prob, double omega, double w_unflagged, int32_t independent,
                             int64_t turn_period, uint64_t seed, const kpzref_options* opt) {
  if (!out) return KPZREF_EINVAL;
  *out = NULL;
  if (L < 4 || (L & 1) || nsamples < 1 || turn_period < 0) return KPZREF_EINVAL;
  if (!valid_prob(p_a) || !valid_prob(p_b) || !valid_prob(rho0) || !valid_prob(turn_prob) || !valid_prob(omega) ||
      !valid_prob(w_unflagged) || (independent != 0 && independent != 1))
    return KPZREF_EINVAL;
  if (L >= ((int64_t)1 << 31)) return KPZREF_EUNSUPPORTED;
  kpzref_options o = {0, 0, 0};
  if (opt) o = *opt;
  if (o.first_sample < 0 || (o.offset_mode != 0 && o.offset_mode != 1)) return KPZREF_EINVAL;
  lanesref_sim* sim = (lanesref_sim*)calloc(1, sizeof(lanesref_sim));
  if (!sim) return KPZREF_ENOMEM;
  sim->L = L;
  sim->S = nsamples;
  sim->first_sample = o.first_sample;
  sim->offset_mode = o.offset_mode;
  sim->seed = seed;
  sim->period = turn_period;
  kpzref_threshold(p_a, &sim->T_pa);
  kpzref_threshold(p_b, &sim->T_pb);
  kpzref_threshold(turn_prob, &sim->T_turn);
  kpzref_threshold(omega, &sim->T_omega);
  kpzref_threshold(w_unflagged, &sim->T_w0);
  sim->independent = independent;
  size_t cells = (size_t)nsamples * (size_t)L;
  sim->A = (uint8_t*)malloc(cells);
  sim->B = (uint8_t*)malloc(cells);
  sim->turn = (uint8_t*)malloc(cells);
  if (independent) sim->turn_v = (uint8_t*)malloc(cells);
  sim->J_A = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  sim->J_B = (int64_t*)calloc((size_t)nsamples, sizeof(int64_t));
  sim->occ_A = (uint32_t*)calloc(cells, sizeof(uint32_t));
  sim->occ_B = (uint32_t*)calloc(cells, sizeof(uint32_t));
  if (!sim->A || !sim->B || !sim->turn || (independent && !sim->turn_v) || !sim->J_A || !sim->J_B || !sim->occ_A || !sim->occ_B) {
    lanesref_destroy(sim);
    return KPZREF_ENOMEM;
  }
  uint64_t T_rho;
  kpzref_threshold(rho0, &T_rho);
  for (int32_t s = 0; s < nsamples; ++s) {
    uint32_t gs = (uint32_t)(o.first_sample + s);
    /* independent Bernoulli(rho0) per site per lane. */
    bernoulli_sites(seed, KPZREF_TAG_INIT_A, gs, 0, T_rho, L, sim->A + (size_t)s * L);
    bernoulli_sites(seed, KPZREF_TAG_INIT_B, gs, 0, T_rho, L, sim->B + (size_t)s * L);
    /* turning-point mask of epoch 0. */
    bernoulli_sites(seed, KPZREF_TAG_TURN, gs, 0, sim->T_turn, L, sim->turn + (size_t)s * L);
    if (independent) bernoulli_sites(seed, KPZREF_TAG_TURN_V, gs, 0, sim->T_turn, L, sim->turn_v + (size_t)s * L);
  }
  *out = sim;
  return KPZREF_OK;
}

int lanesref_set_record_times(lanesref_sim* sim, const int64_t* t, int32_t nt) {
  if (!sim || nt < 0 || (nt > 0 && !t)) return KPZREF_EINVAL;
  for (int32_t k = 0; k < nt; ++k) {
    if (t[k] < 1) return KPZREF_EINVAL;
    if (k == 0 ? t[k] <= sim->t : t[k] <= t[k - 1]) return KPZREF_EINVAL;
  }
  free(sim->rec_t);
  free(sim->rec_JA);
  free(sim->rec_JB);
  free(sim->rec_NA);
  free(sim->rec_NB);
  sim->rec_t = sim->rec_JA = sim->rec_JB = sim->rec_NA = sim->rec_NB = NULL;
  sim->nt = nt;
  sim->nrec = 0;
  if (nt == 0) return KPZREF_OK;
  size_t cells = (size_t)nt * sim->S;
  sim->rec_t = (int64_t*)malloc((size_t)nt * sizeof(int64_t));
  sim->rec_JA = (int64_t*)calloc(cells, sizeof(int64_t));
  sim->rec_JB = (int64_t*)calloc(cells, sizeof(int64_t));
  sim->rec_NA = (int64_t*)calloc(cells, sizeof(int64_t));
  sim->rec_NB = (int64_t*)calloc(cells, sizeof(int64_t));
  if (!sim->rec_t || !sim->rec_JA || !sim->rec_JB || !sim->rec_NA || !sim->rec_NB) return KPZREF_ENOMEM;
  memcpy(sim->rec_t, t, (size_t)nt * sizeof(int64_t));
  return KPZREF_OK;
}

/* In-lane sub-lattice pass of both lanes with the same offset (§R12). */
static void lanes_inlane_pass(lanesref_sim* sim, int32_t s, uint64_t m, uint32_t pass) {
  const int64_t L = sim->L;
  const int64_t npairs = L / 2;
  uint8_t* A = sim->A + (size_t)s * L;
  uint8_t* B = sim->B + (size_t)s * L;
  uint32_t gs = (uint32_t)(sim->first_sample + s);
  uint32_t o = pass;
  if (sim->offset_mode == 0) kpzref_offset(sim->seed, gs, m, pass, &o);
  uint32_t ua[128], ub[128];
  for (int64_t j = 0; j < npairs; ++j) {
    if ((j & 127) == 0) {
      uniform_block128(sim->seed, KPZREF_TAG_PAIR, gs, m, pass, (uint32_t)(j >> 7), block_count(npairs, j), ua);
      uniform_block128(sim->seed, KPZREF_TAG_PAIR_B, gs, m, pass, (uint32_t)(j >> 7), block_count(npairs, j), ub);
    }
    int64_t a = 2 * j + o;
    int64_t b = (a + 1) % L;
    /* lane A: particles move to the right, a -> b */
    if (A[a] == 1 && A[b] == 0 && accept(ua[j & 127], sim->T_pa)) {
      A[a] = 0;
      A[b] = 1;
      sim->J_A[s]++; /* PAPER.md:275 "J±1 by each hopping event" — counted positive per lane (§R15) */
    }
    /* lane B: particles move to the left, b -> a */
    if (B[a] == 0 && B[b] == 1 && accept(ub[j & 127], sim->T_pb)) {
      B[a] = 1;
      B[b] = 0;
      sim->J_B[s]++;
    }
  }
}

/* Lane changes at turning points (§R13): from -> to at sites with turn = 1. */
static void lanes_switch(lanesref_sim* sim, int32_t s, uint64_t m, uint32_t tag, uint8_t* from, uint8_t* to,
                         const uint8_t* flags) {
  const int64_t L = sim->L;
  const uint8_t* turn = flags + (size_t)s * L;
  uint32_t gs = (uint32_t)(sim->first_sample + s);
  uint32_t u[128];
  for (int64_t i = 0; i < L; ++i) {
    if ((i & 127) == 0) uniform_block128(sim->seed, tag, gs, m, 0, (uint32_t)(i >> 7), block_count(L, i), u);
    /* §R13 / §R18: threshold omega at flagged sites, w_unflagged (0 in the turning-point model) elsewhere */
    if (from[i] == 1 && to[i] == 0 && accept(u[i & 127], turn[i] ? sim->T_omega : sim->T_w0)) {
      from[i] = 0;
      to[i] = 1;
    }
  }
}

int lanesref_run(lanesref_sim* sim, int64_t n_mcs) {
  if (!sim || n_mcs < 0) return KPZREF_EINVAL;
  if (((uint64_t)(sim->t + n_mcs) >> 54) != 0) return KPZREF_EUNSUPPORTED;
  const int64_t L = sim->L;
  for (int64_t it = 0; it < n_mcs; ++it) {
    uint64_t m = (uint64_t)sim->t;
    for (int32_t s = 0; s < sim->S; ++s) {
      uint8_t* A = sim->A + (size_t)s * L;
      uint8_t* B = sim->B + (size_t)s * L;
      uint32_t gs = (uint32_t)(sim->first_sample + s);
      /* §R13: positions redrawn at the start of every epoch of `period` MCS (epoch 0 drawn at create). */
      if (sim->period > 0 && m > 0 && m % (uint64_t)sim->period == 0)
      {
        bernoulli_sites(sim->seed, KPZREF_TAG_TURN, gs, m / (uint64_t)sim->period, sim->T_turn, L,
                        sim->turn + (size_t)s * L);
        if (sim->independent)
          bernoulli_sites(sim->seed, KPZREF_TAG_TURN_V, gs, m / (uint64_t)sim->period, sim->T_turn, L,
                          sim->turn_v + (size_t)s * L);
      }
      const uint8_t* fv = sim->independent ? sim->turn_v : sim->turn;
      lanes_inlane_pass(sim, s, m, 0);                                  /* PAPER.md:261 step 1 */
      lanes_switch(sim, s, m, KPZREF_TAG_SWITCH_AB, A, B, sim->turn);   /* PAPER.md:262 step 2, flags u_i */
      lanes_inlane_pass(sim, s, m, 1);                                  /* PAPER.md:263-264 steps 3,4 (closure = pair (L-1,0)) */
      lanes_switch(sim, s, m, KPZREF_TAG_SWITCH_BA, B, A, fv);          /* PAPER.md:265 step 5, flags v_i */
    }
    sim->t += 1;
    /* §R16: occupancy profile accumulated at the end of each turning-point epoch. */
    if (sim->period > 0 && sim->t % sim->period == 0) {
      for (size_t c = 0; c < (size_t)sim->S * (size_t)L; ++c) {
        sim->occ_A[c] += sim->A[c];
        sim->occ_B[c] += sim->B[c];
      }
      sim->nsnap++;
    }
    if (sim->nrec < sim->nt && sim->rec_t[sim->nrec] == sim->t) {
      for (int32_t s = 0; s < sim->S; ++s) {
        int64_t na = 0, nb = 0;
        for (int64_t i = 0; i < L; ++i) {
          na += sim->A[(size_t)s * L + i];
          nb += sim->B[(size_t)s * L + i];
        }
        size_t c = (size_t)sim->nrec * sim->S + s;
        sim->rec_JA[c] = sim->J_A[s];
        sim->rec_JB[c] = sim->J_B[s];
        sim->rec_NA[c] = na;
        sim->rec_NB[c] = nb;
      }
      sim->nrec++;
    }
  }
  return KPZREF_OK;
}

/* As kpzref_set_time; the caller restores lanes and turning-point mask with lanesref_set_state.  Hop counters,
 * profile counts and the snapshot count keep their values. */
int lanesref_set_time(lanesref_sim* sim, int64_t t) {
  if (!sim || t < 0 || ((uint64_t)t >> 54) != 0) return KPZREF_EINVAL;
  int rc = lanesref_set_record_times(sim, NULL, 0);
  if (rc) return rc;
  sim->t = t;
  return KPZREF_OK;
}

int lanesref_time(const lanesref_sim* sim, int64_t* t) {
  if (!sim || !t) return KPZREF_EINVAL;
  *t = sim->t;
  return KPZREF_OK;
}

int lanesref_state(lanesref_sim* sim, uint32_t* a, uint32_t* b, uint32_t* turn) {
  if (!sim) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) {
    if (a) pack_bits(sim->A + (size_t)s * sim->L, sim->L, a + (size_t)s * nw);
    if (b) pack_bits(sim->B + (size_t)s * sim->L, sim->L, b + (size_t)s * nw);
    if (turn) pack_bits(sim->turn + (size_t)s * sim->L, sim->L, turn + (size_t)s * nw);
  }
  return KPZREF_OK;
}

int lanesref_set_state(lanesref_sim* sim, const uint32_t* a, const uint32_t* b, const uint32_t* turn) {
  if (!sim) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) {
    if (a) unpack_bits(a + (size_t)s * nw, sim->L, sim->A + (size_t)s * sim->L);
    if (b) unpack_bits(b + (size_t)s * nw, sim->L, sim->B + (size_t)s * sim->L);
    if (turn) unpack_bits(turn + (size_t)s * nw, sim->L, sim->turn + (size_t)s * sim->L);
  }
  return KPZREF_OK;
}

int lanesref_flags(lanesref_sim* sim, uint32_t* u, uint32_t* v) {
  if (!sim) return KPZREF_EINVAL;
  int64_t nw = words_per_sample(sim->L);
  const uint8_t* fv = sim->independent ? sim->turn_v : sim->turn;
  for (int32_t s = 0; s < sim->S; ++s) {
    if (u) pack_bits(sim->turn + (size_t)s * sim->L, sim->L, u + (size_t)s * nw);
    if (v) pack_bits(fv + (size_t)s * sim->L, sim->L, v + (size_t)s * nw);
  }
  return KPZREF_OK;
}

int lanesref_set_flags(lanesref_sim* sim, const uint32_t* u, const uint32_t* v) {
  if (!sim || (v && !sim->independent)) return KPZREF_EINVAL; /* one shared set: pass it as u */
  int64_t nw = words_per_sample(sim->L);
  for (int32_t s = 0; s < sim->S; ++s) {
    if (u) unpack_bits(u + (size_t)s * nw, sim->L, sim->turn + (size_t)s * sim->L);
    if (v) unpack_bits(v + (size_t)s * nw, sim->L, sim->turn_v + (size_t)s * sim->L);
  }
  return KPZREF_OK;
}

int lanesref_currents(lanesref_sim* sim, int32_t* nt, int64_t* t, int64_t* j_a, int64_t* j_b, int64_t* n_a,
                      int64_t* n_b) {
  if (!sim || !nt) return KPZREF_EINVAL;
  if (*nt < sim->nrec) return KPZREF_ENOMEM;
  size_t cells = (size_t)sim->nrec * sim->S;
  for (int32_t k = 0; k < sim->nrec; ++k)
    if (t) t[k] = sim->rec_t[k];
  if (j_a) memcpy(j_a, sim->rec_JA, cells * sizeof(int64_t));
  if (j_b) memcpy(j_b, sim->rec_JB, cells * sizeof(int64_t));
  if (n_a) memcpy(n_a, sim->rec_NA, cells * sizeof(int64_t));
  if (n_b) memcpy(n_b, sim->rec_NB, cells * sizeof(int64_t));
  *nt = sim->nrec;
  return KPZREF_OK;
}

int lanesref_totals(lanesref_sim* sim, int64_t* j_a, int64_t* j_b, int64_t* n_a, int64_t* n_b) {
  if (!sim) return KPZREF_EINVAL;
  for (int32_t s = 0; s < sim->S; ++s) {
    int64_t na = 0, nb = 0;
    for (int64_t i = 0; i < sim->L; ++i) {
      na += sim->A[(size_t)s * sim->L + i];
      nb += sim->B[(size_t)s * sim->L + i];
    }
    if (j_a) j_a[s] = sim->J_A[s];
    if (j_b) j_b[s] = sim->J_B[s];
    if (n_a) n_a[s] = na;
    if (n_b) n_b[s] = nb;
  }
  return KPZREF_OK;
}

int lanesref_profile(lanesref_sim* sim, uint32_t* occ_a, uint32_t* occ_b, int64_t* nsnap) {
  if (!sim) return KPZREF_EINVAL;
  size_t cells = (size_t)sim->S * (size_t)sim->L;
  if (occ_a) memcpy(occ_a, sim->occ_A, cells * sizeof(uint32_t));
  if (occ_b) memcpy(occ_b, sim->occ_B, cells * sizeof(uint32_t));
  if (nsnap) *nsnap = sim->nsnap;
  return KPZREF_OK;
}
