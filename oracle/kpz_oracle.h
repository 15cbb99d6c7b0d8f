/*
 * oracle/kpz_oracle.h — C interface of the CPU ORACLE (test infrastructure, NOT the product).
 *
 * This library is the plain, slow, single-threaded, byte-per-site restatement of what the
 * hot path of arxiv/paper_1012_0385 computes (sub-lattice Monte-Carlo sweep of the 1+1D
 * RSOS/KPZ model in ASEP form, heights / roughness reduction, two-lane model).  It exists so
 * that tests can prove the CUDA library (include/kpz_b200.h) bit-exact.  Only tests/,
 * __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may load it.
 * It shares no code, header, table or helper with paper_1012_0385_b200/csrc.
 *
 * All pointers are HOST pointers.  All functions return 0 on success or a negative code:
 *   -1 EINVAL (bad argument)   -2 EUNSUPPORTED   -3 ENOMEM
 *
 * Citations: PAPER.md:<line> = /root/reference/PAPER.md; "DESIGN §R<n>" = the numbered reading
 * of the paper in DESIGN.md (taken from SURVEY.md §8(c) / Appendix A).
 */
#ifndef KPZ_ORACLE_H
#define KPZ_ORACLE_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

#define KPZREF_OK 0
#define KPZREF_EINVAL (-1)
#define KPZREF_EUNSUPPORTED (-2)
#define KPZREF_ENOMEM (-3)

/* Random streams (counter field "tag"). */
enum {
  KPZREF_TAG_PAIR = 0,      /* KPZ pair uniforms and lane-A pair uniforms */
  KPZREF_TAG_OFFSET = 1,    /* sub-lattice offset o per (sample, mcs, pass) */
  KPZREF_TAG_SLOW_P = 2,    /* quenched slow-p site mask (Eq. 8) */
  KPZREF_TAG_SLOW_Q = 3,    /* quenched slow-q site mask (Eq. 8) */
  KPZREF_TAG_INIT_A = 4,    /* two-lane initial occupation, lane A */
  KPZREF_TAG_INIT_B = 5,    /* two-lane initial occupation, lane B */
  KPZREF_TAG_PAIR_B = 6,    /* lane-B pair uniforms */
  KPZREF_TAG_TURN = 7,      /* turning-point mask per epoch */
  KPZREF_TAG_SWITCH_AB = 8, /* A->B lane change uniforms */
  KPZREF_TAG_SWITCH_BA = 9, /* B->A lane change uniforms */
  KPZREF_TAG_RSU = 10,      /* oracle-only random-sequential mode */
  KPZREF_TAG_TURN_V = 11    /* flags v_i of the B->A crossings when they are independent of u_i */
};

typedef struct {
  double prob_slow_p; /* Q of Eq. 8 for p_i */
  double p_slow;      /* r*p of Eq. 8, given explicitly */
  double prob_slow_q; /* same law for q_i */
  double q_slow;
} kpzref_disorder;

typedef struct {
  int32_t first_sample; /* global index of local sample 0 (RNG key); default 0 */
  int32_t offset_mode;  /* 0 = offset drawn per pass (normative), 1 = alternating 0,1 */
  int32_t path;         /* ignored by the oracle */
} kpzref_options;

typedef struct kpzref_sim kpzref_sim;
typedef struct lanesref_sim lanesref_sim;

/* ---- random numbers (§R4) -------------------------------------------------- */
/* Philox4x32-10 block function: 4-word counter, 2-word key -> 4 words. */
void kpzref_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* One Philox call of the method's keying: returns words w0..w3 for (seed, tag, sample, timekey, pass, plane, G). */
int kpzref_philox_call(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint32_t pass,
                       uint32_t plane, uint32_t G, uint32_t out[4]);
/* 32-bit uniform of element e (pair index or site index), assembled MSB-first from 32 planes. */
int kpzref_uniform(uint64_t seed, uint32_t tag, uint32_t sample, uint64_t timekey, uint32_t pass,
                   uint64_t element, uint32_t* u);
/* Threshold T(x) = floor(x * 2^32) as uint64 (x in [0,1]); acceptance is (uint64)u < T(x). */
int kpzref_threshold(double x, uint64_t* T);
/* Offset o in {0,1} for (seed, sample, mcs, pass), offset_mode 0. */
int kpzref_offset(uint64_t seed, uint32_t sample, uint64_t mcs, uint32_t pass, uint32_t* o);

/* ---- KPZ / ASEP ring ------------------------------ */
int kpzref_create(kpzref_sim** out, int64_t L, int32_t nsamples, double p, double q,
                  const kpzref_disorder* disorder /* NULL = none */, uint64_t seed,
                  const kpzref_options* opt /* NULL = defaults */);
int kpzref_set_record_times(kpzref_sim*, const int64_t* t, int32_t nt); /* strictly increasing, t[0] > current time */
int kpzref_run(kpzref_sim*, int64_t n_mcs);      /* two-sub-lattice SCA sweep, n_mcs Monte-Carlo steps */
int kpzref_run_rsu(kpzref_sim*, int64_t n_mcs);  /* oracle-only: random-sequential updates */
int kpzref_time(const kpzref_sim*, int64_t* t);
int kpzref_set_time(kpzref_sim*, int64_t t); /* checkpoint restore: continue from MCS count t; drops the record list */
int kpzref_lattice(kpzref_sim*, uint32_t* words);            /* [S][L/32 rounded up]; bit (i&31) of word i>>5 = n_i */
int kpzref_set_lattice(kpzref_sim*, const uint32_t* words);
int kpzref_disorder_masks(kpzref_sim*, uint32_t* slow_p, uint32_t* slow_q); /* same layout; either may be NULL */
int kpzref_set_disorder_masks(kpzref_sim*, const uint32_t* slow_p, const uint32_t* slow_q); /* NULL = leave */
int kpzref_heights(kpzref_sim*, int32_t sample, int32_t* h /* L */);   /* h_x = sum_{i<=x} (2 n_i - 1) */
int kpzref_roughness(kpzref_sim*, int32_t* nt /* in: capacity, out: count */, int64_t* t,
                     int64_t* sum_h, int64_t* sum_h2 /* [nt][S] */, double* w2_mean /* [nt] */);
int kpzref_hops(kpzref_sim*, int64_t* fwd, int64_t* bwd /* [S] accepted p- and q-moves so far */);
int kpzref_destroy(kpzref_sim*);

/* ---- two-lane opposite-direction model -------------- */
int lanesref_create(lanesref_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                    double turn_prob, int64_t turn_period /* 0 = never redraw */, double omega, uint64_t seed,
                    const kpzref_options* opt);
/* the paper's own two-lane model - crossing probability omega where the site's flag is set (flags
 * Bernoulli(turn_prob)), w_unflagged elsewhere; independent = 1: separate flag sets for A->B and B->A. */
int lanesref_create_crossing(lanesref_sim** out, int64_t L, int32_t nsamples, double p_a, double p_b, double rho0,
                             double turn_prob, double omega, double w_unflagged, int32_t independent,
                             int64_t turn_period, uint64_t seed, const kpzref_options* opt);
/* Flag sets u (A->B) and v (B->A) of the current epoch, natural layout; v == u unless independent.  NULL = skip. */
int lanesref_flags(lanesref_sim*, uint32_t* u, uint32_t* v);
int lanesref_set_flags(lanesref_sim*, const uint32_t* u, const uint32_t* v);
int lanesref_set_record_times(lanesref_sim*, const int64_t* t, int32_t nt);
int lanesref_run(lanesref_sim*, int64_t n_mcs);
int lanesref_time(const lanesref_sim*, int64_t* t);
int lanesref_set_time(lanesref_sim*, int64_t t);
int lanesref_state(lanesref_sim*, uint32_t* a, uint32_t* b, uint32_t* turn); /* [S][L/32 rounded up], any may be NULL */
int lanesref_set_state(lanesref_sim*, const uint32_t* a, const uint32_t* b, const uint32_t* turn); /* NULL = leave */
int lanesref_currents(lanesref_sim*, int32_t* nt, int64_t* t, int64_t* j_a, int64_t* j_b, int64_t* n_a,
                      int64_t* n_b /* [nt][S] */);
int lanesref_totals(lanesref_sim*, int64_t* j_a, int64_t* j_b, int64_t* n_a, int64_t* n_b /* [S], now */);
int lanesref_profile(lanesref_sim*, uint32_t* occ_a, uint32_t* occ_b /* [S][L] */, int64_t* nsnap);
int lanesref_destroy(lanesref_sim*);

#ifdef __cplusplus
}
#endif
#endif
