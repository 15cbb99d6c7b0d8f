/*
 * oracle/kpz2d_oracle.h — C interface of the CPU ORACLE of the 2+1D generalisation.
 * Test infrastructure, NOT the product: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl
 * reference legs may load it.  Same conventions as oracle/kpz_oracle.h (host pointers, 0 or a negative code).
 */
#ifndef KPZ2D_ORACLE_H
#define KPZ2D_ORACLE_H
#include "kpz_oracle.h"
#ifdef __cplusplus
extern "C" {
#endif

typedef struct kpz2dref_sim kpz2dref_sim;

/* Lx x Ly periodic lattice (both even, >= 2), flat start h = (x + y) & 1, rates p (forward: both pairs (1,0) -> (0,1)) and
 * q (backward), Philox key = seed; opt as in kpzref_create (first_sample, offset_mode). */
int kpz2dref_create(kpz2dref_sim** out, int32_t Lx, int32_t Ly, int32_t nsamples, double p, double q, uint64_t seed,
                    const kpzref_options* opt);
int kpz2dref_set_record_times(kpz2dref_sim*, const int64_t* t, int32_t nt);
int kpz2dref_run(kpz2dref_sim*, int64_t n_mcs); /* checkerboard sweep, two colour passes per MCS */
int kpz2dref_time(const kpz2dref_sim*, int64_t* t);
/* slope bits [S][Ly][ceil(Lx/32)] words, bit (x & 31) of word x >> 5 of row y = sx[y][x] / sy[y][x]; either may be NULL */
int kpz2dref_slopes(kpz2dref_sim*, uint32_t* sx, uint32_t* sy);
int kpz2dref_set_slopes(kpz2dref_sim*, const uint32_t* sx, const uint32_t* sy);
int kpz2dref_heights(kpz2dref_sim*, int32_t sample, int32_t* h /* [Ly][Lx] */);
int kpz2dref_roughness(kpz2dref_sim*, int32_t* nt, int64_t* t, int64_t* sum_h, int64_t* sum_h2, double* w2_mean);
int kpz2dref_hops(kpz2dref_sim*, int64_t* fwd, int64_t* bwd /* [S] accepted forward / backward moves so far */);
int kpz2dref_destroy(kpz2dref_sim*);

#ifdef __cplusplus
}
#endif
#endif
