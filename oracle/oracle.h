/*
 * oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * A plain, slow, per-spin CPU implementation of the checkerboard Metropolis hot path of
 * arXiv:2503.14688 (Bisson et al.), written from the paper and from the readings listed in
 * DESIGN.md ("Readings of the paper").  It shares no code, header, table or constant
 * generator with the CUDA library in paper_2503_14688_b200/csrc; the two only agree on the
 * documented contract (RNG keying, integer thresholds, update order).
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may load this library.  The product path never calls it.
 *
 * Paper passages followed (PAPER.md line numbers):
 *   Hamiltonian, Eq. (1)
 *   Metropolis + checkerboard + multispin
 *   fully disordered start
 *   time unit = one full-lattice sweep
 *   C(r;t), Eq. (2); E(t), Eq. (3)
 *   xi = I2/I1, Eq. (C1)
 *   32-bit random numbers
 *
 * Parity pins: every function below is pinned by tests/test_oracle_*.py (Philox known
 * answers, closed-form thresholds, exact 4x4 / 2x2 Boltzmann sums, detailed balance built
 * from the threshold table, first-half-sweep acceptance closed form, beta=0 / beta=inf
 * limits, brute-force identities for S(r), closed form for xi).  Nothing is "parity
 * unpinned".
 */
#ifndef ORACLE_H
#define ORACLE_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct oracle_lattice oracle_lattice_t;

enum { ORACLE_ISING = 0, ORACLE_BLUME_CAPEL = 1 };
enum { ORACLE_OK = 0, ORACLE_EINVAL = -1, ORACLE_ENOMEM = -2, ORACLE_ESTATE = -4 };

/* Philox4x32-10 block function (Salmon et al. 2011), from its definition. */
void oracle_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* The acceptance random number of one site: a pure function of (seed, scheme, t, c, P).
 * P = i*(L/2) + (j>>1) is the same-colour linear index. */
uint32_t oracle_u32(uint64_t seed, int scheme, uint32_t t, int colour, uint64_t P);
/* Scheme 2: the 64-bit acceptance number of one site (top 32 bits = scheme 1's u32). */
uint64_t oracle_u64(uint64_t seed, uint32_t t, int colour, uint64_t P);
/* Blume-Capel proposal bit of one site (all schemes). */
int oracle_proposal_bit(uint64_t seed, uint32_t t, int colour, uint64_t P);
/* Initial spin (-1/0/+1) of global site (i,j) for a lattice of side L. */
int oracle_initial_spin(uint64_t seed, int model, uint32_t L, uint64_t i, uint64_t j);

/* Integer acceptance thresholds, entries in [0, 2^32].
 * Ising: out[0] = thr(dE=4), out[1] = thr(dE=8).
 * Blume-Capel: out[(code*2+b)*9 + (h+4)], 54 entries. */
void oracle_thresholds(int model, double delta, double beta, uint64_t *out);
/* Scheme 2: thresholds on the 2^64 scale, same indexing; always[e] = 1 where the move is always
 * accepted (dE <= 0 or the product rounds to 2^64). */
void oracle_thresholds64(int model, double delta, double beta, uint64_t *thr, unsigned char *always);

/* Whole periodic L x L lattice (any even L >= 2), disordered start, t = 0. */
int oracle_create(oracle_lattice_t **out, uint32_t L, int model, double delta, uint64_t seed);
/* A (h x w) window at global origin (i0, j0) of a periodic Lg x Lg lattice, holding the given
 * spins, with time counter t0.  Sites outside the window are frozen at `outside`.  Keying uses
 * global coordinates, so the interior of the window evolves exactly like the full lattice
 * as long as the dependency cone (1 site per half-sweep) has not reached it. */
int oracle_window_create(oracle_lattice_t **out, uint32_t Lg, int model, double delta,
                         uint64_t seed, int scheme, uint64_t t0, uint64_t i0, uint64_t j0,
                         uint32_t h, uint32_t w, const int8_t *spins, int outside);
int oracle_set_rng_scheme(oracle_lattice_t *, int scheme);      /* 0 = quad, 1 = plane+tail, 2 = plane+tail56 */
int oracle_sweep(oracle_lattice_t *, uint64_t n, const double *beta);
/* One colour of sweep t at inverse temperature beta; does not advance t.  A sweep is
 * half_sweep(0) then half_sweep(1) then t += 1. */
int oracle_half_sweep(oracle_lattice_t *, int colour, double beta);
int oracle_measure(oracle_lattice_t *, uint32_t r_max, int64_t *M, int64_t *Q, int64_t *Sx,
                   int64_t *Sy);
int oracle_measure_rows(oracle_lattice_t *, uint64_t i0, uint64_t n_rows, uint32_t r_max,
                        int64_t *M, int64_t *Q, int64_t *Sx, int64_t *Sy);
int oracle_get_spins(oracle_lattice_t *, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                     int8_t *out);
int oracle_set_spins(oracle_lattice_t *, uint64_t i0, uint64_t j0, uint32_t h, uint32_t w,
                     const int8_t *in);
int oracle_run_series(oracle_lattice_t *, uint64_t n, double beta, int64_t *M, int64_t *B,
                      int64_t *Q, int64_t *state /* may be NULL */);
int64_t oracle_pair_sum(const int8_t *a, const int8_t *b, uint64_t n, uint64_t shift);
uint64_t oracle_time(const oracle_lattice_t *);
double oracle_xi(const int64_t *Sx, const int64_t *Sy, uint32_t r_max, int64_t Q, uint32_t L,
                 uint32_t *r_cut_out);
double oracle_energy(const int64_t *Sx, const int64_t *Sy, int64_t Q, double delta, uint32_t L);
int oracle_destroy(oracle_lattice_t *);

void oracle_set_threads(int n);     /* row-parallel half-sweeps / measurements (OpenMP) */
int oracle_get_threads(void);

#ifdef __cplusplus
}
#endif
#endif
