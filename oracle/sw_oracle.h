/*
 * sw_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, sequential CPU implementation of one Swendsen-Wang (SW) multi-cluster step
 * (arXiv 1403.7560, section 2) for the Ising (Eq. 1), q-state Potts (Eq. 2) and
 * classical XY (Eq. 3) models on periodic 2D square / 3D simple-cubic lattices.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * call this.  It shares no code with the CUDA path (paper_1403_7560_b200/csrc) and neither
 * includes the other.  Readings of the paper (where it is silent or garbled) are listed in
 * DESIGN.md section 3 ("Readings"); each function in sw_oracle.c cites the passage it follows.
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu", statistical ones at 3 sigma): Philox
 * known-answer vectors, exact enumeration of 4x4 / 3x3 Ising and 3x3 q=3 Potts, Kaufman's
 * finite-torus energy, structural invariants checked with scipy's connected components, bias /
 * independence of the transposed bond randoms (reading 6), Ising(beta) and Potts(q=2, 2 beta) giving
 * the same bonds and clusters from the same configuration and the same moments (the bit identity of
 * whole trajectories, does not hold: the two models key their cluster draws
 * differently), XY vs an independent Metropolis sampler, the clock model vs enumeration.
 * Nothing in this file is "parity unpinned" except init_spins (the seeded start, reading 15): it is
 * compared with the CUDA path's start state only, which is harmless -- any start state is a valid
 * input of the chain.  For continuous XY the pin is statistical (no closed form exists).
 */
#ifndef SW_ORACLE_H
#define SW_ORACLE_H
#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swo_ctx swo_ctx;

enum { SWO_ISING = 0, SWO_POTTS = 1, SWO_XY = 2, SWO_CLOCK = 3 };

/* Philox4x32-10, exposed so that the tests can pin it to the known-answer vectors. */
void swo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* dim in {2,3}; L >= 3 (any L, not only multiples of 32); model as enum; q = number of Potts states
 * (2..255) or clock states (2..512), ignored otherwise; beta = J/T with J = 1; returns NULL on invalid arguments or out of memory.
 * The start configuration is the seeded random start (S3), step counter t = 0. */
swo_ctx *swo_create(int dim, int L, int model, int q, double beta, uint64_t seed);
void swo_destroy(swo_ctx *o);

/* n SW steps.  Returns 0. */
int swo_step(swo_ctx *o, int n);

/* Instantaneous extensive observables of the current configuration. */
void swo_observables(const swo_ctx *o, double *E, double *M, double *M2, double *M4);

/* Exact integers (Ising: E = -sum s_i s_j, M_or_nk[0] = sum s_i;
 * Potts: E = number of unequal nearest-neighbour pairs, M_or_nk[k] = n[k], k < q). */
int swo_counts(const swo_ctx *o, int64_t *E_int, int64_t *M_or_nk, int n);

/* State access.  Spins are int8 (Ising, +-1), uint8 (Potts, 0..q-1), float (XY angle) or uint16
 * (clock state 0..q-1). */
size_t swo_num_sites(const swo_ctx *o);
uint64_t swo_step_index(const swo_ctx *o);
int swo_get_spins(const swo_ctx *o, void *dst, size_t bytes);
int swo_set_spins(swo_ctx *o, const void *src, size_t bytes, uint64_t step);
int swo_get_bonds(const swo_ctx *o, uint8_t *dst, size_t bytes);    /* bonds of the LAST step  */
int swo_get_labels(const swo_ctx *o, uint32_t *dst, size_t bytes);  /* labels of the LAST step */
/* XY: direction (r_x, r_y as fp32) and reflection constant c of the LAST step. */
int swo_get_xy_dir(const swo_ctx *o, float *rx, float *ry, float *c);
/* Clock model: exact integer histograms of the current configuration: D[d] = number of nearest-
 * neighbour pairs (i, i + e_k) with (p_i - p_j) mod q = d, n[p] = number of sites in state p. */
int swo_clock_hist(const swo_ctx *o, int64_t *D, int64_t *n, int q);
/* Clock model: mirror index m (the paper's ispr) of the LAST step. */
int swo_get_clock_mirror(const swo_ctx *o, int *m);
/* XY test hook (special case R2 in DESIGN.md): force phi for every following step. */
int swo_force_xy_phi(swo_ctx *o, int enable, double phi);

/* Run n steps and record, after every step, E and M (as swo_observables returns them; for
 * Ising M is the signed magnetisation), M2, the number of active bonds, the number of clusters
 * and sum_c n_c^2 of that step's bond configuration.  Any output pointer may be NULL. */
int swo_run_series(swo_ctx *o, int n, double *E, double *M, double *M2, double *n_active,
                   double *n_clusters, double *sum_nc2);

#ifdef __cplusplus
}
#endif
#endif
