/*
 * sw_oracle.h -- C ABI of the CPU oracle for one Swendsen-Wang sweep.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load this library.  It
 * shares no code (no header, helper, table or constant generator) with the
 * CUDA path under paper_1208_2080_b200/csrc and include/sw.h.
 *
 * What it computes, and where that is defined:
 *   - the Potts model and the three steps of a sweep:      PAPER.md:33-40 (sec. 2, eq. 1)
 *   - "proper label = smallest label of the cluster":
 *   - p = 1 - exp(-K), T = floor(p * 2^32), Philox4x32-10 keyed by
 *     (seed, sweep, purpose, site), root-keyed new state:  BASELINE.json north_star
 *   - the frozen field layout of the draws:                DESIGN.md "Readings" R11
 *
 * Parity pins (tests/test_oracle_*.py, all -m "not gpu"): Philox known-answer
 * vectors, threshold closed forms, BFS labels vs scipy connected_components and
 * vs brute force, brute-force Boltzmann averages on 3x3 / 4x4, Kaufman's exact
 * torus energy, the 3x3 random-cluster enumeration, percolation cluster density,
 * K=0 / K=inf limits.  No function here is "parity unpinned".
 */
#ifndef SW_ORACLE_H
#define SW_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swo_ctx swo_ctx;

enum { SWO_OK = 0, SWO_ERR_INVALID_ARG = 1, SWO_ERR_OOM = 2, SWO_ERR_STATE = 4 };
enum { SWO_INIT_ORDERED = 0, SWO_INIT_RANDOM = 1 };

/* -- building blocks, exported so that each can be pinned on its own -------- */

/* Philox4x32-10 (Salmon, Moraes, Dror, Shaw, SC'11): 128-bit counter, 64-bit key. */
void swo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);

/* T = floor((1 - exp(-K)) * 2^32) in IEEE double; K = +inf -> 2^32.  NaN / K < 0 -> error. */
int swo_threshold(double K, uint64_t *T);

/* The three kinds of draw (R11).  dir: 0 = right, 1 = down. */
uint32_t swo_draw_bond(uint64_t seed, uint32_t t, uint64_t site, int dir);
uint32_t swo_draw_flip(uint64_t seed, uint32_t t, uint64_t root);
uint32_t swo_draw_init(uint64_t seed, uint64_t site);
/* uint32 draw -> state in 0..q-1:  floor(w * q / 2^32). */
uint32_t swo_state_from_draw(uint32_t w, uint32_t q);

/* Canonical labels of an arbitrary bond mask on the periodic LxL lattice.
 * bonds[i]: bit0 = bond (i, right(i)) active, bit1 = bond (i, down(i)) active.
 * labels[i] = smallest site index connected to i.  Flood fill in
 * index order.  Optionally returns the number of clusters and the largest size. */
int swo_label_bonds(uint32_t L, const uint8_t *bonds, uint32_t *labels,
                    uint64_t *n_clusters, uint64_t *largest_cluster);

/* -- the simulation object --------------------------------------------------- */

int  swo_create(swo_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed);
int  swo_init(swo_ctx *c, int mode);                 /* sets spins, t = 0, forgets labels */
int  swo_set_state(swo_ctx *c, const uint8_t *spins, uint64_t t);
int  swo_sweep(swo_ctx *c, uint64_t n);
int  swo_measure(swo_ctx *c, uint64_t *energy_bonds, uint64_t *mag_counts /* [q] */,
                 uint64_t *n_clusters, uint64_t *largest_cluster);
/* n times: one sweep, then one measurement; row k of out is
 * [energy_bonds, n_clusters, largest_cluster, mag_counts[0..q-1]] after sweep k. */
int  swo_sweep_measure(swo_ctx *c, uint64_t n, uint64_t *out /* [n][3+q] */);
int  swo_get_spins(swo_ctx *c, uint8_t *dst /* [L*L] */);
int  swo_get_labels(swo_ctx *c, uint32_t *dst /* [L*L] */);   /* of the last sweep */
int  swo_get_bonds(swo_ctx *c, uint8_t *dst /* [L*L] */);     /* of the last sweep */
int  swo_get_threshold(swo_ctx *c, uint64_t *T);
int  swo_get_time(swo_ctx *c, uint64_t *t);
void swo_destroy(swo_ctx *c);

#ifdef __cplusplus
}
#endif
#endif
