/*
 * sw_xy_oracle.h -- C ABI of the CPU oracle for one embedded-cluster Swendsen-Wang sweep of the 2D classical XY model.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (as sw_oracle.h).  Shares no code with the CUDA path.
 *
 * What it computes, and where that is defined:
 *   - the extension the paper names: "This computation is easily extended to continuous spin models, such as the
 *     classical XY model, using the Wolff's idea of embedded cluster"
 *   - the three steps of a sweep are those of PAPER.md:40 applied to the embedded Ising variables: with a random unit
 *     vector r, every spin s_i (a unit vector) is split into its projection a_i = s_i . r and the rest; the energy
 *     -J s_i . s_j contains -J a_i a_j, an Ising coupling J |a_i a_j| between the signs of a_i and a_j
 *     (Wolff, Phys. Rev. Lett. 62 (1989) 361), hence
 *       (1) the bond <ij> is active iff a_i a_j > 0 and draw < floor(p_ij 2^32), p_ij = 1 - exp(-2 K a_i a_j)
 *       (2) clusters of active bonds, canonical label = smallest site index
 *       (3) every cluster is reflected, s -> s - 2 (s . r) r, with probability 1/2
 *   - draws: Philox4x32-10 with the layout of DESIGN.md R11 (BOND, FLIP, INIT as for the Potts model) plus purpose 3
 *     REFLECT (idx 0, sweep t, word 0): the angle of r is 2 pi (w0 + 1/2) / 2^32.  DESIGN.md readings X1-X6.
 *
 * Arithmetic (X4): IEEE double; every product, sum and fused multiply-add below is written out explicitly
 * (this file is compiled with -ffp-contract=off), so that a GPU implementation using the same correctly rounded
 * operations reproduces the spins bit for bit.  The only library functions are cos / sin of ONE angle per sweep (r, on
 * the host on both sides) and expm1 in the bond probability (a draw decides differently only if it hits the one
 * integer threshold on which two libm implementations disagree in the last place: probability ~ 1e-17 per bond).
 */
#ifndef SW_XY_ORACLE_H
#define SW_XY_ORACLE_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct swo_xy swo_xy;

/* the building blocks, exported so that each can be pinned on its own */
void     swo_xy_reflection(uint64_t seed, uint32_t t, double r[2]);           /* unit vector of sweep t */
double   swo_xy_projection(const double s[2], const double r[2]);             /* a = fma(s_x, r_x, s_y r_y) */
uint64_t swo_xy_bond_threshold(double K, double a_i, double a_j);             /* floor((1 - exp(-2 K a_i a_j)) 2^32), 0 if a_i a_j <= 0 */
void     swo_xy_reflect(double s[2], const double r[2]);                      /* s <- s - 2 (s . r) r */
void     swo_xy_init_spin(uint64_t seed, uint64_t site, double s[2]);         /* random unit vector of INIT */

int  swo_xy_create(swo_xy **out, uint32_t L, double K, uint64_t seed);
int  swo_xy_init(swo_xy *c, int mode);               /* 0 ordered: all spins (1, 0); 1 random; t = 0 */
int  swo_xy_set_state(swo_xy *c, const double *spins /* [L*L][2] */, uint64_t t);
int  swo_xy_sweep(swo_xy *c, uint64_t n);
/* energy_sum = sum over bonds of s_i . s_j (E = -J energy_sum); mag = sum of the spins; cluster statistics of the last sweep */
int  swo_xy_measure(swo_xy *c, double *energy_sum, double mag[2], uint64_t *n_clusters, uint64_t *largest_cluster);
int  swo_xy_get_spins(swo_xy *c, double *dst /* [L*L][2] */);
int  swo_xy_get_labels(swo_xy *c, uint32_t *dst);
int  swo_xy_get_bonds(swo_xy *c, uint8_t *dst);      /* bit0 right, bit1 down */
int  swo_xy_get_time(swo_xy *c, uint64_t *t);
void swo_xy_destroy(swo_xy *c);

#ifdef __cplusplus
}
#endif
#endif
