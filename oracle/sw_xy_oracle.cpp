/*
 * sw_xy_oracle.cpp -- plain, slow CPU oracle for one embedded-cluster Swendsen-Wang sweep of the 2D classical XY model
 * (see sw_xy_oracle.h for the definition and the arithmetic contract).  TEST INFRASTRUCTURE, NOT PRODUCT.
 *
 * Lattice and conventions as in sw_oracle.cpp: L x L periodic, site i = y*L + x, a site owns its right
 * and its down bond.  Philox, the draw layout and the flood-fill labeling come from sw_oracle.cpp (the oracle's own
 * pinned pieces: swo_philox4x32_10, swo_draw_bond, swo_draw_flip, swo_label_bonds).
 */
#include "sw_xy_oracle.h"
#include "sw_oracle.h"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

enum { PURPOSE_INIT_XY = 0, PURPOSE_REFLECT = 3 };

static const double TWO_PI = 6.283185307179586476925286766559;

/* DESIGN.md X2: the direction of sweep t: angle 2 pi (w0 + 1/2) / 2^32 of Philox(idx 0, sweep t, purpose REFLECT) */
void swo_xy_reflection(uint64_t seed, uint32_t t, double r[2])
{
    uint32_t ctr[4] = { 0u, 0u, t, (uint32_t)PURPOSE_REFLECT };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    swo_philox4x32_10(ctr, key, w);
    const double phi = TWO_PI * (((double)w[0] + 0.5) * (1.0 / 4294967296.0));
    r[0] = std::cos(phi);
    r[1] = std::sin(phi);
}

/* a = s . r, as one product and one fused multiply-add */
double swo_xy_projection(const double s[2], const double r[2])
{
    return std::fma(s[0], r[0], s[1] * r[1]);
}

/* Wolff's embedded Ising coupling: p = 1 - exp(-2 K a_i a_j) if a_i a_j > 0, else 0; threshold as for the Potts model */
uint64_t swo_xy_bond_threshold(double K, double a_i, double a_j)
{
    const double x = ((2.0 * K) * a_i) * a_j;
    if (!(x > 0.0)) return 0;
    if (std::isinf(x)) return (uint64_t)1 << 32;
    const double scaled = std::floor(std::ldexp(-std::expm1(-x), 32));
    if (scaled <= 0.0) return 0;
    if (scaled >= 4294967296.0) return (uint64_t)1 << 32;
    return (uint64_t)scaled;
}

/* reflection about the line perpendicular to r: s <- s - 2 a r, a = s . r; two fused multiply-adds */
void swo_xy_reflect(double s[2], const double r[2])
{
    const double a = swo_xy_projection(s, r);
    const double m = -2.0 * a;
    const double x = std::fma(m, r[0], s[0]);
    const double y = std::fma(m, r[1], s[1]);
    s[0] = x; s[1] = y;
}

/* DESIGN.md X5: a point of the square (-1, 1)^2 from two words of Philox(idx site, sweep 0, purpose INIT), the second
 * pair of words if the first lies outside the unit disc (or at its centre), normalised: correctly rounded operations only */
void swo_xy_init_spin(uint64_t seed, uint64_t site, double s[2])
{
    uint32_t ctr[4] = { (uint32_t)site, (uint32_t)(site >> 32), 0u, (uint32_t)PURPOSE_INIT_XY };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    uint32_t w[4];
    swo_philox4x32_10(ctr, key, w);
    double x = ((double)w[0] + 0.5) * (1.0 / 2147483648.0) - 1.0;
    double y = ((double)w[1] + 0.5) * (1.0 / 2147483648.0) - 1.0;
    double n2 = std::fma(x, x, y * y);
    if (n2 > 1.0) {
        x = ((double)w[2] + 0.5) * (1.0 / 2147483648.0) - 1.0;
        y = ((double)w[3] + 0.5) * (1.0 / 2147483648.0) - 1.0;
        n2 = std::fma(x, x, y * y);
    }
    const double n = std::sqrt(n2);
    s[0] = x / n;
    s[1] = y / n;
}

struct swo_xy {
    uint64_t L, N, seed, t;
    double K;
    bool have_spins, have_labels;
    uint64_t n_clusters, largest;
    std::vector<double> spins;      /* [N][2] */
    std::vector<uint8_t> bonds;
    std::vector<uint32_t> labels;
};

int swo_xy_create(swo_xy **out, uint32_t L, double K, uint64_t seed)
{
    if (!out) return SWO_ERR_INVALID_ARG;
    *out = nullptr;
    if (L < 2 || L > 65536 || std::isnan(K) || K < 0.0) return SWO_ERR_INVALID_ARG;
    swo_xy *c = new (std::nothrow) swo_xy();
    if (!c) return SWO_ERR_OOM;
    c->L = L; c->N = (uint64_t)L * L; c->K = K; c->seed = seed; c->t = 0;
    c->have_spins = c->have_labels = false; c->n_clusters = c->largest = 0;
    try {
        c->spins.assign(2 * c->N, 0.0);
        c->bonds.assign(c->N, 0);
        c->labels.assign(c->N, 0);
    } catch (const std::bad_alloc &) { delete c; return SWO_ERR_OOM; }
    *out = c;
    return SWO_OK;
}

void swo_xy_destroy(swo_xy *c) { delete c; }

int swo_xy_init(swo_xy *c, int mode)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (mode == 0) {
        for (uint64_t i = 0; i < c->N; ++i) { c->spins[2 * i] = 1.0; c->spins[2 * i + 1] = 0.0; }
    } else if (mode == 1) {
        for (uint64_t i = 0; i < c->N; ++i) swo_xy_init_spin(c->seed, i, &c->spins[2 * i]);
    } else return SWO_ERR_INVALID_ARG;
    c->t = 0; c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;
    return SWO_OK;
}

int swo_xy_set_state(swo_xy *c, const double *spins, uint64_t t)
{
    if (!c || !spins || t > 0xFFFFFFFFull) return SWO_ERR_INVALID_ARG;
    for (uint64_t i = 0; i < 2 * c->N; ++i) if (!std::isfinite(spins[i])) return SWO_ERR_INVALID_ARG;
    std::memcpy(c->spins.data(), spins, 2 * c->N * sizeof(double));
    c->t = t; c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;
    return SWO_OK;
}

static int xy_one_sweep(swo_xy *c)
{
    const uint64_t L = c->L, N = c->N;
    const uint32_t t = (uint32_t)c->t;
    double r[2];
    swo_xy_reflection(c->seed, t, r);

    /* step (1): bonds between the embedded Ising spins */
    for (uint64_t i = 0; i < N; ++i) {
        const uint64_t x = i % L, y = i / L;
        const uint64_t ir = y * L + (x + 1) % L;
        const uint64_t id = ((y + 1) % L) * L + x;
        const double a = swo_xy_projection(&c->spins[2 * i], r);
        uint8_t b = 0;
        if ((uint64_t)swo_draw_bond(c->seed, t, i, 0) < swo_xy_bond_threshold(c->K, a, swo_xy_projection(&c->spins[2 * ir], r))) b |= 1;
        if ((uint64_t)swo_draw_bond(c->seed, t, i, 1) < swo_xy_bond_threshold(c->K, a, swo_xy_projection(&c->spins[2 * id], r))) b |= 2;
        c->bonds[i] = b;
    }

    /* step (2): canonical labels (the Potts oracle's flood fill) */
    int rc = swo_label_bonds((uint32_t)L, c->bonds.data(), c->labels.data(), &c->n_clusters, &c->largest);
    if (rc != SWO_OK) return rc;

    /* step (3): a cluster is reflected iff the draw of its root, mapped to {0, 1} like a q = 2 state, is 1 */
    for (uint64_t i = 0; i < N; ++i)
        if (swo_state_from_draw(swo_draw_flip(c->seed, t, c->labels[i]), 2) == 1) swo_xy_reflect(&c->spins[2 * i], r);
    c->t += 1;
    c->have_labels = true;
    return SWO_OK;
}

int swo_xy_sweep(swo_xy *c, uint64_t n)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    if (c->t + n > 0x100000000ull) return SWO_ERR_STATE;
    for (uint64_t k = 0; k < n; ++k) {
        int rc = xy_one_sweep(c);
        if (rc != SWO_OK) return rc;
    }
    return SWO_OK;
}

int swo_xy_measure(swo_xy *c, double *energy_sum, double mag[2], uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    const uint64_t L = c->L, N = c->N;
    if (energy_sum) {
        double e = 0.0;
        for (uint64_t i = 0; i < N; ++i) {
            const uint64_t x = i % L, y = i / L;
            const double *s = &c->spins[2 * i];
            const double *sr = &c->spins[2 * (y * L + (x + 1) % L)], *sd = &c->spins[2 * (((y + 1) % L) * L + x)];
            e += s[0] * sr[0] + s[1] * sr[1];
            e += s[0] * sd[0] + s[1] * sd[1];
        }
        *energy_sum = e;
    }
    if (mag) {
        mag[0] = mag[1] = 0.0;
        for (uint64_t i = 0; i < N; ++i) { mag[0] += c->spins[2 * i]; mag[1] += c->spins[2 * i + 1]; }
    }
    if (n_clusters) *n_clusters = c->have_labels ? c->n_clusters : 0;
    if (largest_cluster) *largest_cluster = c->have_labels ? c->largest : 0;
    return SWO_OK;
}

int swo_xy_get_spins(swo_xy *c, double *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    std::memcpy(dst, c->spins.data(), 2 * c->N * sizeof(double));
    return SWO_OK;
}

int swo_xy_get_labels(swo_xy *c, uint32_t *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_labels) return SWO_ERR_STATE;
    std::memcpy(dst, c->labels.data(), c->N * sizeof(uint32_t));
    return SWO_OK;
}

int swo_xy_get_bonds(swo_xy *c, uint8_t *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_labels) return SWO_ERR_STATE;
    std::memcpy(dst, c->bonds.data(), c->N);
    return SWO_OK;
}

int swo_xy_get_time(swo_xy *c, uint64_t *t)
{
    if (!c || !t) return SWO_ERR_INVALID_ARG;
    *t = c->t;
    return SWO_OK;
}
