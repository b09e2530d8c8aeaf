/*
 * sw_oracle.cpp -- plain, slow, single-threaded CPU oracle for one Swendsen-Wang
 * multi-cluster sweep of the 2D q-state Potts model on an LxL periodic lattice.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT (see sw_oracle.h).  Shares no code with the
 * CUDA path.  Written from the paper's statement of the method; there is no
 * blocking, fusion or reordering beyond what the definitions state:
 *
 *   step (1)  "Construct a bond lattice of active or non-active bonds depending
 *             upon the temperature"
 *   step (2)  "The active bonds partition the spins into clusters which are
 *             identified and labeled"
 *             proper label = "the smallest label of any spin in the cluster"
 *                                                                  PAPER.md:42
 *   step (3)  "All spins in each cluster are set randomly to one of q"
 *                                                                  PAPER.md:40
 *   lattice   nearest-neighbour pairs, periodic boundaries
 *
 * The paper never prints the bond probability (the end of sec. 2 is
 * garbled); p = 1 - exp(-K), the integer threshold and the Philox
 * draws are fixed by BASELINE.json's north_star and DESIGN.md readings R1, R9-R11.
 *
 * Conventions: site i = y*L + x (x fastest); right(i) = y*L + (x+1)%L;
 * down(i) = ((y+1)%L)*L + x; spins are 0..q-1 in uint8; a site owns its right
 * and its down bond (bit0 / bit1 of bonds[i]).
 */
#include "sw_oracle.h"

#include <cmath>
#include <cstring>
#include <new>
#include <vector>

/* ------------------------------------------------------------------------- */
/* Philox4x32-10, as published (Salmon et al., SC'11, sec. 3.3 / Random123):   */
/* ten rounds of                                                             */
/*   (c0,c1,c2,c3) <- (hi(M1*c2)^c1^k0, lo(M1*c2), hi(M0*c0)^c3^k1, lo(M0*c0)) */
/* with the key bumped by the Weyl constants between rounds.                  */
/* ------------------------------------------------------------------------- */
void swo_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4])
{
    const uint64_t M0 = 0xD2511F53u, M1 = 0xCD9E8D57u;
    const uint32_t W0 = 0x9E3779B9u, W1 = 0xBB67AE85u;
    uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
    uint32_t k0 = key[0], k1 = key[1];
    for (int round = 0; round < 10; ++round) {
        uint64_t p0 = M0 * (uint64_t)c0;
        uint64_t p1 = M1 * (uint64_t)c2;
        uint32_t n0 = (uint32_t)(p1 >> 32) ^ c1 ^ k0;
        uint32_t n1 = (uint32_t)p1;
        uint32_t n2 = (uint32_t)(p0 >> 32) ^ c3 ^ k1;
        uint32_t n3 = (uint32_t)p0;
        c0 = n0; c1 = n1; c2 = n2; c3 = n3;
        k0 += W0; k1 += W1;
    }
    out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* DESIGN.md R11: key = (seed lo, seed hi); counter = (idx lo, idx hi, sweep t, purpose). */
enum { PURPOSE_INIT = 0, PURPOSE_BOND = 1, PURPOSE_FLIP = 2 };

static void draw4(uint64_t seed, uint64_t idx, uint32_t t, uint32_t purpose, uint32_t out[4])
{
    uint32_t ctr[4] = { (uint32_t)idx, (uint32_t)(idx >> 32), t, purpose };
    uint32_t key[2] = { (uint32_t)seed, (uint32_t)(seed >> 32) };
    swo_philox4x32_10(ctr, key, out);
}

/* BOND: one call per pair of consecutive sites; idx = site >> 1;
 * word 2*(site&1) is the right bond of the site, word 2*(site&1)+1 its down bond. */
uint32_t swo_draw_bond(uint64_t seed, uint32_t t, uint64_t site, int dir)
{
    uint32_t w[4];
    draw4(seed, site >> 1, t, PURPOSE_BOND, w);
    return w[2 * (site & 1) + (dir ? 1 : 0)];
}

/* FLIP: idx = canonical root of the cluster, word 0. */
uint32_t swo_draw_flip(uint64_t seed, uint32_t t, uint64_t root)
{
    uint32_t w[4];
    draw4(seed, root, t, PURPOSE_FLIP, w);
    return w[0];
}

/* INIT: idx = site, sweep field 0, word 0. */
uint32_t swo_draw_init(uint64_t seed, uint64_t site)
{
    uint32_t w[4];
    draw4(seed, site, 0, PURPOSE_INIT, w);
    return w[0];
}

/* DESIGN.md R9: state = floor(w*q / 2^32). */
uint32_t swo_state_from_draw(uint32_t w, uint32_t q)
{
    return (uint32_t)(((uint64_t)w * (uint64_t)q) >> 32);
}

/* north_star: "A bond is active iff a uint32 draw is below floor(p*2^32), with p
 * computed once on the host", p = 1 - exp(-K).  DESIGN.md R10: -expm1(-K), floor. */
int swo_threshold(double K, uint64_t *T)
{
    if (!T || std::isnan(K) || K < 0.0) return SWO_ERR_INVALID_ARG;
    if (std::isinf(K)) { *T = (uint64_t)1 << 32; return SWO_OK; }
    double p = -std::expm1(-K);
    double scaled = std::floor(std::ldexp(p, 32));
    if (scaled < 0.0) scaled = 0.0;
    if (scaled > 4294967296.0) scaled = 4294967296.0;
    *T = (uint64_t)scaled;
    return SWO_OK;
}

/* ------------------------------------------------------------------------- */
/* Step (2): canonical labels by flood fill in increasing index order.        */
/* Because seeds are visited in increasing order, the seed of every fill is   */
/* the smallest index of its cluster, so no post-pass is needed.*/
/* ------------------------------------------------------------------------- */
static int label_bonds(uint64_t L, const uint8_t *bonds, uint32_t *labels,
                       uint64_t *n_clusters, uint64_t *largest)
{
    const uint64_t N = L * L;
    std::vector<uint64_t> visited;          /* one bit per site: a uint32 label has no spare value at N = 2^32 */
    std::vector<uint32_t> queue;
    try {
        visited.assign((N + 63) / 64, 0);
    } catch (const std::bad_alloc &) { return SWO_ERR_OOM; }

    uint64_t count = 0, big = 0;
    for (uint64_t s = 0; s < N; ++s) {
        if ((visited[s >> 6] >> (s & 63)) & 1) continue;
        visited[s >> 6] |= (uint64_t)1 << (s & 63);
        labels[s] = (uint32_t)s;
        queue.clear();
        try { queue.push_back((uint32_t)s); } catch (const std::bad_alloc &) { return SWO_ERR_OOM; }
        uint64_t head = 0;
        while (head < queue.size()) {
            const uint64_t i = queue[head++];
            const uint64_t x = i % L, y = i / L;
            const uint64_t r = y * L + (x + 1) % L;
            const uint64_t d = ((y + 1) % L) * L + x;
            const uint64_t l = y * L + (x + L - 1) % L;
            const uint64_t u = ((y + L - 1) % L) * L + x;
            /* the four incident bonds: two owned by i, one by its left and one by its up neighbour */
            const uint64_t nbr[4]   = { r, d, l, u };
            const bool     active[4] = { (bonds[i] & 1) != 0, (bonds[i] & 2) != 0,
                                         (bonds[l] & 1) != 0, (bonds[u] & 2) != 0 };
            for (int k = 0; k < 4; ++k) {
                const uint64_t j = nbr[k];
                if (!active[k]) continue;
                if ((visited[j >> 6] >> (j & 63)) & 1) continue;
                visited[j >> 6] |= (uint64_t)1 << (j & 63);
                labels[j] = (uint32_t)s;
                try { queue.push_back((uint32_t)j); } catch (const std::bad_alloc &) { return SWO_ERR_OOM; }
            }
        }
        ++count;
        if (queue.size() > big) big = queue.size();
    }
    if (n_clusters) *n_clusters = count;
    if (largest) *largest = big;
    return SWO_OK;
}

int swo_label_bonds(uint32_t L, const uint8_t *bonds, uint32_t *labels,
                    uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (L < 2 || L > 65536 || !bonds || !labels) return SWO_ERR_INVALID_ARG;
    return label_bonds(L, bonds, labels, n_clusters, largest_cluster);
}

/* ------------------------------------------------------------------------- */
/* The simulation object.                                                     */
/* ------------------------------------------------------------------------- */
struct swo_ctx {
    uint64_t L, N;
    uint32_t q;
    double   K;
    uint64_t seed;
    uint64_t T;              /* 0 .. 2^32 */
    uint64_t t;              /* sweeps done since init / set_state's t */
    bool     have_spins, have_labels;
    uint64_t n_clusters, largest;
    std::vector<uint8_t>  spins, bonds;
    std::vector<uint32_t> labels;
};

int swo_create(swo_ctx **out, uint32_t L, uint32_t q, double K, uint64_t seed)
{
    if (!out) return SWO_ERR_INVALID_ARG;
    *out = nullptr;
    if (L < 2 || L > 65536 || q < 2 || q > 255) return SWO_ERR_INVALID_ARG;
    uint64_t T;
    if (swo_threshold(K, &T) != SWO_OK) return SWO_ERR_INVALID_ARG;
    swo_ctx *c = new (std::nothrow) swo_ctx();
    if (!c) return SWO_ERR_OOM;
    c->L = L; c->N = (uint64_t)L * L; c->q = q; c->K = K; c->seed = seed; c->T = T; c->t = 0;
    c->have_spins = c->have_labels = false; c->n_clusters = c->largest = 0;
    try {
        c->spins.assign(c->N, 0);
        c->bonds.assign(c->N, 0);
        c->labels.assign(c->N, 0);
    } catch (const std::bad_alloc &) { delete c; return SWO_ERR_OOM; }
    *out = c;
    return SWO_OK;
}

void swo_destroy(swo_ctx *c) { delete c; }

int swo_init(swo_ctx *c, int mode)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (mode == SWO_INIT_ORDERED) {
        for (uint64_t i = 0; i < c->N; ++i) c->spins[i] = 0;
    } else if (mode == SWO_INIT_RANDOM) {
        for (uint64_t i = 0; i < c->N; ++i)
            c->spins[i] = (uint8_t)swo_state_from_draw(swo_draw_init(c->seed, i), c->q);
    } else return SWO_ERR_INVALID_ARG;
    c->t = 0; c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;
    return SWO_OK;
}

int swo_set_state(swo_ctx *c, const uint8_t *spins, uint64_t t)
{
    if (!c || !spins || t > 0xFFFFFFFFull) return SWO_ERR_INVALID_ARG;
    for (uint64_t i = 0; i < c->N; ++i) if (spins[i] >= c->q) return SWO_ERR_INVALID_ARG;
    std::memcpy(c->spins.data(), spins, c->N);
    c->t = t; c->have_spins = true; c->have_labels = false; c->n_clusters = c->largest = 0;
    return SWO_OK;
}

static int one_sweep(swo_ctx *c)
{
    const uint64_t L = c->L, N = c->N;
    const uint32_t t = (uint32_t)c->t;

    /* step (1): bond(i,d) = spins equal AND draw < T  (comparison in 64 bits: T may be 2^32) */
    for (uint64_t i = 0; i < N; ++i) {
        const uint64_t x = i % L, y = i / L;
        const uint64_t r = y * L + (x + 1) % L;
        const uint64_t d = ((y + 1) % L) * L + x;
        uint8_t b = 0;
        if (c->spins[i] == c->spins[r] && (uint64_t)swo_draw_bond(c->seed, t, i, 0) < c->T) b |= 1;
        if (c->spins[i] == c->spins[d] && (uint64_t)swo_draw_bond(c->seed, t, i, 1) < c->T) b |= 2;
        c->bonds[i] = b;
    }

    /* step (2): canonical labels */
    int rc = label_bonds(L, c->bonds.data(), c->labels.data(), &c->n_clusters, &c->largest);
    if (rc != SWO_OK) return rc;

    /* step (3): every cluster gets the state drawn from the key of its root; the
     * root is visited before any other member because it has the smallest index */
    for (uint64_t i = 0; i < N; ++i) {
        const uint64_t r = c->labels[i];
        if (r == i) c->spins[i] = (uint8_t)swo_state_from_draw(swo_draw_flip(c->seed, t, r), c->q);
        else        c->spins[i] = c->spins[r];
    }
    c->t += 1;
    c->have_labels = true;
    return SWO_OK;
}

int swo_sweep(swo_ctx *c, uint64_t n)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    if (c->t + n > 0x100000000ull) return SWO_ERR_STATE;    /* the sweep field of the counter is 32 bits */
    for (uint64_t k = 0; k < n; ++k) {
        int rc = one_sweep(c);
        if (rc != SWO_OK) return rc;
    }
    return SWO_OK;
}

int swo_measure(swo_ctx *c, uint64_t *energy_bonds, uint64_t *mag_counts,
                uint64_t *n_clusters, uint64_t *largest_cluster)
{
    if (!c) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    const uint64_t L = c->L, N = c->N;
    if (energy_bonds) {
        uint64_t e = 0;
        for (uint64_t i = 0; i < N; ++i) {
            const uint64_t x = i % L, y = i / L;
            if (c->spins[i] == c->spins[y * L + (x + 1) % L]) ++e;
            if (c->spins[i] == c->spins[((y + 1) % L) * L + x]) ++e;
        }
        *energy_bonds = e;
    }
    if (mag_counts) {
        for (uint32_t s = 0; s < c->q; ++s) mag_counts[s] = 0;
        for (uint64_t i = 0; i < N; ++i) mag_counts[c->spins[i]] += 1;
    }
    /* cluster statistics belong to the bond configuration of the last sweep (R15) */
    if (n_clusters) *n_clusters = c->have_labels ? c->n_clusters : 0;
    if (largest_cluster) *largest_cluster = c->have_labels ? c->largest : 0;
    return SWO_OK;
}

int swo_sweep_measure(swo_ctx *c, uint64_t n, uint64_t *out)
{
    if (!c || !out) return SWO_ERR_INVALID_ARG;
    const uint64_t stride = 3 + (uint64_t)c->q;
    for (uint64_t k = 0; k < n; ++k) {
        int rc = swo_sweep(c, 1);
        if (rc != SWO_OK) return rc;
        uint64_t *row = out + k * stride;
        rc = swo_measure(c, &row[0], &row[3], &row[1], &row[2]);
        if (rc != SWO_OK) return rc;
    }
    return SWO_OK;
}

int swo_get_spins(swo_ctx *c, uint8_t *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_spins) return SWO_ERR_STATE;
    std::memcpy(dst, c->spins.data(), c->N);
    return SWO_OK;
}

int swo_get_labels(swo_ctx *c, uint32_t *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_labels) return SWO_ERR_STATE;
    std::memcpy(dst, c->labels.data(), c->N * sizeof(uint32_t));
    return SWO_OK;
}

int swo_get_bonds(swo_ctx *c, uint8_t *dst)
{
    if (!c || !dst) return SWO_ERR_INVALID_ARG;
    if (!c->have_labels) return SWO_ERR_STATE;
    std::memcpy(dst, c->bonds.data(), c->N);
    return SWO_OK;
}

int swo_get_threshold(swo_ctx *c, uint64_t *T)
{
    if (!c || !T) return SWO_ERR_INVALID_ARG;
    *T = c->T;
    return SWO_OK;
}

int swo_get_time(swo_ctx *c, uint64_t *t)
{
    if (!c || !t) return SWO_ERR_INVALID_ARG;
    *t = c->t;
    return SWO_OK;
}
