"""Pins for the XY oracle (oracle/sw_xy_oracle.cpp, Wolff embedding) -- CPU only.

Nothing here re-types the oracle's formulas.  What fixes them instead:
  * geometry of a reflection: the component along r changes sign, the component across r and the length do not, two
    reflections are the identity;
  * the structure of a sweep: bonds only join sites whose projections have the same sign, labels are the scipy labels of
    those bonds, a cluster moves as a whole (all reflected or none), half of the clusters move;
  * closed forms: ordered start -> every bond is active with p = 1 - exp(-2 K r_x^2) (binomial count); K = 0 -> no bond,
    every site its own cluster; the reflection angles are uniform;
  * the equilibrium the chain must sample (detailed balance of the embedded dynamics): the exact nearest-neighbour
    correlation of the 2 x 2 torus by direct numerical integration over the three relative angles, the high-temperature
    limit <cos> -> K/2 and the spin-wave limit <cos> -> 1 - (1 - 1/N)/(4K).
"""
import math

import numpy as np
import pytest

from oracle import binding as orc
from oracle import xy_binding as xy
from oracle.xy_binding import OracleXY
from test_oracle_labeling import canonical_by_scipy


def test_reflection_geometry():
    rng = np.random.default_rng(3)
    for _ in range(200):
        th, ph = rng.uniform(0, 2 * math.pi, 2)
        s, r = (math.cos(th), math.sin(th)), (math.cos(ph), math.sin(ph))
        perp = (-r[1], r[0])
        s2 = xy.reflect(s, r)
        assert abs(np.dot(s2, r) + np.dot(s, r)) < 1e-15          # along r: sign flipped
        assert abs(np.dot(s2, perp) - np.dot(s, perp)) < 1e-15    # across r: unchanged
        assert abs(np.hypot(*s2) - 1.0) < 1e-15
        s3 = xy.reflect(s2, r)
        assert abs(s3[0] - s[0]) < 1e-15 and abs(s3[1] - s[1]) < 1e-15
        assert abs(xy.projection(s, r) - np.dot(s, r)) < 3e-16


def test_reflection_directions_are_unit_vectors_with_uniform_angles():
    ang = []
    for t in range(4000):
        r = xy.reflection(11, t)
        assert abs(np.hypot(*r) - 1.0) < 1e-15
        ang.append(math.atan2(r[1], r[0]) % (2 * math.pi))
    counts, _ = np.histogram(ang, bins=8, range=(0, 2 * math.pi))
    assert np.all(np.abs(counts - 500) < 5 * math.sqrt(500 * 7 / 8))
    assert xy.reflection(11, 5) != xy.reflection(12, 5) and xy.reflection(11, 5) != xy.reflection(11, 6)
    # the angle comes from word 0 of Philox(counter (0, 0, t, 3), key seed): phi = 2 pi (w0 + 1/2) / 2^32
    w0 = orc.philox4x32_10((0, 0, 5, 3), (11, 0))[0]
    phi = 2 * math.pi * (w0 + 0.5) / 2 ** 32
    assert np.allclose(xy.reflection(11, 5), (math.cos(phi), math.sin(phi)), atol=1e-15)


def test_bond_threshold_limits_and_monotonicity():
    assert xy.bond_threshold(1.0, 0.5, -0.5) == 0 and xy.bond_threshold(1.0, -0.5, 0.5) == 0 and xy.bond_threshold(1.0, 0.0, 1.0) == 0
    assert xy.bond_threshold(0.0, 1.0, 1.0) == 0
    assert xy.bond_threshold(math.inf, 0.3, 0.2) == 1 << 32 and xy.bond_threshold(math.inf, -0.3, -0.2) == 1 << 32
    assert xy.bond_threshold(math.inf, 0.3, -0.2) == 0
    # with a_i = a_j = 1 the embedded coupling is the Ising one: the threshold of the Potts oracle at coupling 2K
    for K in (0.1, 0.44, 1.0, 3.0):
        assert xy.bond_threshold(K, 1.0, 1.0) == orc.threshold(2 * K) == xy.bond_threshold(K, -1.0, -1.0)
    ts = [xy.bond_threshold(1.1, a, 0.7) for a in np.linspace(0.01, 1.0, 50)]
    assert all(b >= a for a, b in zip(ts, ts[1:])) and ts[0] > 0
    # p = 1 - exp(-2 K a_i a_j), to the resolution of the integer threshold
    assert abs(xy.bond_threshold(0.8, 0.6, 0.9) / 2 ** 32 - (1 - math.exp(-2 * 0.8 * 0.6 * 0.9))) < 2 ** -31


def test_init_spins_are_unit_vectors_spread_over_the_circle():
    s = np.array([xy.init_spin(5, i) for i in range(8000)])
    assert np.all(np.abs(np.hypot(s[:, 0], s[:, 1]) - 1.0) < 1e-15)
    counts, _ = np.histogram(np.arctan2(s[:, 1], s[:, 0]), bins=8, range=(-math.pi, math.pi))
    assert np.all(np.abs(counts - 1000) < 6 * math.sqrt(1000))          # (nearly) uniform: the rejection step keeps the corner bias small
    assert xy.init_spin(5, 3) != xy.init_spin(6, 3)


@pytest.mark.parametrize("L,K,start", [(8, 1.0, "random"), (16, 1.12, "random"), (12, 0.5, "ordered"), (5, 2.0, "random"), (2, 1.0, "random")])
def test_sweep_structure(L, K, start):
    seed = 9
    sim = OracleXY(L, K, seed)
    sim.init(start)
    N = L * L
    moved_clusters = total_clusters = 0
    for t in range(6):
        before = sim.get_spins()
        sim.sweep(1)
        assert sim.get_time() == t + 1
        r = np.array(xy.reflection(seed, t))
        a = before @ r
        bonds = sim.get_bonds().reshape(L, L)
        A = a.reshape(L, L)
        right_ok = A * np.roll(A, -1, axis=1) > 0
        down_ok = A * np.roll(A, -1, axis=0) > 0
        assert not np.any(((bonds & 1) != 0) & ~right_ok) and not np.any(((bonds & 2) != 0) & ~down_ok)
        labels, nc, big = canonical_by_scipy(bonds)
        assert np.array_equal(sim.get_labels(), labels)
        after = sim.get_spins()
        moved = np.abs(after - before).max(axis=1) > 0
        # a reflected spin: projection flipped; an untouched one: identical bits
        assert np.allclose((after @ r)[moved], -a[moved], atol=1e-15)
        perp = np.array([-r[1], r[0]])
        assert np.allclose(after @ perp, before @ perp, atol=1e-15)
        for root in np.unique(labels):
            members = labels == root
            # (a spin with a = 0 exactly would not move; none occurs here)
            assert moved[members].all() or not moved[members].any()
            want = orc.state_from_draw(orc.draw_flip(seed, t, int(root)), 2) == 1
            assert bool(moved[members][0]) == want
            moved_clusters += int(moved[members][0]); total_clusters += 1
        m = sim.measure()
        assert (m["n_clusters"], m["largest_cluster"]) == (nc, big)
        S = after.reshape(L, L, 2)
        e = np.sum(S * np.roll(S, -1, axis=1)) + np.sum(S * np.roll(S, -1, axis=0))
        assert abs(m["energy_sum"] - e) < 1e-9 * N and np.allclose(m["mag"], after.sum(axis=0), atol=1e-9 * N)
        assert np.allclose(np.hypot(after[:, 0], after[:, 1]), 1.0, atol=1e-13)
    if total_clusters > 100:
        assert abs(moved_clusters / total_clusters - 0.5) < 5 * 0.5 / math.sqrt(total_clusters)


def test_ordered_start_bond_count_is_binomial_and_k_zero_has_no_bonds():
    L, K, seed = 64, 0.7, 4
    sim = OracleXY(L, K, seed)
    sim.init("ordered")                                          # all spins (1, 0): a_i = r_x for every site
    sim.sweep(1)
    rx = xy.reflection(seed, 0)[0]
    p = 1 - math.exp(-2 * K * rx * rx)
    b = sim.get_bonds()
    n = int(np.count_nonzero(b & 1) + np.count_nonzero(b & 2))
    assert abs(n - 2 * L * L * p) < 5 * math.sqrt(2 * L * L * p * (1 - p))
    hot = OracleXY(16, 0.0, 1)
    hot.init("random")
    hot.sweep(3)
    assert not hot.get_bonds().any() and np.array_equal(hot.get_labels(), np.arange(256))
    assert hot.measure()["n_clusters"] == 256


def exact_nn_correlation_2x2(K, n=96):
    """<cos(theta_i - theta_j)> for nearest neighbours on the 2 x 2 torus: four sites on a ring, every ring bond doubled
    (periodic wrap), H = -2J sum_ring cos.  Direct integration over the three relative angles (periodic rectangle rule)."""
    g = np.linspace(0, 2 * math.pi, n, endpoint=False)
    a, b, c = np.meshgrid(g, g, g, indexing="ij")                # angles of sites 1, 2, 3 relative to site 0: ring 0-1-3-2-0
    e = np.cos(a) + np.cos(c - a) + np.cos(c - b) + np.cos(b)
    w = np.exp(2 * K * (e - 4.0))
    return float(np.sum(w * e / 4.0) / np.sum(w))


@pytest.mark.parametrize("K,seed", [(0.4, 1), (1.0, 2)])
def test_2x2_torus_matches_direct_integration(K, seed):
    exact = exact_nn_correlation_2x2(K)
    assert abs(exact - exact_nn_correlation_2x2(K, 64)) < 1e-9   # the quadrature has converged
    sim = OracleXY(2, K, seed)
    sim.init("random")
    sim.sweep(200)
    vals = []
    for _ in range(60000):
        sim.sweep(1)
        vals.append(sim.measure()["energy_sum"] / 8.0)
    vals = np.array(vals)
    nb = 30
    se = np.std([b.mean() for b in np.array_split(vals, nb)], ddof=1) / math.sqrt(nb)
    assert abs(vals.mean() - exact) < 4 * se and se < 0.004, (vals.mean(), exact, se)


def test_high_and_low_temperature_limits():
    # K -> 0: <cos> = K/2 + O(K^3) per bond.  K -> inf (spin waves): 1 - (1 - 1/N)/(4K) + O(1/K^2).
    L = 8
    for K, want, tol in ((0.05, 0.025, 0.002), (12.0, 1 - (1 - 1 / 64) / 48.0, 0.0012)):
        sim = OracleXY(L, K, 3)
        sim.init("random" if K < 1 else "ordered")
        sim.sweep(300)
        vals = []
        for _ in range(6000):
            sim.sweep(1)
            vals.append(sim.measure()["energy_sum"] / (2 * L * L))
        assert abs(np.mean(vals) - want) < tol, (K, np.mean(vals), want)
