"""Pins for the oracle's full sweep (PAPER.md:40 steps 1-3) -- CPU only.

  * the two tiny end-to-end vectors of SURVEY.md sec. 8(c-4) (an independent implementation's output);
  * step-by-step invariants tying bonds, labels, new spins and observables together through the
    separately pinned pieces (draws, threshold, scipy labeling);
  * the limits K = 0 and K = +inf, where the result has a closed form.
"""
import math

import numpy as np
import pytest

from oracle import binding as orc
from oracle.binding import Oracle
from paper_1208_2080_b200 import workloads as wl
from test_oracle_labeling import canonical_by_scipy


def test_tiny_golden_sweeps(golden):
    rows = golden("tiny_sweeps.txt")
    sim = None
    checked = 0
    for row in rows:
        f = row.split()
        if f[0] == "case":
            L, q, seed, K = int(f[1]), int(f[2]), int(f[3]), float.fromhex(f[4])
            sim = Oracle(L, q, K, seed)
            sim.init("random")
        elif f[0] == "init":
            assert sim.get_spins().tolist() == [int(v) for v in f[1:]]
        elif f[0] == "bonds":
            sim.sweep(1)
            assert sim.get_bonds().tolist() == [int(v) for v in f[1:]]
        elif f[0] == "labels":
            assert sim.get_labels().tolist() == [int(v) for v in f[1:]]
        elif f[0] == "spins":
            assert sim.get_spins().tolist() == [int(v) for v in f[1:]]
        elif f[0] == "obs":
            v = [int(x) for x in f[1:]]
            m = sim.measure()
            assert [m["energy_bonds"], m["n_clusters"], m["largest_cluster"]] + m["mag_counts"] == v
            checked += 1
    assert checked == 4


def energy_bonds_numpy(s):
    return int(np.count_nonzero(s == np.roll(s, -1, axis=1)) + np.count_nonzero(s == np.roll(s, -1, axis=0)))


@pytest.mark.parametrize("L,q,K,start", [
    (2, 2, 0.7, "random"), (3, 3, 1.0, "random"), (5, 4, 1.2, "random"), (16, 2, wl.k_critical(2), "ordered"),
    (33, 10, wl.k_critical(10), "random"), (64, 3, wl.k_critical(3), "random"), (70, 2, 0.3, "random"),
])
def test_sweep_invariants(L, q, K, start):
    seed = 11
    sim = Oracle(L, q, K, seed)
    sim.init(start)
    T = sim.get_threshold()
    assert T == orc.threshold(K)
    N = L * L
    for t in range(4):
        before = sim.get_spins().reshape(L, L)
        sim.sweep(1)
        assert sim.get_time() == t + 1
        bonds = sim.get_bonds().reshape(L, L)
        labels = sim.get_labels()
        after = sim.get_spins()
        # step 1: a bond is active iff the spins are equal AND the (pinned) draw is below the (pinned) threshold
        eq_r = before == np.roll(before, -1, axis=1)
        eq_d = before == np.roll(before, -1, axis=0)
        dr = np.array([orc.draw_bond(seed, t, i, 0) for i in range(N)], dtype=np.uint64).reshape(L, L)
        dd = np.array([orc.draw_bond(seed, t, i, 1) for i in range(N)], dtype=np.uint64).reshape(L, L)
        want = (eq_r & (dr < T)).astype(np.uint8) | ((eq_d & (dd < T)).astype(np.uint8) << 1)
        assert np.array_equal(bonds, want)
        # step 2: canonical labels of exactly that mask (scipy)
        want_labels, nc, big = canonical_by_scipy(bonds)
        assert np.array_equal(labels, want_labels)
        # step 3: every site takes the state drawn from its root's key
        roots = np.unique(labels)
        state = {int(r): orc.state_from_draw(orc.draw_flip(seed, t, int(r)), q) for r in roots}
        assert np.array_equal(after, np.array([state[int(r)] for r in labels], dtype=np.uint8))
        # observables
        m = sim.measure()
        assert m["energy_bonds"] == energy_bonds_numpy(after.reshape(L, L))
        assert m["mag_counts"] == np.bincount(after, minlength=q).tolist()
        assert (m["n_clusters"], m["largest_cluster"]) == (nc, big)


def test_zero_temperature_limit_follows_the_root_zero_flip_sequence(golden):
    # ordered start + K = inf: one cluster with root 0 forever; the lattice is mulhi(FLIP(root 0, t), q)
    seq = {}
    for row in golden("contract_examples.txt"):
        f = row.split()
        if f[0] == "flipstates":
            seq[int(f[1])] = [int(v) for v in f[2:]]
    for q in (2, 3, 4, 10):
        L = 6
        sim = Oracle(L, q, math.inf, 1)
        sim.init("ordered")
        assert sim.get_threshold() == 1 << 32
        for t in range(8):
            sim.sweep(1)
            s = sim.get_spins()
            assert np.all(s == seq[q][t])
            assert np.all(sim.get_labels() == 0) and np.all(sim.get_bonds() == 3)
            m = sim.measure()
            assert m["energy_bonds"] == 2 * L * L and m["n_clusters"] == 1 and m["largest_cluster"] == L * L
            assert m["mag_counts"][seq[q][t]] == L * L


def test_infinite_temperature_limit():
    # K = 0: no bond is ever active, labels[i] = i, spins are iid uniform draws keyed by the site itself
    L, q, seed = 48, 3, 9
    sim = Oracle(L, q, 0.0, seed)
    sim.init("ordered")
    es, mags = [], []
    for t in range(20):
        sim.sweep(1)
        assert not sim.get_bonds().any()
        assert np.array_equal(sim.get_labels(), np.arange(L * L))
        s = sim.get_spins()
        if t < 2:
            assert s.tolist() == [orc.state_from_draw(orc.draw_flip(seed, t, i), q) for i in range(L * L)]
        m = sim.measure()
        assert m["n_clusters"] == L * L and m["largest_cluster"] == 1
        es.append(m["energy_bonds"]); mags.append(m["mag_counts"])
    N = L * L
    # <energy_bonds> = 2N/q, variance per sweep 2N(1/q)(1-1/q); 20 independent sweeps
    se = math.sqrt(2 * N * (1 / q) * (1 - 1 / q) / 20)
    assert abs(np.mean(es) - 2 * N / q) < 5 * se
    se_m = math.sqrt(N * (1 / q) * (1 - 1 / q) / 20)
    assert np.all(np.abs(np.mean(mags, axis=0) - N / q) < 5 * se_m)


def test_state_machine_and_arguments():
    with pytest.raises(orc.OracleError):
        Oracle(1, 2, 0.5, 1)
    with pytest.raises(orc.OracleError):
        Oracle(4, 1, 0.5, 1)
    with pytest.raises(orc.OracleError):
        Oracle(4, 256, 0.5, 1)
    with pytest.raises(orc.OracleError):
        Oracle(4, 2, -0.5, 1)
    sim = Oracle(4, 2, 0.5, 1)
    with pytest.raises(orc.OracleError):
        sim.sweep(1)                                   # no spins yet
    sim.init("random")
    with pytest.raises(orc.OracleError):
        sim.get_labels()                               # no sweep yet
    m = sim.measure()
    assert m["n_clusters"] == 0 and m["largest_cluster"] == 0
    with pytest.raises(orc.OracleError):
        sim.set_state(np.full(16, 2, dtype=np.uint8), 0)    # state out of range
    # determinism and restartability: (spins, t) is the whole state
    sim.sweep(5)
    snap, t = sim.get_spins(), sim.get_time()
    sim.sweep(3)
    end = sim.get_spins()
    again = Oracle(4, 2, 0.5, 1)
    again.set_state(snap, t)
    again.sweep(3)
    assert np.array_equal(again.get_spins(), end)


def k_for_threshold(target):
    """A coupling K whose integer threshold is exactly `target` (bisection on the pinned, monotone map)."""
    lo, hi = 0.0, 40.0
    for _ in range(200):
        mid = 0.5 * (lo + hi)
        if orc.threshold(mid) < target:
            lo = mid
        else:
            hi = mid
    assert orc.threshold(hi) == target
    return hi


def test_comparison_is_strict_draw_below_threshold(golden):
    # north_star: "active iff a uint32 draw is BELOW floor(p*2^32)".  Choose K so that T equals a known
    # draw exactly: that bond must be inactive, and active once T is one larger.
    draw = orc.draw_bond(1, 0, 0, 0)
    assert draw == 0x127BEE41                                  # SURVEY.md sec. 8(c-3) contract example
    for T, want in ((draw, 0), (draw + 1, 1)):
        sim = Oracle(4, 2, k_for_threshold(T), 1)
        sim.init("ordered")
        sim.sweep(1)
        assert sim.get_bonds()[0] & 1 == want
    draw_d = orc.draw_bond(1, 0, 1, 1)                         # down bond of site 1
    for T, want in ((draw_d, 0), (draw_d + 1, 2)):
        sim = Oracle(4, 2, k_for_threshold(T), 1)
        sim.init("ordered")
        sim.sweep(1)
        assert sim.get_bonds()[1] & 2 == want


@pytest.mark.parametrize("L,q,K,start", [(12, 2, wl.k_critical(2), "random"), (20, 3, 0.9, "random"), (9, 5, 1.3, "ordered")])
def test_sweep_measure_rows_follow_the_header_column_order(L, q, K, start):
    # swo_sweep_measure(n) must equal n x (swo_sweep(1), swo_measure) with the columns of oracle/sw_oracle.h:
    # [energy_bonds, n_clusters, largest_cluster, mag_counts[0..q-1]].  n_clusters and largest_cluster are NOT taken
    # from the oracle's counters here: they are recounted by scipy from the bonds of a second, step-by-step run of the
    # same chain, so a swap of the two columns (or of &row[1] / &row[2]) fails.
    n, seed = 12, 17
    series = Oracle(L, q, K, seed)
    series.init(start)
    rows = series.sweep_measure(n)
    assert rows.shape == (n, 3 + q) and rows.dtype == np.uint64
    step = Oracle(L, q, K, seed)
    step.init(start)
    saw_different = False
    for k in range(n):
        step.sweep(1)
        spins = step.get_spins().reshape(L, L)
        _, nc, big = canonical_by_scipy(step.get_bonds().reshape(L, L))
        want = [energy_bonds_numpy(spins), nc, big] + np.bincount(spins.reshape(-1), minlength=q).tolist()
        assert rows[k].tolist() == want, f"row {k}"
        saw_different |= nc != big
    assert saw_different                                   # otherwise a swap of columns 1 and 2 could hide
    assert np.array_equal(series.get_spins(), step.get_spins()) and series.get_time() == step.get_time() == n


def test_init_and_set_state_reset_the_chain():
    # sw_init sets t = 0 and forgets the labels: a chain re-initialised after some sweeps repeats the fresh chain exactly
    # (the sweep counter is a word of every Philox counter, so a stale t would change every draw)
    L, q, K, seed = 10, 3, 1.0, 5
    fresh = Oracle(L, q, K, seed)
    fresh.init("random")
    fresh.sweep(3)
    again = Oracle(L, q, K, seed)
    again.init("ordered")
    again.sweep(2)
    again.init("random")
    assert again.get_time() == 0
    m = again.measure()
    assert m["n_clusters"] == 0 and m["largest_cluster"] == 0
    with pytest.raises(orc.OracleError):
        again.get_labels()
    again.sweep(3)
    assert again.get_time() == 3
    assert np.array_equal(again.get_spins(), fresh.get_spins()) and np.array_equal(again.get_labels(), fresh.get_labels())
    # set_state(spins, t) resumes at exactly that t
    mid = Oracle(L, q, K, seed)
    mid.init("random")
    mid.sweep(1)
    resumed = Oracle(L, q, K, seed)
    resumed.set_state(mid.get_spins(), 1)
    assert resumed.get_time() == 1
    resumed.sweep(2)
    assert np.array_equal(resumed.get_spins(), fresh.get_spins())
