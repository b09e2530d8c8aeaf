"""Pins for the oracle's cluster labeling (PAPER.md:40 step 2) -- CPU only.

The flood fill is checked against things that are not itself:
  * scipy.sparse.csgraph.connected_components (a library routine) on random and adversarial masks,
    with the canonical label recomputed as the per-component minimum index by numpy;
  * brute force: boolean transitive closure of the adjacency matrix on tiny lattices;
  * structural invariants and the two trivial limits.
"""
import numpy as np
import pytest
import scipy.sparse as sp
from scipy.sparse.csgraph import connected_components

from oracle import binding as orc
from paper_1208_2080_b200 import workloads as wl


def edges_of(bonds):
    """(u, v) arrays of the active bonds of an (L, L) mask on the periodic lattice."""
    L = bonds.shape[0]
    idx = np.arange(L * L).reshape(L, L)
    right = np.roll(idx, -1, axis=1)
    down = np.roll(idx, -1, axis=0)
    r = (bonds & 1) != 0
    d = (bonds & 2) != 0
    return np.concatenate([idx[r], idx[d]]), np.concatenate([right[r], down[d]])


def canonical_by_scipy(bonds):
    L = bonds.shape[0]
    N = L * L
    u, v = edges_of(bonds)
    g = sp.coo_matrix((np.ones(u.size, dtype=np.int8), (u, v)), shape=(N, N))
    ncomp, comp = connected_components(g, directed=False)
    mins = np.full(ncomp, N, dtype=np.int64)
    np.minimum.at(mins, comp, np.arange(N))
    sizes = np.bincount(comp, minlength=ncomp)
    return mins[comp].astype(np.uint32), int(ncomp), int(sizes.max())


def equal_spin_bonds(spins):
    """Bond mask with every bond between equal neighbours active (the K = +inf mask)."""
    r = spins == np.roll(spins, -1, axis=1)
    d = spins == np.roll(spins, -1, axis=0)
    return r.astype(np.uint8) | (d.astype(np.uint8) << 1)


@pytest.mark.parametrize("L", [2, 3, 4, 5, 16, 33, 64, 100])
@pytest.mark.parametrize("density", [0.0, 0.2, 0.5, 0.6, 1.0])
def test_random_masks_match_scipy(L, density):
    bonds = wl.bonds_random(L, density, seed=1000 * L + int(density * 10))
    labels, nc, big = orc.label_bonds(bonds)
    want, want_nc, want_big = canonical_by_scipy(bonds)
    assert np.array_equal(labels, want)
    assert (nc, big) == (want_nc, want_big)


@pytest.mark.parametrize("L", [8, 31, 64, 96])
def test_adversarial_masks_match_scipy(L):
    for name, spins in wl.crafted_lattices(L, 3).items():
        bonds = equal_spin_bonds(spins)
        labels, nc, big = orc.label_bonds(bonds)
        want, want_nc, want_big = canonical_by_scipy(bonds)
        assert np.array_equal(labels, want), name
        assert (nc, big) == (want_nc, want_big), name


def test_spiral_is_one_long_cluster():
    L = 64
    spins = wl.spins_spiral(L)
    labels, _, _ = orc.label_bonds(equal_spin_bonds(spins))
    path = labels.reshape(L, L)[spins == 0]
    assert path.size > L * L // 3 and np.all(path == path[0]) and path[0] == L + 1


@pytest.mark.parametrize("L", [2, 3, 4])
def test_brute_force_transitive_closure(L):
    N = L * L
    rng = np.random.default_rng(L)
    for trial in range(40):
        bonds = wl.bonds_random(L, rng.uniform(0.1, 0.9), seed=trial + 17 * L)
        u, v = edges_of(bonds)
        reach = np.eye(N, dtype=bool)
        reach[u, v] = True
        reach[v, u] = True
        for _ in range(N):                               # N squarings are more than enough
            reach = reach | ((reach.astype(np.int32) @ reach.astype(np.int32)) > 0)
        want = np.array([np.flatnonzero(reach[i])[0] for i in range(N)], dtype=np.uint32)
        labels, nc, big = orc.label_bonds(bonds)
        assert np.array_equal(labels, want)
        assert nc == len(set(want.tolist()))
        assert big == max(np.bincount(want))


def test_invariants_on_a_critical_like_mask():
    L = 128
    bonds = wl.bonds_random(L, 0.5, seed=3)
    labels, nc, big = orc.label_bonds(bonds)
    i = np.arange(L * L, dtype=np.uint32)
    assert np.all(labels <= i)                                   # proper label = smallest
    assert np.array_equal(labels[labels], labels)                # roots are fixed points
    u, v = edges_of(bonds)
    assert np.array_equal(labels[u], labels[v])                  # an active bond joins equal labels
    assert nc == int(np.count_nonzero(labels == i))
    assert big == int(np.bincount(labels).max())
    # every non-root site has an active bond to a site with the same label (connectedness, locally)
    has = np.zeros(L * L, dtype=bool)
    has[u] = True
    has[v] = True
    assert np.all(has[labels != i])


def test_limits_and_double_bonds():
    for L in (2, 3, 7, 32):
        N = L * L
        labels, nc, big = orc.label_bonds(np.zeros((L, L), dtype=np.uint8))
        assert np.array_equal(labels, np.arange(N)) and (nc, big) == (N, 1)
        labels, nc, big = orc.label_bonds(np.full((L, L), 3, dtype=np.uint8))
        assert np.all(labels == 0) and (nc, big) == (1, N)
    # L = 2: right(x=1) = x=0, so a site pair is joined by two distinct bonds; either one suffices
    b = np.zeros((2, 2), dtype=np.uint8)
    b[0, 1] = 1                                                   # only the wrap-around bond (1,0)->(0,0)
    labels, nc, _ = orc.label_bonds(b)
    assert labels.tolist() == [0, 0, 2, 3] and nc == 3
    b = np.zeros((2, 2), dtype=np.uint8)
    b[1, 0] = 2                                                   # wrap-around down bond (0,1)->(0,0)
    labels, nc, _ = orc.label_bonds(b)
    assert labels.tolist() == [0, 1, 0, 3] and nc == 3
    # only-right bonds: every row is one ring; only-down bonds: every column
    L = 9
    labels, nc, big = orc.label_bonds(np.full((L, L), 1, dtype=np.uint8))
    assert np.array_equal(labels.reshape(L, L), np.repeat(np.arange(L)[:, None] * L, L, axis=1)) and (nc, big) == (L, L)
    labels, nc, big = orc.label_bonds(np.full((L, L), 2, dtype=np.uint8))
    assert np.array_equal(labels.reshape(L, L), np.repeat(np.arange(L)[None, :], L, axis=0)) and (nc, big) == (L, L)
