"""Seeded synthetic inputs and the workload table -- shared by the tests, bench.py and smoke().

This module holds NONE of the method's arithmetic (no Philox, no threshold, no
labeling): only the parameters of BASELINE.json's five configs and generators of
hand-crafted spin lattices / bond masks used as adversarial inputs.  Random
numbers the method itself draws are never produced here; both the CUDA library
and the CPU oracle implement the counter-based generator on their own.

Lattice conventions: L x L periodic square lattice, site
i = y*L + x, spins 0..q-1 as uint8.
"""
from __future__ import annotations

import math

import numpy as np


def k_critical(q: int) -> float:
    """K_c = ln(1 + sqrt(q)); the paper states it for q = 2 as T_c/J = 1/ln(1+sqrt 2)."""
    return math.log(1.0 + math.sqrt(float(q)))


# BASELINE.json "configs", restated concretely (seed = 1 everywhere).
CONFIGS = {
    "c1_L256_q2": dict(L=256, q=2, K=k_critical(2), start="random", sweeps=200, seed=1),
    "c2_L4096_q2": dict(L=4096, q=2, K=k_critical(2), start="ordered", sweeps=1000, seed=1),
    "c3_L8192_q3": dict(L=8192, q=3, K=k_critical(3), start="random", sweeps=500, seed=1),
    "c3_L8192_q4": dict(L=8192, q=4, K=k_critical(4), start="random", sweeps=500, seed=1),
    "c4_L16384_q10_above": dict(L=16384, q=10, K=k_critical(10) * 1.005, start="random", sweeps=200, seed=1),
    "c4_L16384_q10_below": dict(L=16384, q=10, K=k_critical(10) * 0.995, start="random", sweeps=200, seed=1),
    "c5_L65536_q2": dict(L=65536, q=2, K=k_critical(2), start="random", sweeps=100, seed=1),
}
# not a BASELINE.json config: the headline physics at a size whose working set (1.3 GiB) is well beyond
# the L2 but small enough for an `ncu --set full` capture (ncu replays each kernel ~40 times)
CONFIGS["p_L16384_q2"] = dict(L=16384, q=2, K=k_critical(2), start="random", sweeps=100, seed=1)
HEADLINE = "c5_L65536_q2"


# --------------------------------------------------------------------------
# Hand-crafted spin lattices.  With K = +inf every bond between equal
# neighbours is active, so the clusters are exactly the connected regions of
# equal spin: these lattices are adversarial inputs for the labeling step.
# --------------------------------------------------------------------------

def spins_uniform_random(L: int, q: int, seed: int) -> np.ndarray:
    rng = np.random.default_rng(seed)
    return rng.integers(0, q, size=(L, L), dtype=np.uint8)


def spins_spiral(L: int) -> np.ndarray:
    """A single one-site-wide path of 0s spiralling inwards from (1,1); everything else is 1.

    The rim stays wall so the periodic seam does not short-cut the path: the path is one
    cluster whose graph diameter is ~L*L/2, the worst case for propagation-style labeling.
    """
    s = np.ones((L, L), dtype=np.uint8)
    if L < 4:
        s[0, 0] = 0
        return s
    lo, hi = 1, L - 2

    def inside(a, b):
        return lo <= a <= hi and lo <= b <= hi

    def can_move(x, y, dx, dy):
        nx, ny = x + dx, y + dy
        if not inside(nx, ny) or s[ny, nx] == 0:
            return False
        ax, ay = nx + dx, ny + dy                      # keep a wall in front ...
        if inside(ax, ay) and s[ay, ax] == 0:
            return False
        lx, ly = nx + dy, ny - dx                      # ... and on the outer (left-hand) side
        if inside(lx, ly) and s[ly, lx] == 0:
            return False
        return True

    x, y, dx, dy = lo, lo, 1, 0
    s[y, x] = 0
    while True:
        if can_move(x, y, dx, dy):
            x, y = x + dx, y + dy
            s[y, x] = 0
            continue
        dx, dy = -dy, dx                               # turn right (clockwise in screen coordinates)
        if not can_move(x, y, dx, dy):
            break
    return s


def spins_comb(L: int) -> np.ndarray:
    """Two interlocked combs: teeth of 0 on the even columns hanging from a spine on row 0, and
    teeth of 1 on the odd columns standing on a spine on row L-1 (which also cuts the 0-teeth
    from wrapping back onto their own spine across the periodic seam)."""
    s = np.ones((L, L), dtype=np.uint8)
    s[:, 0::2] = 0
    s[0, :] = 0
    s[L - 1, :] = 1
    return s


def spins_stripes(L: int, q: int, width: int, vertical: bool) -> np.ndarray:
    idx = (np.arange(L) // max(1, width)) % q
    s = np.broadcast_to(idx[None, :] if vertical else idx[:, None], (L, L))
    return np.ascontiguousarray(s, dtype=np.uint8)


def spins_checkerboard(L: int, q: int = 2) -> np.ndarray:
    y, x = np.mgrid[0:L, 0:L]
    return ((x + y) % q).astype(np.uint8)


def spins_blocks(L: int, q: int, block: int, seed: int) -> np.ndarray:
    """Random state per block x block square (large clusters with ragged merges across tile borders)."""
    rng = np.random.default_rng(seed)
    nb = (L + block - 1) // block
    coarse = rng.integers(0, q, size=(nb, nb), dtype=np.uint8)
    return np.ascontiguousarray(np.kron(coarse, np.ones((block, block), dtype=np.uint8))[:L, :L])


def spins_dominoes(L: int, dx: int, dy: int, vertical: bool, q: int = 251) -> np.ndarray:
    """A tiling by 1 x 2 (or 2 x 1) dominoes shifted by (dx, dy), each domino with its own state (distinct from its
    neighbours' except for rare hash collisions): with K = inf every domino is one cluster, the densest packing of
    small components a block of the lattice can hold; shifted tilings put half of every border domino in the next
    block / tile, i.e. as many single-site components with a link out of the block as possible."""
    y, x = np.mgrid[0:L, 0:L]
    if vertical:
        a, b = x, ((y - dy) % L) // 2
    else:
        a, b = ((x - dx) % L) // 2, y
    h = (a.astype(np.uint64) * 0x9E3779B1 + b.astype(np.uint64) * 0x85EBCA77 + 12345) % 0xFFFFFFFB
    return (h % q).astype(np.uint8)


def bonds_random(L: int, density: float, seed: int) -> np.ndarray:
    """Random bond mask, bit0 = right bond of the site, bit1 = its down bond (for labeling tests)."""
    rng = np.random.default_rng(seed)
    r = rng.random((L, L)) < density
    d = rng.random((L, L)) < density
    return (r.astype(np.uint8) | (d.astype(np.uint8) << 1))


def crafted_lattices(L: int, q: int, seed: int = 7):
    """Name -> spins, the adversarial set used by the labeling parity tests."""
    out = {
        "uniform_random": spins_uniform_random(L, q, seed),
        "all_equal": np.zeros((L, L), dtype=np.uint8),
        "checkerboard": spins_checkerboard(L, q),
        "stripes_v1": spins_stripes(L, q, 1, True),
        "stripes_h3": spins_stripes(L, q, 3, False),
        "spiral": spins_spiral(L) % q,
        "comb": spins_comb(L),
        "blocks5": spins_blocks(L, q, 5, seed),
        "blocks37": spins_blocks(L, q, 37, seed + 1),
    }
    return out
