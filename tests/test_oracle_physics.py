"""Statistical pins of the whole oracle chain against exact results (CPU only).

Swendsen-Wang satisfies detailed balance for the Boltzmann weight exp(K * n_eq) (H = -J sum delta,
north_star; the paper's eq. (1), differs by a constant), so long oracle runs must
reproduce exact finite-lattice averages.  Every exact value is recomputed here (brute force, the
Kaufman formula, the 2^18-configuration random-cluster enumeration) and cross-checked against the
survey's independently computed numbers in tests/golden/exact_small.txt.  Statistical tolerance:
4 standard errors from a binning analysis, fixed seeds (north_star: "to a stated number of
standard errors").
"""
import math

import mpmath
import numpy as np
import pytest

from oracle import binding as orc
from oracle.binding import Oracle
from paper_1208_2080_b200 import workloads as wl

N_SE = 4.0


def binned_se(x, nbins=40):
    x = np.asarray(x, dtype=np.float64)
    n = (len(x) // nbins) * nbins
    means = x[:n].reshape(nbins, -1).mean(axis=1)
    return float(means.std(ddof=1) / math.sqrt(nbins))


def golden_rows(golden, kind):
    return [r.split()[1:] for r in golden("exact_small.txt") if r.split()[0] == kind]


# ---------------------------------------------------------------- brute-force Boltzmann averages

def boltzmann_exact(q, L, K, chunk=1 << 20):
    """<n_eq>, var(n_eq), <n_max> by enumerating all q^(N-1) states with spin 0 fixed (S_q symmetry)."""
    N = L * L
    idx = np.arange(N).reshape(L, L)
    right = np.roll(idx, -1, axis=1).reshape(-1)
    down = np.roll(idx, -1, axis=0).reshape(-1)
    total = q ** (N - 1)
    hist = {}
    for start in range(0, total, chunk):
        codes = np.arange(start, min(total, start + chunk), dtype=np.int64)
        s = np.empty((codes.size, N), dtype=np.int8)
        s[:, 0] = 0
        c = codes.copy()
        for k in range(1, N):
            s[:, k] = c % q
            c //= q
        n_eq = (s == s[:, right]).sum(axis=1) + (s == s[:, down]).sum(axis=1)
        n_max = np.max([(s == a).sum(axis=1) for a in range(q)], axis=0)
        key = n_eq * 64 + n_max
        vals, cnt = np.unique(key, return_counts=True)
        for v, m in zip(vals.tolist(), cnt.tolist()):
            hist[v] = hist.get(v, 0) + m
    mp = mpmath.mp
    mp.dps = 40
    Z = mp.mpf(0); e1 = mp.mpf(0); e2 = mp.mpf(0); m1 = mp.mpf(0)
    for v, m in hist.items():
        ne, nm = divmod(v, 64)
        w = m * mp.exp(mp.mpf(K) * ne)
        Z += w; e1 += w * ne; e2 += w * ne * ne; m1 += w * nm
    e1 /= Z; e2 /= Z; m1 /= Z
    return float(e1), float(e2 - e1 * e1), float(m1)


@pytest.mark.parametrize("q,L", [(2, 3), (3, 3), (2, 4)])
def test_brute_force_matches_survey_values(golden, q, L):
    rows = [r for r in golden_rows(golden, "boltzmann") if int(r[0]) == q and int(r[1]) == L]
    assert rows
    for r in rows:
        K = float(r[2])
        e, var, nmax = boltzmann_exact(q, L, K)
        assert abs(e - float(r[3])) < 1e-9 and abs(var - float(r[4])) < 1e-8 and abs(nmax - float(r[5])) < 1e-9


@pytest.mark.parametrize("q,L,K,seed", [
    (2, 3, wl.k_critical(2), 1), (2, 3, 0.5, 2), (3, 3, wl.k_critical(3), 3), (3, 3, 0.5, 1),
    (2, 4, wl.k_critical(2), 2), (2, 4, 0.5, 3), (3, 4, wl.k_critical(3), 1),
])
def test_long_runs_reproduce_boltzmann_averages(q, L, K, seed):
    e_exact, var_exact, nmax_exact = boltzmann_exact(q, L, K)
    sim = Oracle(L, q, K, seed)
    sim.init("random")
    sim.sweep(1000)
    series = sim.sweep_measure(400000).astype(np.float64)
    e = series[:, 0]
    nmax = series[:, 3:].max(axis=1)
    assert abs(e.mean() - e_exact) < N_SE * binned_se(e)
    assert abs(nmax.mean() - nmax_exact) < N_SE * binned_se(nmax)
    v = (e - e.mean()) ** 2
    assert abs(v.mean() - var_exact) < N_SE * binned_se(v) + 1e-3
    if q == 2:                                            # <|M|> = <|n_0 - n_1|> = 2<n_max> - N
        absm = np.abs(series[:, 3] - series[:, 4])
        assert abs(absm.mean() - (2 * nmax_exact - L * L)) < N_SE * binned_se(absm)


# ---------------------------------------------------------------- Kaufman's exact torus result, q = 2

def kaufman_mean_n_eq(L, K):
    """<energy_bonds> of the q=2 Potts model (= Ising at K_I = K/2) on the LxL torus, Kaufman 1949."""
    mp = mpmath.mp
    mp.dps = 60

    def lnZ(KI):
        def gamma(l):
            if l == 0:
                return 2 * KI + mp.log(mp.tanh(KI))
            return mp.acosh(mp.cosh(2 * KI) ** 2 / mp.sinh(2 * KI) - mp.cos(mp.pi * l / L))
        odd = [gamma(2 * r + 1) for r in range(L)]
        even = [gamma(2 * r) for r in range(L)]
        prod = lambda f, g: mp.fprod([2 * f(L * x / 2) for x in g])
        s = prod(mp.cosh, odd) + prod(mp.sinh, odd) + prod(mp.cosh, even) + prod(mp.sinh, even)
        return mp.log(s / 2) + (L * L / mp.mpf(2)) * mp.log(2 * mp.sinh(2 * KI))
    KI = mp.mpf(K) / 2
    dlnZ = mp.diff(lnZ, KI)
    # Z_Ising = sum exp(K_I sum sigma sigma'), sum sigma sigma' = 2 n_eq - 2N  ->  <n_eq> = N + dlnZ/dK_I / 2
    return float(L * L + dlnZ / 2)


def test_kaufman_formula_against_brute_force_and_survey(golden):
    K = wl.k_critical(2)
    assert abs(kaufman_mean_n_eq(3, K) - boltzmann_exact(2, 3, K)[0]) < 1e-9
    assert abs(kaufman_mean_n_eq(4, 0.5) - boltzmann_exact(2, 4, 0.5)[0]) < 1e-9
    for r in golden_rows(golden, "kaufman"):
        L = int(r[0])
        if L <= 64:
            assert abs(kaufman_mean_n_eq(L, K) / float(r[1]) - 1) < 1e-12


@pytest.mark.parametrize("L,sweeps,seed", [(16, 60000, 1), (32, 20000, 2)])
def test_critical_ising_energy_matches_kaufman(L, sweeps, seed):
    K = wl.k_critical(2)
    sim = Oracle(L, 2, K, seed)
    sim.init("ordered")
    sim.sweep(500)
    e = sim.sweep_measure(sweeps)[:, 0].astype(np.float64)
    assert abs(e.mean() - kaufman_mean_n_eq(L, K)) < N_SE * binned_se(e)


def test_critical_energy_per_site_q2_within_half_percent():
    # north_star: e_c = 1 + 1/sqrt(q) per site for large L, to within 0.5 %.  At q=2 the exact finite-size
    # excess is +0.182/L (Kaufman), 0.14 % at L=128.
    L, q = 128, 2
    sim = Oracle(L, q, wl.k_critical(q), 1)
    sim.init("ordered")
    sim.sweep(150)
    e = sim.sweep_measure(1200)[:, 0].astype(np.float64) / (L * L)
    assert abs(e.mean() / (1 + 1 / math.sqrt(q)) - 1) < 0.005
    # and the active-bond density at K_c is p_c * e -> exactly 1 per site (self-duality)
    assert abs(e.mean() * math.sqrt(q) / (1 + math.sqrt(q)) - 1) < 0.005


def test_critical_energy_per_site_q3_within_half_percent():
    L, q = 160, 3
    sim = Oracle(L, q, wl.k_critical(q), 2)
    sim.init("ordered")
    sim.sweep(200)
    e = sim.sweep_measure(800)[:, 0].astype(np.float64) / (L * L)
    assert abs(e.mean() / (1 + 1 / math.sqrt(q)) - 1) < 0.005


# ---------------------------------------------------------------- random-cluster (FK) side

def fk_exact_3x3(q, K):
    """Exact FK averages on the 3x3 torus: all 2^18 bond configurations, weight p^b (1-p)^(18-b) q^C."""
    L, N, B = 3, 9, 18
    idx = np.arange(N).reshape(L, L)
    ends = [(int(i), int(j)) for i, j in zip(idx.reshape(-1), np.roll(idx, -1, axis=1).reshape(-1))]
    ends += [(int(i), int(j)) for i, j in zip(idx.reshape(-1), np.roll(idx, -1, axis=0).reshape(-1))]
    conf = np.arange(1 << B, dtype=np.int64)
    active = ((conf[:, None] >> np.arange(B)[None, :]) & 1).astype(bool)          # (2^18, 18)
    lab = np.tile(np.arange(N, dtype=np.int8), (conf.size, 1))
    for _ in range(N):                                                             # min-propagation to a fixed point
        for b, (i, j) in enumerate(ends):
            m = np.minimum(lab[:, i], lab[:, j])
            a = active[:, b]
            lab[a, i] = m[a]
            lab[a, j] = m[a]
    for _ in range(4):                                                             # flatten chains
        lab = np.take_along_axis(lab, lab.astype(np.int64), axis=1)
    onehot = (lab[:, :, None] == np.arange(N)[None, None, :])
    sizes = onehot.sum(axis=1)                                                     # (2^18, 9)
    ncl = (sizes > 0).sum(axis=1)
    largest = sizes.max(axis=1)
    sumsq = (sizes.astype(np.int64) ** 2).sum(axis=1)
    nb = active.sum(axis=1)
    p = -math.expm1(-K)
    w = p ** nb * (1 - p) ** (B - nb) * float(q) ** ncl
    w /= w.sum()
    return float((w * ncl).sum()), float((w * largest).sum()), float((w * sumsq).sum()), float((w * nb).sum())


@pytest.fixture(scope="module")
def fk_cache():
    return {}


@pytest.mark.parametrize("q,K,seed", [(2, wl.k_critical(2), 1), (2, 0.5, 2), (3, wl.k_critical(3), 3), (3, 0.5, 1)])
def test_cluster_statistics_match_fk_enumeration(golden, q, K, seed):
    ncl, largest, sumsq, nact = fk_exact_3x3(q, K)
    row = [r for r in golden_rows(golden, "fk") if int(r[0]) == q and abs(float(r[1]) - K) < 1e-12][0]
    for got, want in zip((ncl, largest, sumsq, nact), row[2:6]):
        assert abs(got - float(want)) < 1e-8
    L, N = 3, 9
    sim = Oracle(L, q, K, seed)
    sim.init("random")
    sim.sweep(500)
    n = 120000
    s_ncl = np.empty(n); s_big = np.empty(n); s_sq = np.empty(n); s_act = np.empty(n); s_ns2 = np.empty(n)
    for k in range(n):
        sim.sweep(1)
        m = sim.measure()
        s_ncl[k] = m["n_clusters"]; s_big[k] = m["largest_cluster"]
        s_sq[k] = float((np.bincount(sim.get_labels(), minlength=N).astype(np.int64) ** 2).sum())
        b = sim.get_bonds()
        s_act[k] = np.count_nonzero(b & 1) + np.count_nonzero(b & 2)
        s_ns2[k] = float(sum(v * v for v in m["mag_counts"]))
    assert abs(s_ncl.mean() - ncl) < N_SE * binned_se(s_ncl)
    assert abs(s_big.mean() - largest) < N_SE * binned_se(s_big)
    assert abs(s_sq.mean() - sumsq) < N_SE * binned_se(s_sq)
    assert abs(s_act.mean() - nact) < N_SE * binned_se(s_act)
    # improved-estimator identity: q <sum_s n_s^2> - N^2 = (q-1) <sum_clusters |c|^2>
    assert abs(s_ns2.mean() - (N * N + (q - 1) * sumsq) / q) < N_SE * binned_se(s_ns2)


def test_critical_bond_percolation_cluster_density():
    # ordered start, p = 1/2 (K = ln 2): the first sweep's bonds are critical bond percolation.
    # clusters per site = (3*sqrt(3) - 5)/2 (Temperley-Lieb) + 0.8835/N on the torus (Ziff-Finch-Adamchik)
    L = 256
    N = L * L
    vals = []
    for seed in range(1, 25):
        sim = Oracle(L, 2, math.log(2.0), seed)
        sim.init("ordered")
        sim.sweep(1)
        vals.append(sim.measure()["n_clusters"] / N)
    vals = np.array(vals)
    want = (3 * math.sqrt(3) - 5) / 2 + 0.8835 / N
    se = vals.std(ddof=1) / math.sqrt(len(vals))
    assert abs(vals.mean() - want) < N_SE * se
    assert se < 0.001                                          # per-sample sd ~ 0.4/L


def test_bond_count_statistics_from_an_ordered_start():
    # all spins equal: each of the 2N bonds is active independently with probability p
    L = 200
    N = L * L
    for K in (0.2, wl.k_critical(2), 2.5):
        p = -math.expm1(-K)
        counts = []
        for seed in range(1, 9):
            sim = Oracle(L, 2, K, seed)
            sim.init("ordered")
            sim.sweep(1)
            b = sim.get_bonds()
            counts.append((np.count_nonzero(b & 1), np.count_nonzero(b & 2)))
        counts = np.array(counts, dtype=np.float64)
        sd = math.sqrt(N * p * (1 - p))
        # right and down separately, each Binomial(N, p), 8 samples
        assert np.all(np.abs(counts.mean(axis=0) - N * p) < N_SE * sd / math.sqrt(8))
        assert np.all(np.abs(counts - N * p) < 5 * sd)
