"""Physics check of the CUDA path itself (the paper's own correctness check):
PAPER.md:90 -- the authors "checked our code by plotting the temperature dependence of the moment ratio of
magnetization".  At the critical coupling of the 2D Ising model on a periodic square lattice the ratio
<m^2>^2 / <m^4> tends to the universal value 0.856216 (Kamieniarz and Bloete, J. Phys. A 26 (1993) 201), i.e.
<m^4> / <m^2>^2 = 1.16792; away from K_c it moves to 1 (ordered) or 3 (disordered)."""
import math

import numpy as np
import pytest

from paper_1208_2080_b200 import workloads as wl
from paper_1208_2080_b200.binding import SwendsenWang

pytestmark = pytest.mark.gpu

Q_UNIVERSAL = 0.856216


def moment_ratio(L, K, sweeps, warm, seed):
    g = SwendsenWang(L, 2, K, seed)
    g.init("random")
    g.sweep(warm)
    rows = g.sweep_measure(sweeps)
    g.close()
    mag = rows[:, 3:5].astype(np.float64)                      # row layout: energy, n_clusters, largest, mag_counts[q]
    assert np.all(mag.sum(axis=1) == L * L)
    m = (mag[:, 0] - mag[:, 1]) / (L * L)
    m2, m4 = np.mean(m ** 2), np.mean(m ** 4)
    # binned error of the ratio (bins of 500 sweeps >> the SW autocorrelation time of a few sweeps)
    nb = sweeps // 500
    r_bins = [np.mean(b ** 4) / np.mean(b ** 2) ** 2 for b in np.array_split(m, nb)]
    return m4 / m2 ** 2, np.std(r_bins, ddof=1) / math.sqrt(nb)


@pytest.mark.parametrize("L", [64, 128])
def test_moment_ratio_at_criticality(L):
    r, err = moment_ratio(L, wl.k_critical(2), sweeps=20000, warm=500, seed=11)
    assert err < 0.01
    assert abs(r - 1.0 / Q_UNIVERSAL) < max(5 * err, 0.012), (r, err)


def test_moment_ratio_orders_with_temperature():
    # the curves of Fig. 4 of the paper's Ref. [10]: monotone in K, towards 3 (Gaussian) when disordered, 1 when ordered
    kc = wl.k_critical(2)
    r_hot, _ = moment_ratio(64, 0.8 * kc, sweeps=4000, warm=300, seed=5)
    r_crit, _ = moment_ratio(64, kc, sweeps=4000, warm=300, seed=5)
    r_cold, _ = moment_ratio(64, 1.2 * kc, sweeps=4000, warm=300, seed=5)
    assert 2.5 < r_hot < 3.3 and 1.0 <= r_cold < 1.01 and r_cold < r_crit < r_hot
