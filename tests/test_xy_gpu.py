"""Parity of the CUDA embedded-cluster XY path (sw_xy_*) against the XY oracle
-- needs a B200, `-m gpu`.

Bonds and canonical labels are integer results: bit-exact.  The bond decision is taken in IEEE double on both sides
(threshold floor((1 - exp(-2 K a_i a_j)) 2^32), X3-X4) and the spins are updated with the same correctly
rounded operations, so the spins must agree bit for bit too (np.array_equal on the doubles), sweep after sweep.  Sums
(energy, magnetisation) are accumulated in a different order: relative tolerance 1e-12 of the number of terms.
"""
import math

import numpy as np
import pytest

from oracle.xy_binding import OracleXY
from paper_1208_2080_b200 import binding as sw
from paper_1208_2080_b200.binding import XYModel

pytestmark = pytest.mark.gpu


def compare(gpu, cpu, what):
    assert np.array_equal(gpu.get_bonds(), cpu.get_bonds()), f"bonds {what}"
    assert np.array_equal(gpu.get_labels(), cpu.get_labels()), f"labels {what}"
    gs, cs = gpu.get_spins(), cpu.get_spins()
    if not np.array_equal(gs, cs):
        bad = np.flatnonzero((gs != cs).any(axis=1))
        raise AssertionError(f"spins {what}: {bad.size} sites differ, first {bad[:4]}: max |diff| {np.abs(gs - cs).max():.3e}")
    mg, mc = gpu.measure(), cpu.measure()
    n = gpu.N
    assert abs(mg["energy_sum"] - mc["energy_sum"]) <= 1e-12 * 2 * n, what
    assert np.allclose(mg["mag"], mc["mag"], rtol=0, atol=1e-12 * n), what
    assert (mg["n_clusters"], mg["largest_cluster"]) == (mc["n_clusters"], mc["largest_cluster"]), what


@pytest.mark.parametrize("L", [2, 3, 5, 16, 33, 64, 100, 256])
@pytest.mark.parametrize("K", [0.0, 0.5, 1.12, 3.0, math.inf])
def test_xy_sweeps_match_the_oracle_bit_for_bit(L, K):
    gpu, cpu = XYModel(L, K, 7), OracleXY(L, K, 7)
    gpu.init("random"); cpu.init("random")
    assert np.array_equal(gpu.get_spins(), cpu.get_spins()), "initial spins"
    for k in range(5):
        gpu.sweep(1); cpu.sweep(1)
        assert gpu.get_time() == cpu.get_time()
        compare(gpu, cpu, f"(L={L} K={K} sweep {k})")
    r = gpu.get_reflection()
    assert abs(math.hypot(*r) - 1.0) < 1e-15


def test_xy_long_run_ordered_start_and_state_changes():
    L, K = 128, 1.1199                                          # close to the Kosterlitz-Thouless point K ~ 1.12
    gpu, cpu = XYModel(L, K, 3), OracleXY(L, K, 3)
    gpu.init("ordered"); cpu.init("ordered")
    gpu.sweep(40); cpu.sweep(40)                                # 40 sweeps without looking: no drift between the two
    compare(gpu, cpu, "(40 sweeps in one call)")
    norms = np.hypot(*gpu.get_spins().T)
    assert np.all(np.abs(norms - 1.0) < 1e-13)
    rng = np.random.default_rng(5)
    th = rng.uniform(0, 2 * math.pi, L * L)
    spins = np.stack([np.cos(th), np.sin(th)], axis=1)
    gpu.set_state(spins, 0xFFFFFFF0); cpu.set_state(spins, 0xFFFFFFF0)
    gpu.sweep(3); cpu.sweep(3)
    compare(gpu, cpu, "(after set_state, late sweep counter)")
    gpu.init("random"); cpu.init("random")
    gpu.sweep(2); cpu.sweep(2)
    compare(gpu, cpu, "(after init)")


def test_xy_state_machine_and_errors():
    g = XYModel(16, 1.0, 1)
    with pytest.raises(sw.SwError) as e:
        g.sweep(1)
    assert e.value.code == sw.ERR_STATE
    g.init("ordered")
    with pytest.raises(sw.SwError):
        g.get_labels()
    bad = np.zeros((256, 2)); bad[3, 1] = np.nan
    with pytest.raises(sw.SwError) as e:
        g.set_state(bad, 0)
    assert e.value.code == sw.ERR_INVALID_ARG
    for L, K in ((1, 1.0), (8, -1.0), (8, float("nan"))):
        with pytest.raises(sw.SwError):
            XYModel(L, K, 1)
    m = g.measure()
    assert m["n_clusters"] == 0 and abs(m["energy_sum"] - 2 * 256) < 1e-9 and np.allclose(m["mag"], [256.0, 0.0])


def test_xy_physics_low_temperature_order_and_high_temperature_disorder():
    # |M|/N: close to 1 deep in the quasi-ordered phase, ~ N^-1/2 at high temperature (GPU chain on its own)
    L = 64
    res = {}
    for K in (0.3, 2.0):
        g = XYModel(L, K, 11)
        g.init("random")
        g.sweep(300)
        ms, es = [], []
        for _ in range(300):
            g.sweep(2)
            m = g.measure()
            ms.append(math.hypot(*m["mag"]) / (L * L)); es.append(m["energy_sum"] / (2 * L * L))
        res[K] = (np.mean(ms), np.mean(es))
    assert res[0.3][0] < 0.08 and abs(res[0.3][1] - 0.15) < 0.03          # <cos> ~ K/2 at small K
    assert res[2.0][0] > 0.8 and abs(res[2.0][1] - (1 - 1 / 8.0)) < 0.03   # spin waves: 1 - 1/(4K)
