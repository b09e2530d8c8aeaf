"""Parity in EQUILIBRATED states at BASELINE.json's sizes -- needs a B200, `-m gpu`.

The first sweeps after a random start only ever see tiny clusters; after an ordered start, one giant cluster.  The
states a long run spends its time in (a critical giant cluster with long hooked chains across thousands of tiles, merge
contention on its root, the coexisting phases of q = 10) are reached here by letting the CUDA path run, and are then
checked one transition at a time: the GPU's spins after sweep t - 1 are handed to the oracle (`swo_set_state`), the
oracle makes ONE sweep, and bonds, canonical labels, spins and all observables of the GPU's sweep t must match bit for
bit.  A sweep is a deterministic function of (spins, t, seed), so exact agreement at sampled t on top of the
whole-trajectory comparisons at small L is the strongest statement the oracle's speed affords; the t checked are in the
test ids.
"""
import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1208_2080_b200 import workloads as wl
from paper_1208_2080_b200.binding import SwendsenWang

pytestmark = pytest.mark.gpu


def transition_check(gpu, cpu, what):
    """One sweep on both sides from the GPU's current state; everything compared."""
    t = gpu.get_time()
    cpu.set_state(gpu.get_spins(), t)
    gpu.sweep(1); cpu.sweep(1)
    assert gpu.get_time() == cpu.get_time() == t + 1
    assert np.array_equal(gpu.get_bonds(), cpu.get_bonds()), f"bonds {what} t={t}"
    gl, cl = gpu.get_labels(), cpu.get_labels()
    if not np.array_equal(gl, cl):
        bad = np.flatnonzero(gl != cl)
        raise AssertionError(f"labels {what} t={t}: {bad.size} sites differ, first {bad[:6]}: gpu {gl[bad[:6]]} oracle {cl[bad[:6]]}")
    assert np.array_equal(gpu.get_spins(), cpu.get_spins()), f"spins {what} t={t}"
    m = gpu.measure()
    assert m == cpu.measure(), f"observables {what} t={t}"
    return m


def test_config2_L4096_ordered_start_first_20_sweeps_and_equilibrium():
    # config 2: one giant cluster at t = 0 (worst-case merge contention), relaxing towards criticality
    c = wl.CONFIGS["c2_L4096_q2"]
    gpu = SwendsenWang(c["L"], c["q"], c["K"], c["seed"])
    cpu = Oracle(c["L"], c["q"], c["K"], c["seed"])
    gpu.init(c["start"]); cpu.init(c["start"])
    for k in range(20):                                       # the whole trajectory, every sweep
        gpu.sweep(1); cpu.sweep(1)
        assert np.array_equal(gpu.get_bonds(), cpu.get_bonds()), f"bonds sweep {k}"
        assert np.array_equal(gpu.get_labels(), cpu.get_labels()), f"labels sweep {k}"
        assert np.array_equal(gpu.get_spins(), cpu.get_spins()), f"spins sweep {k}"
        assert gpu.measure() == cpu.measure(), f"observables sweep {k}"
    gpu.sweep(80)                                             # t = 100: equilibrated
    m = transition_check(gpu, cpu, "c2 equilibrated")
    N = c["L"] ** 2
    assert 0.2 * N < m["largest_cluster"] < 0.6 * N           # a critical giant cluster is what this state is about
    gpu.sweep(37)
    transition_check(gpu, cpu, "c2 equilibrated, later")


@pytest.mark.parametrize("name,late", [("c3_L8192_q3", 80), ("c3_L8192_q4", 80), ("c4_L16384_q10_above", 70), ("c4_L16384_q10_below", 70)])
def test_configs_3_and_4_early_and_equilibrated_transitions(name, late):
    c = wl.CONFIGS[name]
    gpu = SwendsenWang(c["L"], c["q"], c["K"], c["seed"])
    cpu = Oracle(c["L"], c["q"], c["K"], c["seed"])
    gpu.init(c["start"])
    gpu.sweep(1)
    transition_check(gpu, cpu, f"{name} early")               # t = 1
    gpu.sweep(late - gpu.get_time())
    transition_check(gpu, cpu, f"{name} late")                # t = late
