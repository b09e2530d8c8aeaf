"""The super-lattice decomposition against the SAME single-address-space
oracle -- needs a B200, `-m gpu`.

gx x gy sub-lattices, each with its own arrays, stage-1 labeling inside the pieces, stage-2 union over the boundary
sites, resolve, flatten + flip: bonds, canonical labels (global site indices), spins and observables must equal the
oracle's bit for bit, for every decomposition.  All pieces live on one device here (one B200 per box); the kernels
reach their neighbours through the same pointers they would use over NVLink.
"""
import math

import numpy as np
import pytest

from oracle.binding import Oracle
from paper_1208_2080_b200 import binding as sw
from paper_1208_2080_b200 import workloads as wl
from paper_1208_2080_b200.binding import SuperLattice, SwendsenWang

pytestmark = pytest.mark.gpu


def compare(gpu, cpu, what):
    assert np.array_equal(gpu.get_bonds(), cpu.get_bonds()), f"bonds {what}"
    gl, cl = gpu.get_labels(), cpu.get_labels()
    if not np.array_equal(gl, cl):
        bad = np.flatnonzero(gl != cl)
        raise AssertionError(f"labels {what}: {bad.size} sites differ, first {bad[:6]}: gpu {gl[bad[:6]]} oracle {cl[bad[:6]]}")
    assert np.array_equal(gpu.get_spins(), cpu.get_spins()), f"spins {what}"
    assert gpu.measure() == cpu.measure(), f"observables {what}"


GRIDS = [(2, 2), (1, 4), (4, 1), (2, 1), (1, 1), (4, 2)]


@pytest.mark.parametrize("gx,gy", GRIDS)
@pytest.mark.parametrize("L,q", [(512, 2), (1024, 3)])
def test_super_lattice_matches_the_oracle_at_criticality(gx, gy, L, q):
    K = wl.k_critical(q)
    gpu, cpu = SuperLattice(L, q, K, 1, gx, gy), Oracle(L, q, K, 1)
    gpu.init("random"); cpu.init("random")
    assert np.array_equal(gpu.get_spins(), cpu.get_spins())
    m0 = gpu.measure()
    assert m0 == cpu.measure() and m0["n_clusters"] == 0
    for k in range(4):
        gpu.sweep(1); cpu.sweep(1)
        compare(gpu, cpu, f"(L={L} q={q} {gx}x{gy} sweep {k})")
    gpu.sweep(3); cpu.sweep(3)                                  # several sweeps per call
    compare(gpu, cpu, f"(L={L} q={q} {gx}x{gy} after 3 more)")
    st = gpu.stats()
    assert (st["gx"], st["gy"], st["piece_w"], st["piece_h"]) == (gx, gy, L // gx, L // gy)
    assert st["boundary_sites_per_piece"] == 2 * (L // gx + L // gy) and st["inter_links"] > 0 and st["sweeps"] == 7


@pytest.mark.parametrize("gx,gy", [(2, 2), (1, 4), (4, 4)])
def test_ordered_start_one_giant_cluster_across_all_pieces(gx, gy):
    # K = inf from an ordered start: ONE cluster whose root (site 0) lives in piece 0; every other piece learns it through stage 2
    L = 512
    for K in (math.inf, wl.k_critical(2), 0.0):
        gpu, cpu = SuperLattice(L, 2, K, 3, gx, gy), Oracle(L, 2, K, 3)
        gpu.init("ordered"); cpu.init("ordered")
        for k in range(3):
            gpu.sweep(1); cpu.sweep(1)
            compare(gpu, cpu, f"(ordered K={K} {gx}x{gy} sweep {k})")


@pytest.mark.parametrize("gx,gy", [(2, 2), (4, 1), (1, 2)])
def test_adversarial_lattices_across_piece_borders(gx, gy):
    # spirals, combs, stripes, blocks: clusters that cross the piece borders many times (K = inf: clusters = equal-spin regions)
    L = 256
    for name, spins in wl.crafted_lattices(L, 3).items():
        for K in (math.inf, 2.0):
            gpu, cpu = SuperLattice(L, 3, K, 1, gx, gy), Oracle(L, 3, K, 1)
            gpu.set_state(spins, 5); cpu.set_state(spins, 5)
            gpu.sweep(1); cpu.sweep(1)
            compare(gpu, cpu, f"({name}, K={K}, {gx}x{gy})")
            gpu.close(); cpu.close()


def test_long_snake_through_every_piece():
    L = 512
    spins = wl.spins_spiral(L)
    gpu, cpu = SuperLattice(L, 2, math.inf, 1, 2, 4), Oracle(L, 2, math.inf, 1)
    gpu.set_state(spins, 0); cpu.set_state(spins, 0)
    gpu.sweep(1); cpu.sweep(1)
    compare(gpu, cpu, "(spiral 512, 2x4)")
    assert gpu.stats()["resolved_links"] > 0


def test_equilibrated_L4096_2x2_and_same_trajectory_as_the_single_lattice():
    # the paper's own per-GPU size is 4096^2; here 4096^2 in all, 2 x 2 pieces of 2048^2, equilibrated
    c = wl.CONFIGS["c2_L4096_q2"]
    one = SwendsenWang(c["L"], c["q"], c["K"], c["seed"])
    sup = SuperLattice(c["L"], c["q"], c["K"], c["seed"], 2, 2)
    one.init("ordered"); sup.init("ordered")
    one.sweep(60); sup.sweep(60)
    assert np.array_equal(one.get_spins(), sup.get_spins())      # the same chain, sweep for sweep
    cpu = Oracle(c["L"], c["q"], c["K"], c["seed"])
    cpu.set_state(sup.get_spins(), sup.get_time())
    sup.sweep(1); cpu.sweep(1)
    compare(sup, cpu, "(L=4096 2x2 equilibrated)")
    m = sup.measure()
    assert m["largest_cluster"] > 0.2 * c["L"] ** 2               # the giant cluster spans all four pieces


def test_non_power_of_two_size_and_state_machine():
    L = 384                                                     # 3 x 2 pieces of 128 x 192
    gpu, cpu = SuperLattice(L, 4, wl.k_critical(4), 7, 3, 2), Oracle(L, 4, wl.k_critical(4), 7)
    with pytest.raises(sw.SwError) as e:
        gpu.sweep(1)
    assert e.value.code == sw.ERR_STATE
    gpu.init("random"); cpu.init("random")
    with pytest.raises(sw.SwError):
        gpu.get_labels()
    gpu.sweep(2); cpu.sweep(2)
    compare(gpu, cpu, "(L=384 3x2)")
    with pytest.raises(sw.SwError) as e:
        gpu.set_state(np.full(L * L, 4, dtype=np.uint8), 0)
    assert e.value.code == sw.ERR_INVALID_ARG
    spins = wl.spins_uniform_random(L, 4, 3)
    gpu.set_state(spins, 0xFFFFFFF0); cpu.set_state(spins, 0xFFFFFFF0)
    gpu.sweep(2); cpu.sweep(2)
    compare(gpu, cpu, "(late sweep counter)")
    for bad in ((3, 3), (0, 1), (9, 9)):
        with pytest.raises(sw.SwError):
            SuperLattice(512, 2, 0.5, 1, *bad)


def test_config4_size_q10_in_2x2_pieces_one_transition():
    # BASELINE config 4 (L = 16384, q = 10, just below K_c) in 2 x 2 pieces of 8192^2: one equilibrated transition against the oracle
    c = wl.CONFIGS["c4_L16384_q10_below"]
    sup = SuperLattice(c["L"], c["q"], c["K"], c["seed"], 2, 2)
    cpu = Oracle(c["L"], c["q"], c["K"], c["seed"])
    sup.init(c["start"])
    sup.sweep(40)
    cpu.set_state(sup.get_spins(), sup.get_time())
    sup.sweep(1); cpu.sweep(1)
    compare(sup, cpu, "(c4 below, 2x2 pieces, t = 40)")


def _n_devices():
    import torch
    return torch.cuda.device_count() if torch.cuda.is_available() else 0


@pytest.mark.parametrize("gx,gy,devices", [(2, 1, [0, 1]), (2, 2, [0, 1, 1, 0]), (1, 2, [1, 0])])
def test_pieces_on_two_devices_peer_path(gx, gy, devices):
    """The path the paper is about: pieces on DIFFERENT GPUs, neighbours' boundary spins read over the
    link, roots hooked with system-scope atomics in the owner's memory.  Needs two devices with peer access and native
    atomics between them (NVLink); skipped on a one-GPU box, so it runs the first time such hardware is there."""
    if _n_devices() < 2:
        pytest.skip("needs two CUDA devices (the peer / NVLink path)")
    L, q = 512, 2
    K = wl.k_critical(q)
    try:
        gpu = SuperLattice(L, q, K, 5, gx, gy, devices=devices)
    except sw.SwError as e:                                   # peer access or native atomics missing: say so, do not fail
        pytest.skip(f"sw_create_super refused these devices: {sw.lib().sw_super_last_error(None).decode()} ({e})")
    cpu = Oracle(L, q, K, 5)
    gpu.init("random"); cpu.init("random")
    assert gpu.stats()["devices"] == 2
    for k in range(4):
        gpu.sweep(1); cpu.sweep(1)
        compare(gpu, cpu, f"({gx}x{gy} on devices {devices}, sweep {k})")
    gpu.sweep(3); cpu.sweep(3)
    compare(gpu, cpu, f"({gx}x{gy} on devices {devices}, after 3 more)")
    assert gpu.stats()["inter_links"] > 0
