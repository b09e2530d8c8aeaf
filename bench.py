#!/usr/bin/env python
"""bench.py -- spin flips per nanosecond of the Swendsen-Wang sweep on B200 (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload NAME] [--impl reference]

A step is ONE full sweep (bond activation, tile-local labeling, border merge, flatten to canonical
labels, flip: SURVEY.md sec. 8(a) rows a1-a5) of the headline workload of BASELINE.json: q = 2 Potts at
K_c on the 65536 x 65536 periodic lattice (2^32 sites), random start, Philox seed 1.  W untimed sweeps,
then exactly K sweeps timed with CUDA events on the stream the kernels run on.  The 23.5 GiB working
set is far larger than the 126 MB L2, so no L2 flush is needed between sweeps.  The per-kernel split and
the per-sweep time series come from a SECOND pass of K sweeps (events around every kernel), outside the
headline region.

N > 1: the path does not shard without collectives ("replicas only"), so every
rank runs an independent replica (seed 1 + rank) and the value is the aggregate of all replicas
over the slowest rank's time.  `--gpus N` without a torchrun environment starts the N ranks itself
(re-exec under `python -m torch.distributed.run`); under torchrun WORLD_SIZE must equal N.

--impl reference times the CPU oracle (oracle/, plain single-threaded C++) on the host cores on a
bounded sample of the same workload; it is a deliberately slow reference program, not a target.
"""
from __future__ import annotations

import argparse
import json
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_1208_2080_b200 import workloads as wl  # noqa: E402

METRIC = "spin_flips_per_ns"
UNIT = "flips/ns"
PAPER_FLIPS_PER_NS = 37.30        # PAPER.md:103 (Table 1): L = 65536, q = 2, T_c, 256 x Tesla M2050
HBM_FALLBACK_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md, used only if MEASURED_PEAKS.json is absent

# Algorithmic bytes per site per launch: what the METHOD must move.
ALGORITHMIC_BYTES_PER_SITE = {
    "k_tile_blocks": 1.0 + 0.25 + 4.0,          # a1 + a2: spins R, bond bits W, labels W
    "k_tile_merge": 24.0 / 64.0,                # a3: 2/T_tile border bonds per site x (two 4-byte finds + one 4-byte atomic), T_tile = 64
    "k_tile_flip": 4.0 + 4.0 + 1.0,             # a4 + a5: labels R, canonical labels W, spins W
}
# What THIS design moves on top of that (its own auxiliary arrays), reported separately.
OVERHEAD_BYTES_PER_SITE = {
    "k_tile_blocks": 0.25 + 0.125 + (16.0 + 1024.0) / 4096.0,   # draw masks R, root bitmap W, border + edge records W
    "k_tile_merge": (16.0 + 1024.0) / 4096.0 - 24.0 / 64.0 + 1.25,   # records R instead of label reads, + 64-byte DRAM bursts per root link (measured)
    "k_tile_flip": 0.125 + 0.25,                # root bitmap R, next sweep's draw masks W
}
LAZY_SAVES = 4.0                                # SW_FLAG_LAZY_LABELS: no canonical-label write in k_tile_flip

# Integer-ALU view of the whole sweep: algorithmic lane-operations per site = 0.5 Philox4x32-10 bond
# calls x (20 32x32->64 multiplies + 20 three-input XORs) + 2 threshold tests + 2 spin compares, + one Philox call (40)
# per cluster; peak = SMs x 128 int32 lanes x SM clock.
ALU_OPS_PER_SITE_BONDS = 0.5 * 40 + 2 + 2
ALU_OPS_PER_CLUSTER = 40
B200_SMS, B200_LANES_PER_SM = 148, 128

# the other BASELINE.json configs, measured in the same run: (name, warm-up sweeps, timed sweeps, observables the config
# asks for every sweep -- None = update only, start -- None = the config's own).  Warm-up + timed = the config's own
# number of sweeps: the timed half is the second half of the run the config describes, and the record carries the ratio
# of the first to the second half of its per-sweep series (1.00 = flat, i.e. no transient left in the number).
# q = 4 starts ordered: from a random start it is still 3 % off after 100 sweeps at L = 1024.
OTHER_CONFIGS = [
    ("c1_L256_q2", 100, 100, "all", None),
    ("c2_L4096_q2", 500, 500, None, None),
    ("c3_L8192_q3", 250, 250, "energy+mag", None),
    ("c3_L8192_q4", 250, 250, "energy+mag", "ordered"),
    ("c4_L16384_q10_above", 100, 100, "clusters+largest", None),
    ("c4_L16384_q10_below", 100, 100, "clusters+largest", None),
]


def rank_info():
    return int(os.environ.get("RANK", 0)), int(os.environ.get("LOCAL_RANK", 0)), int(os.environ.get("WORLD_SIZE", 1))


def free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


class ClockSampler:
    """Samples nvidia-smi clocks and throttle reasons while the timed region runs."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc, self.thread = index, [], None, None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits", "-lms", "100", "-i", str(self.index)],
                stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None
            return
        self.thread = threading.Thread(target=self._read, daemon=True)
        self.thread.start()

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smax, reasons, power = [], [], set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (ts, r) in self.rows if t0 - 0.05 <= ts <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except (ValueError, IndexError):
                continue
            for name, val in zip(names, f[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


def hbm_peak():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy bandwidth)"
    except Exception:
        return HBM_FALLBACK_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(workload, kernel):
    """DRAM bytes per launch of `kernel` from the committed ncu summary, if one exists for this workload."""
    try:
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.json")) as f:
            return json.load(f).get(workload, {}).get(kernel)
    except Exception:
        return None


def cpu_model():
    try:
        with open("/proc/cpuinfo") as f:
            for line in f:
                if line.startswith("model name"):
                    return line.split(":", 1)[1].strip()
    except OSError:
        pass
    return "unknown"


# ------------------------------------------------------------------------------------------------ reference arm

def run_reference(args):
    """--impl reference: the oracle as it stands, one thread, on a bounded sample of the workload."""
    rank, _, world = rank_info()
    if rank != 0:
        return 0
    c = wl.CONFIGS[args.workload]
    L = min(c["L"], args.reference_L)
    from oracle.binding import Oracle
    sim = Oracle(L, c["q"], c["K"], c["seed"])
    sim.init(c["start"])
    sim.sweep(args.warmup)
    t0 = time.perf_counter()
    sim.sweep(args.steps)
    dt = time.perf_counter() - t0
    value = L * L * args.steps / dt / 1e9
    sample = (f"oracle/libsw_oracle.so, 1 thread, each step = one sweep of an L={L} lattice with the workload's q, K, "
              f"start and seed ({L * L} of the workload's {c['L'] ** 2} sites)")
    print(json.dumps({
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": args.workload, "L": c["L"], "q": c["q"], "K": c["K"], "start": c["start"], "seed": c["seed"],
                   "sample_L": L},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample,
                         "nproc": os.cpu_count(), "cpu_model": cpu_model()},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }))
    return 0


# ------------------------------------------------------------------------------------------------ CPU baseline leg

def time_cpu_baseline(args, equilibrated):
    """The oracle as it stands on this box's host cores, one thread.  `equilibrated` maps a lattice
    size to (spins, t, q, K, seed) taken from the GPU after its warm-up, so the oracle is timed on a steady-state lattice."""
    from oracle.binding import Oracle
    out = {}
    # headline sample: >= 20 sweeps at L = 4096, q = 2, K_c, from an equilibrated state
    spins, t, q, K, seed = equilibrated[4096]
    sim = Oracle(4096, q, K, seed)
    sim.set_state(spins, t)
    t0 = time.perf_counter()
    sim.sweep(args.cpu_baseline_sweeps)
    dt = time.perf_counter() - t0
    sim.close()
    out["L4096"] = {"flips_per_ns": 4096 * 4096 * args.cpu_baseline_sweeps / dt / 1e9, "ns_per_site_sweep": dt * 1e9 / (4096 * 4096 * args.cpu_baseline_sweeps),
                    "sweeps": args.cpu_baseline_sweeps, "seconds": dt}
    # config 1: all 200 sweeps from its own random start
    c1 = wl.CONFIGS["c1_L256_q2"]
    sim = Oracle(c1["L"], c1["q"], c1["K"], c1["seed"])
    sim.init(c1["start"])
    t0 = time.perf_counter()
    sim.sweep(c1["sweeps"])
    dt1 = time.perf_counter() - t0
    sim.close()
    out["c1_L256"] = {"flips_per_ns": c1["L"] ** 2 * c1["sweeps"] / dt1 / 1e9, "ns_per_site_sweep": dt1 * 1e9 / (c1["L"] ** 2 * c1["sweeps"]),
                      "sweeps": c1["sweeps"], "seconds": dt1}
    # one sweep at L = 8192 (q = 3, K_c), equilibrated state
    if 8192 in equilibrated:
        spins, t, q, K, seed = equilibrated[8192]
        sim = Oracle(8192, q, K, seed)
        sim.set_state(spins, t)
        t0 = time.perf_counter()
        sim.sweep(1)
        dt2 = time.perf_counter() - t0
        sim.close()
        out["L8192_q3"] = {"flips_per_ns": 8192 * 8192 / dt2 / 1e9, "ns_per_site_sweep": dt2 * 1e9 / (8192 * 8192), "sweeps": 1, "seconds": dt2}
    total = sum(v["seconds"] for v in out.values())
    return {"value": out["L4096"]["flips_per_ns"], "unit": UNIT, "cores": 1, "kind": "oracle",
            "nproc": os.cpu_count(), "cpu_model": cpu_model(),
            "sample": f"{args.cpu_baseline_sweeps} sweeps of an equilibrated L=4096 lattice (q=2, K_c: the headline physics; state taken from the GPU "
                      f"after its warm-up and loaded with swo_set_state), single thread; also config 1 (L=256, all 200 sweeps) and one sweep "
                      f"at L=8192 (q=3): {total:.1f} s of CPU in all",
            "samples": out}


# ------------------------------------------------------------------------------------------------ GPU arm

def measure_config(name, warm, steps, what, start, torch, SwendsenWang, sw):
    """One of the other BASELINE.json configs: update-only, and with the observables it asks for."""
    c = dict(wl.CONFIGS[name])
    if start:
        c["start"] = start
    L, N = c["L"], c["L"] ** 2
    sim = SwendsenWang(L, c["q"], c["K"], c["seed"])
    sim.init(c["start"])
    sim.sweep(warm)
    sim.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(); sim.sweep(steps); e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1) / steps
    rec = {"L": L, "q": c["q"], "start": c["start"], "warmup": warm, "steps": steps, "config_sweeps": c["sweeps"],
           "flips_per_ns": N / (ms * 1e-3) / 1e9, "ms_per_sweep": ms, "path": sim.stats()["path_name"]}
    if sim.stats()["path"] == 1:                                    # per-sweep series (a second pass, events around every kernel)
        sim.profile_begin(); sim.sweep(steps); sim.profile_end()
        ser = sim.last_series
        if len(ser) >= 4:
            h = len(ser) // 2
            rec["series_first_half_over_second_half"] = (sum(ser[:h]) / h) / (sum(ser[h:]) / (len(ser) - h))
    if what:
        mask = {"all": sw.OBS_ALL, "energy+mag": sw.OBS_ENERGY | sw.OBS_MAG, "clusters+largest": sw.OBS_CLUSTERS | sw.OBS_LARGEST}[what]
        sim.sweep_measure(2, mask)                                  # warm (first call allocates / sizes scratch)
        m_steps = min(steps, 50)
        e0.record(); rows = sim.sweep_measure(m_steps, mask); e1.record()
        torch.cuda.synchronize()
        ms_m = e0.elapsed_time(e1) / m_steps
        rec.update({"observables_every_sweep": what, "flips_per_ns_with_measurement": N / (ms_m * 1e-3) / 1e9,
                    "ms_per_sweep_with_measurement": ms_m, "last_row": [int(v) for v in rows[-1]]})
    sim.close()
    return rec


def run_gpu(args):
    import torch
    import torch.distributed as dist

    from paper_1208_2080_b200 import binding as sw
    from paper_1208_2080_b200 import replicas
    from paper_1208_2080_b200.binding import FLAG_DEFAULT, FLAG_LABEL_EQUIVALENCE, FLAG_LAZY_LABELS, SwendsenWang

    rank, local_rank, world = rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    distributed = world > 1
    if distributed:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    c = dict(wl.CONFIGS[args.workload])
    L, q, K = c["L"], c["q"], c["K"]
    N = L * L
    flags = FLAG_LAZY_LABELS if args.lazy else FLAG_DEFAULT
    if args.label_equivalence:
        flags = FLAG_LABEL_EQUIVALENCE
    sim = SwendsenWang(L, q, K, replicas.replica_seed(c["seed"], rank), flags=flags)
    sim.init(c["start"])
    sim.sweep(args.warmup)
    sim.synchronize()

    def barrier():
        if distributed:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: exactly K sweeps, CUDA events on the stream the kernels are enqueued on; nothing else in it
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    launches0 = sim.stats()["kernel_launches"]
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    wall0 = time.time()
    ev0.record()
    sim.sweep(args.steps)
    ev1.record()
    barrier()
    wall1 = time.time()
    elapsed_ms = ev0.elapsed_time(ev1)
    launches = sim.stats()["kernel_launches"] - launches0
    clocks = sampler.stop(wall0, wall1) if rank == 0 else None
    # replicas only: total units of all ranks over the slowest rank's device time
    total_units, elapsed_s, rate = replicas.aggregate_throughput(N * args.steps, elapsed_ms * 1e-3, device="cuda")
    elapsed_ms = elapsed_s * 1e3
    value = rate / 1e9

    # ---- second pass, outside the headline region: events around every kernel -> per-kernel split and per-sweep series
    sim.profile_begin()
    sim.sweep(args.steps)
    prof = sim.profile_end()
    series = sim.last_series

    # ---- update + measurement (the paper's second column): sweep + all observables each step
    m_steps = max(1, min(args.steps, 10))
    sim.measure(largest=False)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(m_steps):
        sim.sweep(1)
        obs = sim.measure(largest=False)
    e1.record()
    torch.cuda.synchronize()
    value_meas = N * m_steps / (e0.elapsed_time(e1) * 1e-3) / 1e9
    # the same with ALL FOUR outputs of sw_measure (largest_cluster too: a 4 N-byte size counter per site, 16 GiB at
    # L = 65536, allocated by the library on first use), once as sweep + sw_measure per step, once as ONE
    # sw_sweep_measure call (sizes counted inside the tile / flip kernels, no per-site counting pass)
    value_meas_all = value_series_all = None
    if world == 1 and not args.lazy and not args.label_equivalence:
        a_steps = max(1, min(args.steps, 5))
        sim.measure()                                          # (untimed: allocates the size counters)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(a_steps):
            sim.sweep(1)
            obs_all = sim.measure()
        e1.record()
        torch.cuda.synchronize()
        value_meas_all = N * a_steps / (e0.elapsed_time(e1) * 1e-3) / 1e9
        sim.sweep_measure(1)                                   # (untimed: first use of the counting instantiations)
        torch.cuda.synchronize()
        e0.record()
        rows_all = sim.sweep_measure(a_steps)
        e1.record()
        torch.cuda.synchronize()
        value_series_all = N * a_steps / (e0.elapsed_time(e1) * 1e-3) / 1e9
        assert int(rows_all[-1, 2]) >= 1 and int(rows_all[-1, 1]) >= 1

    # ---- end to end through the C ABI with HOST buffers: H2D of the state, one sweep, D2H of the new state, every step.
    # The state crosses PCIe in the library's packed form (sw_set_state_packed / sw_get_spins_packed: 1 bit per spin at
    # q = 2), which is lossless and what a checkpoint would move; the byte-per-spin form is timed beside it.
    bits = next(b for b in (1, 2, 4, 8) if q <= (1 << b))
    e2e_steps = max(1, min(args.steps, args.e2e_steps))
    host = torch.empty(N * bits // 8, dtype=torch.uint8, pin_memory=True)
    sim.get_spins_packed(bits, out=host.data_ptr())
    t_now = sim.get_time()
    sim.set_state_packed(host.data_ptr(), bits, t_now)     # (untimed: one round trip so that every buffer has been touched)
    barrier()
    w0 = time.perf_counter()
    for k in range(e2e_steps):
        sim.set_state_packed(host.data_ptr(), bits, t_now + k)     # H2D + unpack + validation of every value
        sim.sweep(1)
        sim.get_spins_packed(bits, out=host.data_ptr())            # pack + D2H; synchronises
    barrier()
    e2e_s = time.perf_counter() - w0
    e2e_value = replicas.aggregate_throughput(N * e2e_steps, e2e_s, device="cuda")[2] / 1e9
    del host
    e2e_unpacked = None
    if world == 1:
        host = torch.empty(N, dtype=torch.uint8, pin_memory=True)
        sim.get_spins_ptr(host.data_ptr())
        t_now = sim.get_time()
        torch.cuda.synchronize()
        w0 = time.perf_counter()
        for k in range(min(2, e2e_steps)):
            sim.set_state_ptr(host.data_ptr(), t_now + k)
            sim.sweep(1)
            sim.get_spins_ptr(host.data_ptr())
        e2e_unpacked = {"value": N * min(2, e2e_steps) / (time.perf_counter() - w0) / 1e9, "unit": UNIT, "h2d_bytes_per_step": N, "d2h_bytes_per_step": N,
                        "what": "sw_set_state + sw_sweep(1) + sw_get_spins, one byte per spin: PCIe-bound (8 GiB per step at L = 65536)"}
        del host

    stats = sim.stats()
    if rank != 0:
        if distributed:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel: SURVEY.md sec. 8(d) algorithmic bytes over its CUDA-event duration
    peak, peak_src = hbm_peak()
    alg = dict(ALGORITHMIC_BYTES_PER_SITE)
    if args.lazy:
        alg["k_tile_flip"] -= LAZY_SAVES
    kernels = {}
    for name, rec in (prof or {}).items():
        avg_ms = rec["ms"] / rec["launches"]
        b = alg.get(name)
        kernels[name] = {"ms_per_launch": avg_ms, "launches_per_sweep": rec["launches"] / args.steps, "share": None,
                         "algorithmic_bytes_per_site": b, "overhead_bytes_per_site": OVERHEAD_BYTES_PER_SITE.get(name),
                         "achieved_gbs": (b * N / (avg_ms * 1e-3) / 1e9) if b else None}
    tot = sum(k["ms_per_launch"] * k["launches_per_sweep"] for k in kernels.values()) or 1.0
    for k in kernels.values():
        k["share"] = k["ms_per_launch"] * k["launches_per_sweep"] / tot
    roofline = None
    tiled = stats["path"] == 1 and not args.label_equivalence
    if kernels and tiled:
        top = max(kernels, key=lambda n: kernels[n]["ms_per_launch"])
        a = kernels[top]["achieved_gbs"]
        roofline = {"kernel": top, "bound": "hbm", "achieved": a, "peak": peak, "unit": "GB/s",
                    "frac": (a / peak) if a else None, "traffic": ncu_traffic(args.workload, top),
                    "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": alg.get(top, 0) * N,
                    "algorithmic_bytes_per_site": alg.get(top),
                    "overhead_bytes_per_site": OVERHEAD_BYTES_PER_SITE.get(top),
                    "bytes_source": "SURVEY.md sec. 8(d): spins R 1 + bond bits W 0.25 + labels W 4 (a1+a2); labels R 4 + W 4 + spins W 1 (a4+a5); "
                                    "the design's auxiliary arrays are the separate overhead_bytes_per_site",
                    "limited_by": "integer ALU pipe (instruction issue), not HBM: see profiles/README.md"}
    roofline_alu = None
    if kernels and roofline:
        clk = ((clocks or {}).get("sm_mhz") or 1965.0) * 1e6
        ops = ALU_OPS_PER_SITE_BONDS * N + ALU_OPS_PER_CLUSTER * float(obs.get("n_clusters", 0))
        a = ops / (elapsed_ms / args.steps * 1e-3) / 1e12
        pk = B200_SMS * B200_LANES_PER_SM * clk / 1e12
        tr = [ncu_traffic(args.workload, k) for k in kernels]
        roofline_alu = {"kernel": "whole sweep (" + " + ".join(kernels) + ")", "bound": "alu", "achieved": a, "peak": pk,
                        "unit": "Tlane-op/s", "frac": a / pk, "traffic": sum(tr) if all(tr) else None,
                        "algorithmic_ops_per_sweep": ops,
                        "peak_source": "148 SMs x 128 int32 lanes x SM clock under load (B200_PROFILING.md unit counts)"}
    sweep_alg = sum(alg.values())
    sweep_floor_ms = sweep_alg * N / (peak * 1e9) * 1e3
    per_gpu_ms = elapsed_ms / args.steps
    half = series[len(series) // 2:] if series else []
    time_series = {"ms_per_sweep": [round(v, 4) for v in series], "second_half_mean_ms": (sum(half) / len(half)) if half else None,
                   "second_half_flips_per_ns": (N / (sum(half) / len(half) * 1e-3) / 1e9) if half else None,
                   "what": "device time of each sweep of the second (profiled) pass, first kernel start to last kernel end; sweeps "
                           f"{args.warmup + args.steps} .. {args.warmup + 2 * args.steps - 1} since the start"}

    # ---- the other BASELINE.json configs, briefly (each closes its context before the next)
    other = None
    equilibrated = {}
    if world == 1 and args.workload == wl.HEADLINE and not args.no_other_configs:
        sim.close()
        torch.cuda.empty_cache()
        other = {}
        for name, warm, steps, what, start in OTHER_CONFIGS:
            try:
                other[name] = measure_config(name, warm, steps, what, start, torch, SwendsenWang, sw)
            except Exception as e:                                   # a failed side measurement must not lose the headline line
                other[name] = {"error": repr(e)}

    # ---- the super-lattice decomposition on ONE device: 2 x 2 pieces of the ncu-sized lattice, all on
    # this GPU -- what the two-stage labeling (stage 2 over the boundary sites, resolve pass, event-ordered phases) costs next
    # to the single-lattice path on the same sites.  The NVLink path itself cannot be measured on a one-GPU box.
    if other is not None:
        try:
            from paper_1208_2080_b200.binding import SuperLattice
            cs = wl.CONFIGS["p_L16384_q2"]
            sup = SuperLattice(cs["L"], cs["q"], cs["K"], cs["seed"], 2, 2)
            sup.init(cs["start"]); sup.sweep(30); sup.synchronize()
            t0 = time.perf_counter(); sup.sweep(20); sup.synchronize(); dt = time.perf_counter() - t0
            st = sup.stats()
            sup.close()
            one = SwendsenWang(cs["L"], cs["q"], cs["K"], cs["seed"])
            one.init(cs["start"]); one.sweep(30); one.synchronize()
            t0 = time.perf_counter(); one.sweep(20); one.synchronize(); dt1 = time.perf_counter() - t0
            one.close()
            other["super_2x2_L16384_q2_one_device"] = {
                "flips_per_ns": cs["L"] ** 2 * 20 / dt / 1e9, "ms_per_sweep": dt / 20 * 1e3,
                "single_lattice_flips_per_ns": cs["L"] ** 2 * 20 / dt1 / 1e9,
                "inter_piece_links_per_sweep": st["inter_links"] / st["sweeps"], "inter_piece_label_loads_per_sweep": st["inter_hops"] / st["sweeps"],
                "resolved_links_per_sweep": st["resolved_links"] / st["sweeps"], "boundary_sites_per_piece": st["boundary_sites_per_piece"],
                "what": "wall clock around 20 sweeps + synchronize, all four pieces on this GPU; NVLink unmeasured"}
        except Exception as e:
            other["super_2x2_L16384_q2_one_device"] = {"error": repr(e)}

    # ---- the extension the paper names: embedded-cluster sweeps of the XY model.
    # It runs on the any-L generic kernels (global union-find), untuned: the number says where it stands, not what the
    # hardware allows.  Bytes per site per sweep as built: spins R 16 + W 16 (double x, y), labels 4 x 3 passes, bond bits 0.5.
    if other is not None:
        try:
            from paper_1208_2080_b200.binding import XYModel
            for Lxy in (4096, 8192):
                xy = XYModel(Lxy, 1.12, 1)                         # K near the Kosterlitz-Thouless point: clusters of all sizes
                xy.init("random"); xy.sweep(10); xy.measure()
                t0 = time.perf_counter(); xy.sweep(10); m_xy = xy.measure(); dt = time.perf_counter() - t0
                xy.close()
                other[f"xy_L{Lxy}"] = {"flips_per_ns": Lxy * Lxy * 10 / dt / 1e9, "ms_per_sweep": dt / 10 * 1e3, "K": 1.12, "warmup": 10, "steps": 10,
                                       "bytes_per_site_as_built": 44.5, "n_clusters": m_xy["n_clusters"],
                                       "what": "wall clock around sw_xy_sweep(10) + one sw_xy_measure (synchronises); generic kernels, untuned"}
        except Exception as e:
            other["xy"] = {"error": repr(e)}

    # ---- the oracle on this box's host cores (reported baseline, rank 0, N = 1 only), on equilibrated lattices
    cpu_baseline = None
    if world == 1 and not args.no_cpu_baseline:
        for Lc, qc, warm in ((4096, 2, 100), (8192, 3, 60)):
            g = SwendsenWang(Lc, qc, wl.k_critical(qc), 1)
            g.init("random")
            g.sweep(warm)
            equilibrated[Lc] = (g.get_spins(), g.get_time(), qc, wl.k_critical(qc), 1)
            g.close()
        cpu_baseline = time_cpu_baseline(args, equilibrated)

    out = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": per_gpu_ms, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": (value / PAPER_FLIPS_PER_NS) if args.workload == wl.HEADLINE else None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": args.workload, "L": L, "q": q, "K": K, "start": c["start"], "seed": c["seed"],
                   "labels": "label equivalence (comparison variant)" if args.label_equivalence else "lazy" if args.lazy else "canonical every sweep",
                   "parallelism": "replicas only" if world > 1 else "1 GPU",
                   "l2": f"working set {stats['device_bytes'] / 2**30:.1f} GiB >> 126 MB L2, no flush needed" if stats["device_bytes"] > (1 << 30)
                         else "working set fits L2: HBM roofline fractions are not meaningful at this size"},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": N * bits // 8, "d2h_bytes_per_step": N * bits // 8, "steps": e2e_steps,
                "what": f"sw_set_state_packed(host, {bits} bit(s) per spin) + sw_sweep(1) + sw_get_spins_packed(host) per step, pinned host memory; "
                        "input of step k + 1 = output of step k"},
        "e2e_unpacked": e2e_unpacked,
        "gpu_launches": launches,
        "roofline": roofline,
        "roofline_alu": roofline_alu,
        "cpu_baseline": cpu_baseline,
        "kernels": kernels,
        "sweep_model": {"algorithmic_bytes_per_site": sweep_alg, "overhead_bytes_per_site": sum(OVERHEAD_BYTES_PER_SITE.values()) if tiled else None,
                        "floor_ms_at_peak": sweep_floor_ms, "frac_of_min_traffic_roofline": sweep_floor_ms / per_gpu_ms,
                        "what": "SURVEY.md sec. 8(d): 14.5 + 24/T_tile bytes per site per sweep over the measured copy bandwidth"},
        "time_series": time_series,
        "update_plus_measurement": {"value": value_meas, "unit": UNIT, "steps": m_steps,
                                    "what": "sw_sweep(1) + sw_measure(energy, magnetisation, n_clusters) per step: THREE of the four observables",
                                    "all_four_observables": None if value_meas_all is None else {
                                        "sweep_then_sw_measure": value_meas_all, "sw_sweep_measure_ex_OBS_ALL": value_series_all, "unit": UNIT,
                                        "steps": a_steps, "what": "the same with largest_cluster as well (all outputs of sw_measure): per-step "
                                        "sw_sweep(1) + sw_measure, and one sw_sweep_measure(n) call"}},
        "other_configs": other,
        "last_observables": obs,
        "label_equivalence_rounds_per_sweep": (stats["le_rounds_total"] / stats["sweeps"]) if args.label_equivalence else None,
        "paper_context": {"flips_per_ns_256xM2050_L65536": PAPER_FLIPS_PER_NS, "flips_per_ns_1xM2050_L4096": 0.232,
                          "source": "PAPER.md:97-103 (Table 1)"},
    }
    print(json.dumps(out))
    if distributed:
        dist.destroy_process_group()
    return 0


# ------------------------------------------------------------------------------------------------ control plane only (tests)

def run_super(args):
    """`--super GXxGY`: ONE lattice cut into gx x gy pieces, the axis the paper's Table 1 scales along.
    With N = gx*gy ranks (torchrun) every rank owns one piece on its own GPU and reaches the others through CUDA IPC
    peer pointers (NVLink); with one rank all the pieces sit on this GPU.  value = L^2 * sweeps / time of the ONE lattice
    (strong scaling).  The phases of a sweep are ordered by the host (events in one process, a process-group barrier
    between ranks), so the clock is the wall clock around sweep + synchronize, max over ranks."""
    import torch
    import torch.distributed as dist

    from paper_1208_2080_b200.binding import SuperLattice
    gx, gy = (int(v) for v in args.super.lower().split("x"))
    rank, local_rank, world = rank_info()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product has no CPU path")
    if world not in (1, gx * gy):
        raise SystemExit(f"bench.py: --super {args.super} needs 1 rank (all pieces on one GPU) or {gx * gy} ranks (one piece each), not {world}")
    torch.cuda.set_device(local_rank)
    c = wl.CONFIGS[args.workload]
    L, q, K, N = c["L"], c["q"], c["K"], c["L"] ** 2
    if world > 1:
        from paper_1208_2080_b200.super_ranks import SuperLatticeRanks
        dist.init_process_group("gloo")          # control plane only (64-byte handles, barriers); the data path is peer memory
        sim = SuperLatticeRanks(L, q, K, c["seed"], gx, gy)
    else:
        sim = SuperLattice(L, q, K, c["seed"], gx, gy)
    sync = (lambda: None) if world > 1 else sim.synchronize     # (a rank-mode sweep ends with synchronize + barrier already)
    sim.init(c["start"])
    sim.sweep(args.warmup); sync()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.25)
    if world > 1:
        dist.barrier()
    wall0 = time.time()
    t0 = time.perf_counter()
    sim.sweep(args.steps); sync()
    dt = time.perf_counter() - t0
    wall1 = time.time()
    clocks = sampler.stop(wall0, wall1) if rank == 0 else None
    st = sim.backend.stats() if world > 1 else sim.stats()
    sums = torch.tensor([st["inter_links"], st["inter_hops"], st["inter_retries"], st["resolved_links"], st["kernel_launches"]], dtype=torch.int64)
    slowest = torch.tensor([dt], dtype=torch.float64)
    if world > 1:
        dist.all_reduce(slowest, op=dist.ReduceOp.MAX)
        dist.all_reduce(sums, op=dist.ReduceOp.SUM)               # every rank counts its own piece's share
    dt = float(slowest.item())
    sweeps = st["sweeps"]
    obs = sim.measure()
    if rank == 0:
        value = N * args.steps / dt / 1e9
        print(json.dumps({
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True, "scaling": "strong",
            "vs_baseline": (value / PAPER_FLIPS_PER_NS) if args.workload == wl.HEADLINE else None,
            "dtype": "u32", "data": "synthetic",
            "config": {"workload": args.workload, "L": L, "q": q, "K": K, "start": c["start"], "seed": c["seed"],
                       "decomposition": f"{gx}x{gy} pieces of {L // gx}x{L // gy}", "parallelism": f"{world} GPU(s), {gx * gy // world} piece(s) each",
                       "timing": "wall clock around sw_super_sweep + synchronize, max over ranks (host-ordered phases)",
                       "l2": "working set >> 126 MB L2, no flush needed" if N * 6 > (126 << 20) * 4 else "lattice fits L2"},
            "clocks": clocks, "gpu_launches": int(sums[4]) * args.steps // max(1, sweeps),
            "super": {"inter_piece_links_per_sweep": int(sums[0]) / sweeps, "inter_piece_label_loads_per_sweep": int(sums[1]) / sweeps,
                      "lost_hook_races_per_sweep": int(sums[2]) / sweeps, "resolved_links_per_sweep": int(sums[3]) / sweeps,
                      "boundary_sites_per_piece": st["boundary_sites_per_piece"],
                      "what": "label loads of stage 2 + resolve = the traffic that crosses NVLink when the pieces sit on different GPUs "
                              "(4 bytes each; the paper exchanges 4 N_x labels per GPU per round, PAPER.md:68)"},
            "last_observables": obs}))
    sim.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def run_control_plane_only(args):
    """Test hook (tests/test_bench_ranks.py): the rank plumbing of the N > 1 path on CPU -- gloo rendezvous, replica seeds,
    sum of units over the max of times, ONE line from rank 0 -- with the GPU work replaced by fixed numbers.  It measures
    nothing: `value` is null and the line says so."""
    import torch.distributed as dist

    from paper_1208_2080_b200 import replicas
    rank, local_rank, world = rank_info()
    if world > 1:
        dist.init_process_group("gloo")
    units, secs, rate = replicas.aggregate_throughput(1000.0 * args.steps, 1.0 + rank)
    if rank == 0:
        print(json.dumps({"metric": METRIC, "value": None, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
                          "control_plane_only": True, "units_all_ranks": units, "max_seconds": secs,
                          "replica_seeds": [replicas.replica_seed(1, r) for r in range(world)]}))
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


def spawn_ranks(args):
    """`--gpus N` without a torchrun environment: start the N ranks ourselves, one per GPU, the way the driver would."""
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(free_port()), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--workload", choices=sorted(wl.CONFIGS), default=wl.HEADLINE)
    ap.add_argument("--lazy", action="store_true", help="SW_FLAG_LAZY_LABELS: canonical labels flattened on demand only")
    ap.add_argument("--label-equivalence", action="store_true",
                    help="SW_FLAG_LABEL_EQUIVALENCE: the paper's scan + analysis labeling (comparison variant, not the product path)")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-other-configs", action="store_true")
    ap.add_argument("--cpu-baseline-sweeps", type=int, default=20)
    ap.add_argument("--reference-L", type=int, default=2048)
    ap.add_argument("--super", default=None, metavar="GXxGY",
                    help="the super-lattice decomposition of ONE lattice (PAPER.md:62-84): gx*gy ranks with one piece per GPU, or 1 rank")
    ap.add_argument("--control-plane-only", action="store_true", help=argparse.SUPPRESS)
    args = ap.parse_args()
    if args.gpus < 1:
        ap.error("--gpus must be >= 1")
    if args.impl == "reference":
        args.steps = 20 if args.steps is None else args.steps
        args.warmup = 5 if args.warmup is None else args.warmup
        return run_reference(args)
    # N ranks: either torchrun started us (WORLD_SIZE must then agree with --gpus), or we start them ourselves
    if "WORLD_SIZE" in os.environ:
        if int(os.environ["WORLD_SIZE"]) != args.gpus:
            raise SystemExit(f"bench.py: --gpus {args.gpus} but WORLD_SIZE={os.environ['WORLD_SIZE']}: refusing to run a different number of ranks")
    elif args.gpus > 1:
        return spawn_ranks(args)
    args.steps = 40 if args.steps is None else args.steps
    args.warmup = 60 if args.warmup is None else args.warmup
    if args.control_plane_only:
        return run_control_plane_only(args)
    if args.super:
        return run_super(args)
    return run_gpu(args)


if __name__ == "__main__":
    sys.exit(main())
