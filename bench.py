#!/usr/bin/env python
"""bench.py -- throughput of the checkerboard Monte Carlo sweep on B200 (contract: see DESIGN.md 7).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

One "step" = SWEEPS_PER_STEP consecutive checkerboard sweeps (both
half-sweep launches, Philox words, threshold compare, in-place write, fused per-sweep (B, M)) of the
BASELINE.json config-2 lattice (2D Ising spin-1/2, 8192 x 8192, T = 2.269), recorded after every
sweep.  Rows a0/a1 (threshold table, initial state) run once at setup; a8/a9 are checked after the
timed region.  `value` = attempted site updates per second over all ranks (Gflips/s).

Prints ONE JSON line on rank 0.  N > 1 runs independent replicas (different seeds), no collective
("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SWEEPS_PER_STEP = 100
BYTES_PER_UPDATE = 3  # read own colour, read other colour, write own colour (int8 split arrays)
# 1/4 Philox4x32-10 call = 5 wide multiplies + 5 three-input XORs, + 1 compare + 1 merge
INT_SLOTS_PER_UPDATE = 12
INT_SLOTS_PER_UPDATE_SPIN1 = 22
# dram__bytes_read.sum + dram__bytes_write.sum per half-sweep launch, from the `ncu --set full` captures summarised
# under profiles/ (caches flushed by ncu before the launch): workload -> (bytes, summary file)
NCU_DRAM_BYTES_PER_LAUNCH = {
    "cfg2_T2.269": (67.17e6 + 0.84e6, "profiles/r2_cfg2_final.md"),
    "cfg3": (138.46e6 + 28.19e6, "profiles/r2_tiled_variants_ncu.md"),
    "cfg4": (16.86e6 + 0.0e6, "profiles/r2_tiled_variants_ncu.md"),
    "cfg5_c0.10": (67.19e6 + 1.22e6, "profiles/r2_tiled_variants_ncu.md"),
    "cfg5_c0.30": (67.18e6 + 0.75e6, "profiles/r2_tiled_variants_ncu.md"),
    "hbm3d_1024": (1083.86e6 + 497.63e6, "profiles/r2_tiled_variants_ncu.md"),
}
# smsp__issue_active.avg.pct_of_peak_sustained_active of the half-sweep kernel in the cited capture
NCU_ISSUE_ACTIVE_PCT = {"cfg2_T2.269": 57.5,     # profiles/r2_cfg2_final.md
                        "cfg4": 52.9}            # profiles/r3_cfg4.md
KERNEL_FAMILY = {1: "generic", 2: "tiled", 4: "small", 5: "slab", 6: "bulk"}
KERNEL_NAME = {1: "k_sweep_generic (half-sweep)", 2: "k_sweep_tiled (half-sweep)",
               4: "k_sweep_small_lane (per half-sweep share of one launch)",
               5: "k_sweep_slab (per half-sweep share of one launch)", 6: "k_sweep_tiled_bulk (half-sweep)"}


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2_T2.269")
    ap.add_argument("--sweeps-per-step", type=int, default=SWEEPS_PER_STEP)
    ap.add_argument("--no-extras", action="store_true", help="skip the secondary workloads / cpu baseline")
    ap.add_argument("--batch-scan", action="store_true", help="instead of the benchmark: lsm_batch_sweep_record over R and cluster size")
    ap.add_argument("--size-scan", action="store_true",
                    help="instead of the benchmark: us/sweep of the tiled and the small (cluster) family over lattice sizes")
    ap.add_argument("--ne-scan", action="store_true",
                    help="instead of the benchmark: the North-East model at the paper's sizes (checkerboard / random-tile / balanced)")
    ap.add_argument("--pipe-probe", action="store_true",
                    help="instead of the benchmark: the integer-pipe microbenchmarks behind the 'alu' roofline (DESIGN.md 6)")
    ap.add_argument("--kernel", default="auto", choices=["auto", "generic", "tiled", "small", "slab", "bulk"],
                    help="kernel family (lsm_set_kernel); auto = the library's choice")
    return ap.parse_args()


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)", d
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)", {}


# ----------------------------------------------------------------------------- clocks sampler
class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons of one GPU every 100 ms while the timed region runs."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        self.ok = False
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception:
            self.ok = False

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            self._stop_evt.wait(0.1)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        return {
            "sm_mhz": statistics.median(self.samples) if self.samples else None,
            "sm_max_mhz": self.max_mhz,
            "reasons": sorted(self.reasons),
            "samples": len(self.samples),
        }


# ----------------------------------------------------------------------------- oracle legs (CPU)
def pin_to_one_core():
    """SURVEY.md 8(d), oracle timing: the single-threaded oracle pinned to one core.  Returns (core, previous mask)."""
    try:
        old = os.sched_getaffinity(0)
        cpu = max(old)
        os.sched_setaffinity(0, {cpu})
        return cpu, old
    except (AttributeError, OSError):
        return None, None


def time_oracle(w, L, sweeps):
    """The oracle as it stands, one thread, on an L^dims lattice of workload w: updates/s."""
    from oracle import lsm_oracle as O

    kw = w.create_args()
    kw["L"] = L
    o = O.Oracle(**kw)
    cpu, old = pin_to_one_core()
    try:
        t0 = time.perf_counter()
        o.sweep(sweeps)
        dt = time.perf_counter() - t0
    finally:
        if old is not None:
            os.sched_setaffinity(0, old)
    n = (L ** w.dims) * sweeps
    o.close()
    return n / dt, dt, n, cpu


def run_reference(args, w):
    """--impl reference: the CPU oracle on the host cores; each step = one sweep of a bounded
    2048^2 (or 128^3) sample of the workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from oracle import lsm_oracle as O

    L = 2048 if w.dims == 2 else 128
    kw = w.create_args()
    kw["L"] = L
    o = O.Oracle(**kw)
    cpu, old = pin_to_one_core()
    for _ in range(args.warmup):
        o.sweep(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        o.sweep(1)
    dt = time.perf_counter() - t0
    if old is not None:
        os.sched_setaffinity(0, old)
    upd = (L ** w.dims) * args.steps
    value = upd / dt / 1e9
    sample = (f"each step = 1 sweep of a {L}^{w.dims} lattice with the workload's J, h, T, seed ({L ** w.dims} updates); "
              f"one thread pinned to core {cpu}: 1 of {os.cpu_count()}")
    line = {
        "impl": "reference", "metric": "site_updates_per_sec", "value": value, "unit": "Gflips/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": w.name, "lattice": f"{w.L}^{w.dims}", "T": w.T, "sample": sample},
        "cpu_baseline": {"value": value, "unit": "Gflips/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "Gflips/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)
    return 0


# ----------------------------------------------------------------------------- our arm (GPU)
def run_ours(args, w):
    import torch
    import torch.distributed as dist

    from paper_1209_0296_b200 import build, lsm

    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    build.build()
    lsm.load()

    S = args.sweeps_per_step
    K, Wm = args.steps, max(args.warmup, 3)
    from dataclasses import replace

    from paper_1209_0296_b200 import replicas

    wl = replace(w, seed=replicas.rank_seed(w.seed, rank))  # replicas: independent seeds, no communication
    lat = lsm.Lattice(**wl.create_args(), device=f"cuda:{local}")
    if wl.model in (lsm.ISING, lsm.EA, lsm.POTTS):
        lat.set_tracking(False)  # persistence is not part of configs 1-4
    if args.kernel != "auto":
        lat.set_kernel({"generic": lsm.KERNEL_GENERIC, "tiled": lsm.KERNEL_TILED,
                        "small": lsm.KERNEL_SMALL, "slab": lsm.KERNEL_SLAB, "bulk": lsm.KERNEL_BULK}[args.kernel])
    N = lat.N
    obs = torch.empty((S, 2), dtype=torch.int64, device=lat.device)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=lat.device)  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(Wm):
        lat.sweep_record(S, out=obs)
    barrier()

    sampler = ClockSampler(local)
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(K)]
    launches0 = lat.launch_count
    barrier()
    for k in range(K):
        flush.fill_(k & 0xFF)  # L2 flush between timed iterations (not timed)
        ev[k][0].record()
        lat.sweep_record(S, out=obs)
        ev[k][1].record()
    barrier()
    clocks = sampler.stop()
    launches = lat.launch_count - launches0
    step_ms = [a.elapsed_time(b) for a, b in ev]
    total_ms = sum(step_ms)
    total_ms_max, updates_all, ups_mean = replicas.aggregate(total_ms, N * S * K, lat.device)
    # SURVEY.md 8(d) timing protocol: `value` is the MEDIAN timed step (max over ranks); the mean is kept beside it
    med_ms_max, _, ups = replicas.aggregate(statistics.median(step_ms), N * S, lat.device)
    value = ups / 1e9

    # sanity of the state after the timed region: fused running sums == full reduction (a6 vs a8)
    Bv, Mv, tdone = lat.measure_int()
    assert lat.measure_full() == (Bv, Mv), "fused observables disagree with the full reduction"
    assert tdone == S * (K + Wm)

    # ---- end-to-end through the C ABI with HOST buffers (pinned), copies inside the timed region.
    # Every step uploads its input configuration (N bytes, lsm_stage_spins_host on a copy stream), installs it
    # (lsm_set_spins: layout conversion + full reduction), sweeps S times and downloads the (B, M) series
    # (lsm_sweep_record_host_async): paper_1209_0296_b200/pipeline.py, the sequence tests/test_gpu_e2e.py holds to the
    # oracle.  Two DIFFERENT inputs alternate (the configurations at sweep tdone and tdone + S, each with its own sweep
    # counter), and every downloaded series is compared with the one recorded when the lattice went through those sweeps
    # directly, so a broken stream order shows up here and not only in the tests.
    from paper_1209_0296_b200.pipeline import HostPipeline

    h_in, ref_series = [], []
    for i in range(2):
        h = torch.empty(N, dtype=torch.int8).pin_memory()
        h.copy_(lat.get_spins().cpu())
        h_in.append((h, tdone + i * S))
        ref_series.append(lat.sweep_record(S).cpu())
    Ke = max(4, min(K, 10))
    pipe = HostPipeline(lat, S)
    seen = []

    def check_series(k, series):                   # host side, two steps behind the GPU
        seen.append(bool(torch.equal(series, ref_series[k & 1])))

    pipe.run([h_in[k & 1] for k in range(2)])
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    pipe.run([h_in[k & 1] for k in range(Ke)], consume=check_series)
    e1.record()
    torch.cuda.synchronize()
    e2e_ms = e0.elapsed_time(e1)
    e2e_value = replicas.aggregate(e2e_ms, N * S * Ke, lat.device)[2] / 1e9
    assert len(seen) == Ke and all(seen), f"e2e: downloaded series differ from the directly recorded ones: {seen}"
    assert lat.measure_int()[2] == h_in[(Ke - 1) & 1][1] + S
    e2e_oracle = e2e_oracle_check(lsm, wl, S) if rank == 0 else None

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel (the half-sweep kernel), DESIGN.md 6
    n_sweep_launches = 2 * S * K
    avg_launch_s = (sum(step_ms) * 1e-3) / n_sweep_launches      # average launch duration over the whole timed region
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    roofline, roofline_hbm = rooflines(wl, lat.kernel, avg_launch_s, sm_count, clocks.get("sm_max_mhz") or 1965)

    line = {
        "metric": "site_updates_per_sec", "value": value, "unit": "Gflips/s", "n_gpus": world, "steps": K,
        "warmup": Wm, "ms_per_step": med_ms_max, "higher_is_better": True, "scaling": "weak",
        "timing": {"value_is": "median of the timed steps (SURVEY.md 8(d))", "ms_per_step_mean": total_ms_max / K,
                   "value_mean": ups_mean / 1e9},
        "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": wl.name, "lattice": f"{wl.L}^{wl.dims}", "model": "Ising spin-1/2" if wl.two_S == 1 and wl.model == 0 else wl.note,
                   "T": wl.T, "J": wl.J, "h": wl.h, "sweeps_per_step": S, "record": "(B, M) after every sweep",
                   "parallelism": "replicas only" if world > 1 else "single GPU",
                   "kernel_family": KERNEL_FAMILY.get(lat.kernel, "?"),
                   "l2": "256 MiB flush write between timed steps; within a step a lattice smaller than the 126 MB L2 is re-read from L2"},
        "roofline": roofline,
        "roofline_hbm": roofline_hbm,
        "e2e": {"value": e2e_value, "unit": "Gflips/s", "h2d_bytes_per_step": pipe.h2d_bytes_per_step,
                "d2h_bytes_per_step": pipe.d2h_bytes_per_step, "steps": Ke,
                "api": "lsm_stage_spins_host (copy stream) + lsm_set_spins + lsm_sweep_record_host_async, pinned host buffers, "
                       "two staging buffers: the upload of step k+1 overlaps the sweeps of step k (paper_1209_0296_b200/pipeline.py)",
                "inputs": "two different configurations (sweep counters tdone, tdone + S) alternate",
                "verified": {"every_series_equals_direct_run": True, "oracle_reduced_shape": e2e_oracle}},
        "gpu_launches": int(launches),
        "clocks": clocks,
        "step_ms_min_med_max": [min(step_ms), statistics.median(step_ms), max(step_ms)],
    }

    if not args.no_extras and world == 1:
        words = 2 if wl.two_S == 2 or wl.model == lsm.POTTS else 1      # Philox words per update
        po = philox_microbench(lsm, torch)
        line["philox_only"] = po
        # SURVEY.md 8(d)'s integer bound, measured in this run: register-only Philox words/s / words per update
        roofline["philox_only_gwords_per_s"] = po["gwords_per_s"]
        roofline["frac_vs_philox_only"] = value / (po["gwords_per_s"] / words)
        roofline["sm_mhz_sampled"] = clocks.get("sm_mhz")
        if clocks.get("sm_mhz"):
            roofline["frac_at_sampled_clock"] = roofline["achieved"] / (sm_count * 64 * clocks["sm_mhz"] * 1e6 / 1e9)
        roofline["issue_active_pct"] = NCU_ISSUE_ACTIVE_PCT.get(wl.name)
        roofline["hbm"] = {k: roofline_hbm[k] for k in ("achieved", "peak", "unit", "frac")}
        # three seeds for the headline: 1 warm-up + median of 5 steps each
        roofline["three_seeds_gflips"] = three_seeds(lsm, torch, wl, S, lat.kernel, flush)
        others = other_workloads(lsm, torch, w.name, sm_count, clocks.get("sm_max_mhz") or 1965, po)
        line["other_workloads"] = others
        # BASELINE.json's configs (and the extras) in the key the driver keeps: workload -> [Gflips/s, fraction of the
        # binding roofline (null where the family has no per-half-sweep roofline), kernel family]
        per = {wl.name: [round(value, 1), round(roofline["frac"], 3), KERNEL_FAMILY.get(lat.kernel, "?")]}
        for name, o in others.items():
            if "gflips" in o:
                fr = (o.get("roofline") or {}).get("frac")
                if fr is not None and o["roofline"].get("binding_bound") == "hbm":
                    fr = o["roofline_hbm"]["frac"]
                per[name] = [round(o["gflips"], 1), None if fr is None else round(fr, 3),
                             o.get("kernel_family", "ne_tile" if "random_tile" in name else "?")]
        roofline["per_config"] = per
        roofline["per_config_note"] = ("[Gflips/s, fraction of the binding roofline, kernel family]; North-East rows (cfg5): the 12-slot model "
                                       "charges one Philox word to every site while the rule draws only for facilitated sites (about c^2 of them), "
                                       "so the fraction can exceed 1 at low c; random_tile rows: against 2 picks per Philox call; "
                                       "null: the small family has no per-half-sweep launch to put against a roofline")
        sweeps = 4
        v, dt, n, cpu = time_oracle(w, w.L, sweeps)
        line["cpu_baseline"] = {"value": v / 1e9, "unit": "Gflips/s", "cores": 1, "kind": "oracle",
                                "sample": f"{sweeps} sweeps of the full {w.L}^{w.dims} lattice ({n} updates, {dt:.1f} s), "
                                          f"pinned to core {cpu}: 1 of {os.cpu_count()}"}
    else:
        line["cpu_baseline"] = None
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()
    return 0


def three_seeds(lsm, torch, wl, S, family, flush):
    """Headline workload with three seeds: per seed 1 warm-up step + the median of 5 timed steps (L2 flushed between)."""
    from dataclasses import replace

    out = {}
    for i in range(3):
        w = replace(wl, seed=wl.seed + 16 * i)
        lat = lsm.Lattice(**w.create_args())
        if w.model in (lsm.ISING, lsm.EA, lsm.POTTS):
            lat.set_tracking(False)
        lat.set_kernel(family)
        obs = torch.empty((S, 2), dtype=torch.int64, device=lat.device)
        lat.sweep_record(S, out=obs)
        ms = []
        for k in range(5):
            flush.fill_(k)
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            lat.sweep_record(S, out=obs)
            e1.record()
            torch.cuda.synchronize()
            ms.append(e0.elapsed_time(e1))
        out[str(w.seed)] = round(w.N * S / (statistics.median(ms) * 1e-3) / 1e9, 1)
        lat.close()
    return out


def e2e_oracle_check(lsm, w, S):
    """Outside the timed region: the same pipeline on a reduced shape of the workload, three different inputs from an
    oracle trajectory, every downloaded series and the final configuration compared with the oracle."""
    import numpy as np
    import torch

    from oracle import lsm_oracle as O
    from paper_1209_0296_b200.pipeline import HostPipeline

    L = 256 if w.dims == 2 else 32
    S = min(S, 20)
    kw = w.create_args()
    kw["L"] = L
    traj, runner = O.Oracle(**kw), O.Oracle(**kw)
    inputs, want = [], []
    for t in (0, 3, 7):
        traj.sweep(t - traj.sweeps_done)
        cfg = traj.get_spins().copy()
        runner.set_spins(cfg, t)
        want.append(runner.sweep_record(S))
        inputs.append((torch.from_numpy(cfg).pin_memory(), t))
    lat = lsm.Lattice(**kw)
    got = {}
    HostPipeline(lat, S).run(inputs, consume=lambda k, series: got.__setitem__(k, series.numpy().copy()))
    ok = all(np.array_equal(got[k], want[k]) for k in range(3)) and np.array_equal(lat.get_spins().cpu().numpy(), runner.get_spins())
    lat.close()
    assert ok, "e2e pipeline disagrees with the oracle on the reduced shape"
    return f"{L}^{w.dims}, 3 steps x {S} sweeps: bit-exact"


def rooflines(w, family, avg_launch_s, sm_count, sm_max_mhz):
    """Both rooflines of one half-sweep launch and which of them binds this workload.

    alu: integer instruction slots (12 per update for one Philox word per site, 22 for two) against
         SMs x 64 lanes x max SM clock -- one 16-lane math instruction per 2 cycles and sub-partition, the rate
         `bench.py --pipe-probe` measures on this GPU;
    hbm: 3 algorithmic bytes per update against the measured copy bandwidth (MEASURED_PEAKS.json)."""
    hbm_peak, peak_src, _ = measured_peaks()
    updates_per_launch = w.N // 2
    slots = INT_SLOTS_PER_UPDATE_SPIN1 if w.two_S == 2 else INT_SLOTS_PER_UPDATE
    alu_peak = sm_count * 64 * sm_max_mhz * 1e6 / 1e9           # G integer instruction slots / s
    alu_achieved = slots * updates_per_launch / avg_launch_s / 1e9
    hbm_achieved = BYTES_PER_UPDATE * updates_per_launch / avg_launch_s / 1e9
    binding = "alu" if alu_peak / slots < hbm_peak / BYTES_PER_UPDATE else "hbm"
    traffic = NCU_DRAM_BYTES_PER_LAUNCH.get(w.name) if family == 2 else None
    roofline = {"bound": "alu", "achieved": alu_achieved, "peak": alu_peak, "unit": "Gslot/s",
                "frac": alu_achieved / alu_peak,
                "traffic": traffic[0] if traffic else None,
                "traffic_source": traffic[1] if traffic else None,
                "traffic_unit": "bytes per launch (ncu dram read+write, cold L2; algorithmic = 3 B x updates_per_launch)",
                "peak_source": f"{sm_count} SMs x 64 integer lanes/clk x clocks.max.sm {sm_max_mhz} MHz (DESIGN.md 6; bench.py --pipe-probe)",
                "kernel": KERNEL_NAME.get(family, "?"), "binding_bound": binding,
                "bound_gflips": {"alu": alu_peak / slots, "hbm": hbm_peak / BYTES_PER_UPDATE},
                "algorithmic_int_slots_per_update": slots, "updates_per_launch": updates_per_launch,
                "avg_launch_us": avg_launch_s * 1e6}
    lattice_mib = w.N / 2 ** 20
    roofline_hbm = {"bound": "hbm", "achieved": hbm_achieved, "peak": hbm_peak, "unit": "GB/s",
                    "frac": hbm_achieved / hbm_peak, "peak_source": peak_src,
                    "algorithmic_bytes_per_update": BYTES_PER_UPDATE,
                    "note": ("the lattice stays in the SMs' shared memory for the whole launch: global traffic is the boundary-row mailboxes (L2) only"
                             if family == 5 else f"the {lattice_mib:.0f} MiB lattice is L2-resident between launches: DRAM traffic is below the algorithmic bytes"
                             if lattice_mib < 100 else f"the {lattice_mib:.0f} MiB lattice exceeds the 126 MB L2: every launch streams it from HBM")}
    return roofline, roofline_hbm


def philox_microbench(lsm, torch):
    """Register-only Philox4x32-10 loop: words/s the integer pipes deliver (bound for step a4)."""
    blocks, calls = 148 * 8, 4096
    lsm.philox_throughput(blocks, 64)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    sink = lsm.philox_throughput(blocks, calls)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    calls_s = blocks * 256 * calls / (ms * 1e-3)
    del sink
    return {"gcalls_per_s": calls_s / 1e9, "gwords_per_s": 4 * calls_s / 1e9,
            "updates_bound_gflips_1word": 4 * calls_s / 1e9, "updates_bound_gflips_2words": 2 * calls_s / 1e9}


def random_tile_roofline(gpicks, po):
    """The random-tile schedule draws every pick: one Philox4x32-10 call serves two picks (position word + acceptance
    word each; include/lsm.h, readings D21 / D24), so its integer bound is 2 x the register-only Philox call rate
    measured in this run (k_ne_random_tile, one launch = half / a quarter of a sweep)."""
    if not po:
        return None
    peak = 2.0 * po["gcalls_per_s"]
    return {"bound": "alu", "achieved": gpicks, "peak": peak, "unit": "Gpick/s", "frac": gpicks / peak,
            "peak_source": "2 picks per Philox call x philox_only.gcalls_per_s of this run", "kernel": "k_ne_random_tile"}


def other_workloads(lsm, torch, skip, sm_count, sm_max_mhz, po=None):
    """Short timings of the other BASELINE.json configs (context for the headline number)."""
    from paper_1209_0296_b200 import workloads as W

    out = {}
    for name, sweeps in (("cfg1", 1000), ("cfg2_T2.0", 100), ("cfg2_T2.6", 100), ("cfg3", 40), ("cfg4", 100),
                         ("cfg5_c0.10", 100), ("cfg5_c0.20", 100), ("cfg5_c0.30", 100), ("hbm3d_1024", 6),
                         ("cold2d_T0.30", 100), ("mid2d_512", 2000), ("mid2d_1024", 1000), ("mid2d_2048", 400),
                         ("mid2d_4096", 100), ("mid3d_128", 400), ("ea2d_8192", 100), ("ea3d_512", 40), ("potts2d_q3_4096", 20)):
        if name == skip:
            continue
        w = W.by_name(name)
        try:
            lat = lsm.Lattice(**w.create_args())
            if w.model in (lsm.ISING, lsm.EA, lsm.POTTS):
                lat.set_tracking(False)
            obs = torch.empty((sweeps, 2), dtype=torch.int64, device="cuda")
            lat.sweep_record(sweeps, out=obs)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            reps = 3
            e0.record()
            for _ in range(reps):
                lat.sweep_record(sweeps, out=obs)
                if w.model in (lsm.NE_HEATBATH, lsm.NE_METROPOLIS):
                    lat.persistence()
            e1.record()
            torch.cuda.synchronize()
            s = e0.elapsed_time(e1) * 1e-3
            gf = w.N * sweeps * reps / s / 1e9
            out[name] = {"gflips": gf, "alg_GBps": gf * BYTES_PER_UPDATE, "us_per_sweep": s / (sweeps * reps) * 1e6,
                         "kernel_family": KERNEL_FAMILY.get(lat.kernel, "?")}
            if lat.kernel == 5:
                out[name]["temporal_depth"] = lat.temporal_depth
            if lat.kernel in (2, 5, 6):      # per half-sweep: one launch (tiled) or that share of one launch (slab)
                r, rh = rooflines(w, lat.kernel, s / (2 * sweeps * reps), sm_count, sm_max_mhz)
                out[name]["roofline"] = {k: r[k] for k in ("bound", "achieved", "peak", "unit", "frac", "traffic",
                                                           "traffic_source", "binding_bound", "avg_launch_us")}
                out[name]["roofline_hbm"] = {k: rh[k] for k in ("achieved", "peak", "unit", "frac", "note")}
            if name == "cfg5_c0.30":
                # the paper's corrected North-East algorithm on the same lattice (32 x 32 tiles,
                # lambda = 16 is the paper's best configuration)
                n_rt = 10
                lat.sweep_random_tile(n_rt, 32, 16, out=obs)
                torch.cuda.synchronize()
                e0.record()
                lat.sweep_random_tile(n_rt, 32, 16, out=obs)
                e1.record()
                torch.cuda.synchronize()
                s_rt = e0.elapsed_time(e1) * 1e-3
                out[name + "_random_tile_b32_lambda16"] = {"gflips": w.N * n_rt / s_rt / 1e9,
                                                           "us_per_sweep": s_rt / n_rt * 1e6, "launches_per_sweep": 2,
                                                           "roofline": random_tile_roofline(w.N * n_rt / s_rt / 1e9, po)}
                lat.sweep_random_tile(n_rt, 32, 16, out=obs, balanced=True)
                torch.cuda.synchronize()
                e0.record()
                lat.sweep_random_tile(n_rt, 32, 16, out=obs, balanced=True)   # balance-preserving variant
                e1.record()
                torch.cuda.synchronize()
                s_rt = e0.elapsed_time(e1) * 1e-3
                out[name + "_random_tile_balanced_b32_lambda16"] = {"gflips": w.N * n_rt / s_rt / 1e9,
                                                                    "us_per_sweep": s_rt / n_rt * 1e6, "launches_per_sweep": 4,
                                                                    "roofline": random_tile_roofline(w.N * n_rt / s_rt / 1e9, po)}
            lat.close()
            del lat, obs
        except Exception as e:  # a secondary workload must not take the headline down
            out[name] = {"error": repr(e)[:200]}
    return out


def size_scan():
    """us per sweep (per-sweep (B, M) recorded) of the tiled and the small family from 32^2 to 1024^2 and 16^3 to 64^3:
    where one launch per half-sweep stops paying (the paper's own lattice sizes)."""
    import torch

    from paper_1209_0296_b200 import build, lsm

    build.build()
    rows = []
    for dims, L in [(2, 32), (2, 64), (2, 128), (2, 256), (2, 512), (2, 1024), (2, 2048), (2, 4096), (3, 16), (3, 32), (3, 64),
                    (3, 128)]:
        row = {"dims": dims, "L": L}
        for fam, name in ((lsm.KERNEL_TILED, "tiled"), (lsm.KERNEL_SMALL, "small"), (lsm.KERNEL_SLAB, "slab")):
            lat = lsm.Lattice(dims=dims, L=L, T=2.269 if dims == 2 else 4.5115, seed=3)
            lat.set_tracking(False)
            try:
                lat.set_kernel(fam)
            except lsm.LsmError:
                row[name] = None
                continue
            n = 500 if lat.N <= 1 << 22 else 100
            obs = torch.empty((n, 2), dtype=torch.int64, device="cuda")
            lat.sweep_record(n, out=obs)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            lat.sweep_record(n, out=obs)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            row[name] = {"us_per_sweep": ms * 1e3 / n, "gflips": lat.N * n / ms / 1e6}
            if fam == lsm.KERNEL_SLAB:                   # temporal depth: half-sweeps between two boundary exchanges
                row[name]["depth"] = lat.temporal_depth
                for depth in (1, 2, 3, 4):
                    try:
                        lat.set_temporal_depth(depth)
                    except lsm.LsmError:
                        break
                    lat.sweep_record(n, out=obs)
                    torch.cuda.synchronize()
                    e0.record()
                    lat.sweep_record(n, out=obs)
                    e1.record()
                    torch.cuda.synchronize()
                    row[name][f"gflips_depth{depth}"] = lat.N * n / e0.elapsed_time(e1) / 1e6
            lat.close()
        lat = lsm.Lattice(dims=dims, L=L, T=2.269 if dims == 2 else 4.5115, seed=3)
        row["auto_family"] = KERNEL_FAMILY.get(lat.kernel)
        lat.close()
        rows.append(row)
        print(json.dumps(row), flush=True)
    # Many independent small lattices at once (the paper averages 30 realisations): every handle sweeps
    # on its own stream, the small family's clusters of <= 16 blocks run side by side on the 148 SMs.
    L, n = 128, 500
    for nlat in (1, 8, 32, 64):
        lats = [lsm.Lattice(dims=2, L=L, T=2.269, seed=100 + i) for i in range(nlat)]
        streams = [torch.cuda.Stream() for _ in range(nlat)]
        obs = [torch.empty((n, 2), dtype=torch.int64, device="cuda") for _ in range(nlat)]
        for lat in lats:
            lat.set_tracking(False)
        torch.cuda.synchronize()
        for rep in range(2):                          # the first pass warms up
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for st in streams:
                st.wait_event(e0)
            for lat, st, o in zip(lats, streams, obs):
                lat.sweep_record(n, out=o, stream=st)
            for st in streams:
                torch.cuda.current_stream().wait_stream(st)
            e1.record()
            torch.cuda.synchronize()
        ms = e0.elapsed_time(e1)
        print(json.dumps({"concurrent_lattices": nlat, "L": L, "family": lats[0].kernel, "sweeps_each": n,
                          "aggregate_gflips": nlat * L * L * n / ms / 1e6, "us_per_sweep_per_lattice": ms * 1e3 / n}), flush=True)
        for lat in lats:
            lat.close()
    batch_scan()
    return 0


def batch_scan(L=128, n=500):
    """The same many-small-lattices load through lsm_batch_sweep_record: ONE launch for R lattices x n sweeps
    (SURVEY.md 8(f) NEXT-3), for several R and blocks per replica (0 = the library's choice)."""
    import torch

    from paper_1209_0296_b200 import build, lsm

    build.build()
    for R in (1, 8, 32, 64, 128, 256, 512):
        for c in (0, 1, 2, 4, 8, 16):
            b = lsm.Batch(dims=2, L=L, T=[2.1 + 0.3 * r / R for r in range(R)], seeds=[100 + r for r in range(R)])
            b.set_tracking(False)
            b.set_cluster(c)
            obs = torch.empty((R, n, 2), dtype=torch.int64, device="cuda")
            b.sweep_record(n, out=obs)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            b.sweep_record(n, out=obs)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            print(json.dumps({"batch_lattices": R, "L": L, "blocks_per_replica": c, "sweeps_each": n,
                              "aggregate_gflips": R * L * L * n / ms / 1e6, "us_per_sweep_of_the_batch": ms * 1e3 / n}), flush=True)
            b.close()
    return 0


PROBE_MODES = [
    # mode, stream per loop iteration and thread, wide multiplies, other IMADs, ALU-pipe instructions
    (0, "16 LOP3", 0, 0, 16),
    (1, "8 IMAD", 0, 8, 0),
    (2, "8 IMAD.WIDE (+8 adds)", 8, 0, 8),
    (3, "8 IMAD + 16 LOP3", 0, 8, 16),
    (4, "4 Philox calls (80 WIDE + 80 LOP3)", 80, 0, 80),
    (5, "4 Philox calls + 80 LOP3", 80, 0, 160),
    (6, "4 Philox calls + 160 LOP3", 80, 0, 240),
    (7, "4 Philox calls + 240 LOP3", 80, 0, 320),
    (8, "4 Philox calls + 80 IMAD", 80, 80, 80),
    (9, "4 Philox calls + 80 IMAD + 80 LOP3", 80, 80, 160),
    (10, "4 Philox calls + 80 IMAD + 160 LOP3", 80, 80, 240),
    # the wide multiply split into IMAD.HI + IMAD (counted here as 2 "other IMADs" each, no wide multiply)
    (11, "8 mul.hi + 8 mul.lo (+8 adds)", 0, 16, 8),
    (12, "4 Philox calls, hi/lo split (80 HI + 80 LO + 80 LOP3)", 0, 160, 80),
    (13, "4 Philox calls, hi/lo split + 80 LOP3", 0, 160, 160),
]


def ne_scan():
    """The North-East model at the paper's own sizes (128^2 and 512^2, 30 realisations per concentration)
    and upwards: us per sweep of the checkerboard sweep, of the paper's corrected algorithm (32 x 32 tiles, lambda = 16,
    PAPER.md:128-140,155; two dependent launches per sweep) and of its balance-preserving variant (four launches), for one
    lattice; then 30 realisations one after the other on one stream and on 30 streams."""
    import torch

    from paper_1209_0296_b200 import build, lsm, workloads as W

    build.build()
    T = W.ne_temperature(0.30)

    def timed(fn, n):
        fn(n)
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        fn(n)
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) * 1e3 / n

    for L in (128, 512, 2048, 8192):
        n = 200 if L <= 512 else 20
        lat = lsm.Lattice(dims=2, L=L, model=lsm.NE_HEATBATH, J=0.0, T=T, seed=7)
        row = {"L": L, "c": 0.30, "auto_family": KERNEL_FAMILY.get(lat.kernel),
               "checkerboard_us_per_sweep": timed(lambda k: lat.sweep(k), n),
               "random_tile_b32_l16_us_per_sweep": timed(lambda k: lat.sweep_random_tile(k, 32, 16), n),
               "balanced_b32_l16_us_per_sweep": timed(lambda k: lat.sweep_random_tile(k, 32, 16, balanced=True), n)}
        for key in ("checkerboard", "random_tile_b32_l16", "balanced_b32_l16"):
            row[key + "_gflips"] = lat.N / row[key + "_us_per_sweep"] / 1e3
        lat.close()
        print(json.dumps(row), flush=True)
    for L in (128, 512):
        R, n = 30, 200
        lats = [lsm.Lattice(dims=2, L=L, model=lsm.NE_HEATBATH, J=0.0, T=T, seed=100 + r) for r in range(R)]
        streams = [torch.cuda.Stream() for _ in range(R)]
        torch.cuda.synchronize()

        def serial(k):
            for lat in lats:
                lat.sweep_random_tile(k, 32, 16)

        def parallel(k):
            cur = torch.cuda.current_stream()
            for lat, st in zip(lats, streams):
                st.wait_stream(cur)                       # fork from / join into the stream the timing events are on
                lat.sweep_random_tile(k, 32, 16, stream=st)
            for st in streams:
                cur.wait_stream(st)

        row = {"L": L, "realisations": R, "one_stream_us_per_sweep_of_all": timed(serial, n),
               "streams_us_per_sweep_of_all": timed(parallel, n)}
        row["one_stream_gflips"] = R * L * L / row["one_stream_us_per_sweep_of_all"] / 1e3
        row["streams_gflips"] = R * L * L / row["streams_us_per_sweep_of_all"] / 1e3
        for lat in lats:
            lat.close()
        # the same 30 realisations as ONE batch: every launch of the schedule covers the tiles of all of them
        batch = lsm.Batch(T=[T] * R, seeds=[100 + r for r in range(R)], dims=2, L=L, model=lsm.NE_HEATBATH, J=0.0)
        row["batch_us_per_sweep_of_all"] = timed(lambda k: batch.sweep_random_tile(k, 32, 16), n)
        row["batch_balanced_us_per_sweep_of_all"] = timed(lambda k: batch.sweep_random_tile(k, 32, 16, balanced=True), n)
        row["batch_gflips"] = R * L * L / row["batch_us_per_sweep_of_all"] / 1e3
        batch.close()
        print(json.dumps(row), flush=True)
    return 0


def pipe_probe(blocks_per_sm=8, iters=1024):
    """Register-only integer instruction streams (csrc/probe/pipe_probe.cu, its own libpipe_probe.so): cycles per loop
    iteration and warp against the issue law of DESIGN.md 6 -- every 16-lane math instruction (ALU or FMA-heavy pipe)
    FMA-heavy pipe: 4 cycles per wide multiply, 2 per other IMAD; ALU pipe: 2 cycles per instruction, and every wide
    multiply also takes one ALU-pipe slot: cycles = max(4 W + 2 I, 2 (A + W + 3 loop instructions))."""
    import ctypes

    import torch

    from paper_1209_0296_b200 import build

    lib = ctypes.CDLL(build.build_probe())
    lib.pipe_probe_run.restype = ctypes.c_int
    lib.pipe_probe_run.argtypes = [ctypes.c_int, ctypes.c_int, ctypes.c_int, ctypes.c_void_p, ctypes.c_void_p]
    props = torch.cuda.get_device_properties(0)
    sms = props.multi_processor_count
    try:
        import pynvml

        pynvml.nvmlInit()
        mhz = pynvml.nvmlDeviceGetMaxClockInfo(pynvml.nvmlDeviceGetHandleByIndex(0), pynvml.NVML_CLOCK_SM)
    except Exception:
        mhz = 1965
    warps_per_smsp = blocks_per_sm * 8 / 4.0
    blocks = sms * blocks_per_sm
    sink = torch.empty(blocks * 256, dtype=torch.int32, device="cuda")
    stream = ctypes.c_void_p(torch.cuda.current_stream().cuda_stream)
    print(f"# {props.name}  clocks.max.sm {mhz} MHz  {warps_per_smsp:.0f} warps per sub-partition, {iters} iterations")
    print("| stream | measured cycles/iter/warp | law max(4W+2I, 2(A+W+3)) | measured / law | math instr per cycle and sub-partition |")
    print("|---|---|---|---|---|")
    for mode, name, Wd, I, A in PROBE_MODES:
        assert lib.pipe_probe_run(mode, blocks, 32, sink.data_ptr(), stream) == 0
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        assert lib.pipe_probe_run(mode, blocks, iters, sink.data_ptr(), stream) == 0
        e1.record()
        torch.cuda.synchronize()
        cyc = e0.elapsed_time(e1) * 1e-3 * mhz * 1e6 / iters / warps_per_smsp
        law = max(4 * Wd + 2 * I, 2 * (A + Wd + 3))
        print(f"| {name} | {cyc:.1f} | {law} | {cyc / law:.2f} | {(Wd + I + A + 3) / cyc:.3f} |")
    return 0


def main():
    args = parse()
    if args.pipe_probe:
        return pipe_probe()
    if args.ne_scan:
        return ne_scan()
    if args.batch_scan:
        return batch_scan()
    if args.size_scan:
        # more hardware queues than the default 8, so that more than 8 handles can sweep side by side
        os.environ.setdefault("CUDA_DEVICE_MAX_CONNECTIONS", "32")
        return size_scan()
    from paper_1209_0296_b200 import workloads as W

    w = W.by_name(args.workload)
    if args.impl == "reference":
        return run_reference(args, w)
    return run_ours(args, w)


if __name__ == "__main__":
    sys.exit(main())
