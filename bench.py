#!/usr/bin/env python
"""bench.py -- one JSON line for the headline metric of BASELINE.json:

    "Plummer 4M theta=0.75 particles/s per full step; walk flop/s vs FP32 peak"

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload NAME]

A "step" is one pass of the whole hot path (bbox, keys, sort, reorder, build, groups,
multipoles, walk) over the seeded Plummer sphere of BASELINE.json configs[3] (N = 2^22, eps = 0.00125,
theta = 0.75), all particles active.  `value` = particles / device time of a step with the particles already
resident in HBM; `e2e` = the same through bonsai_step_host() with HOST buffers (H2D of the particles and D2H of
acc/pot inside the timed region).  The path does not shard ("replicas only"): with
--gpus N > 1 every rank runs the same step on its own replica, no collective on the data path, and `value` is
the sum over ranks of N / (max over ranks of the time).

The timed region (`value`, `ms_per_step`) runs the library UN-instrumented; the per-stage split (`stages`, and the
walk time behind `roofline`) comes from a second set of K steps with the library's stage events switched on, and
`instrumented_ms_per_step` says what that instrumentation costs.  `roofline.peak` is derived (SMs x 128 lanes x 2 flop
x clocks.max.sm); `roofline.peak_measured` is bonsai_measure_fp32_peak() run in this process (FFMA2 and FFMA).

--impl reference times the CPU oracle (oracle/, single thread, fp64), as it stands, on a bounded sample of the
same workload; it needs no GPU.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "particles_per_second_full_step"
UNIT = "particles/s"
FLOP_PP, FLOP_PC = 20, 63          # DESIGN.md R20: FMA = 2 flop, rsqrt = 1
FP32_LANES_PER_SM = 128            # B200 (sm_100): 4 SMSPs x 32 FP32 lanes, 2 flop per lane per clock (FMA)
L2_FLUSH_BYTES = 256 << 20         # > 126 MB L2


def _workload(name: str):
    from paper_1204_2280_b200 import workloads as W
    cfg = W.CONFIGS[name]
    return W, cfg["n"], cfg["theta"], cfg["eps"]


# ------------------------------------------------------------------------------------------------------
# CPU oracle legs (cpu_baseline of the default run, and --impl reference)
# ------------------------------------------------------------------------------------------------------
def oracle_step_sample(pm, theta, eps, ncrit, group_mode, group_cell, walk_budget_s):
    """The oracle's full step, its walk restricted to an evenly spaced sample of the groups.

    All stages before the walk run in full; the walk (>= 98 % of the oracle's time) is first probed on 64
    groups, then timed on every `stride`-th group with `stride` the smallest power of two that keeps it within
    `walk_budget_s`, and scaled by n_particles / n_sinks_sampled (the groups are evenly spaced along the Morton curve).
    Returns (estimated seconds of one full step, description of the sample, {"stride", "measured_s"}): the third
    value says what was actually executed -- every `stride`-th group, `measured_s` seconds of wall clock.
    """
    import oracle as O
    t0 = time.perf_counter()
    s = O.build(pm, 16, ncrit, group_mode, None, None, group_cell)
    t_build = time.perf_counter() - t0
    ng = s.groups.n_groups
    probe = np.unique(np.linspace(0, ng - 1, min(ng, 64)).astype(np.uint32))
    t0 = time.perf_counter()
    O.walk(theta, eps, s.sorted_pos_mass, s.tree, s.groups, probe)
    per_group = (time.perf_counter() - t0) / len(probe)
    stride = 1
    while per_group * ng / stride > walk_budget_s and stride < ng:
        stride *= 2
    sel = np.arange(0, ng, stride, dtype=np.uint32)
    t0 = time.perf_counter()
    O.walk(theta, eps, s.sorted_pos_mass, s.tree, s.groups, sel)
    t_walk = time.perf_counter() - t0
    n_sinks = int(s.groups.count[sel].sum())
    est = t_build + t_walk * (s.groups.n_active / n_sinks)
    what = (f"all pre-walk stages on all {pm.shape[0]} particles ({t_build:.2f} s) + walk of {len(sel)} of {ng} "
            f"groups (every {stride}th, {n_sinks} sinks, {t_walk:.2f} s) scaled by {s.groups.n_active}/{n_sinks}")
    return est, what, {"stride": int(stride), "measured_s": float(t_build + t_walk)}


def cpu_baseline(pm, theta, eps, ncrit, group_mode, group_cell, budget_s=12.0):
    est, what, _ = oracle_step_sample(pm, theta, eps, ncrit, group_mode, group_cell, budget_s)
    return {"value": pm.shape[0] / est, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what,
            "est_full_step_s": est}


def cpu_baseline_all_cores(pm, theta, eps, ncrit, group_mode, group_cell, budget_s=10.0):
    """The same oracle with its walk under an outer parallel loop over groups (groups are independent) on every host
    core -- SURVEY.md section 8(d) (ii); the paper's CPU side is a 4-core Xeon.  The stages before the
    walk stay single-threaded as the oracle has them (~2 % of its time).  `cores` is read at run time."""
    import oracle as O
    cores = len(os.sched_getaffinity(0)) if hasattr(os, "sched_getaffinity") else (os.cpu_count() or 1)
    t0 = time.perf_counter()
    s = O.build(pm, 16, ncrit, group_mode, None, None, group_cell)
    t_build = time.perf_counter() - t0
    ng = s.groups.n_groups
    probe = np.unique(np.linspace(0, ng - 1, min(ng, 16 * cores)).astype(np.uint32))
    t0 = time.perf_counter()
    O.walk_threads(theta, eps, s.sorted_pos_mass, s.tree, s.groups, probe, cores)
    per_group = (time.perf_counter() - t0) / len(probe)
    stride = 1
    while per_group * ng / stride > budget_s and stride < ng:
        stride *= 2
    sel = np.arange(0, ng, stride, dtype=np.uint32)
    t0 = time.perf_counter()
    O.walk_threads(theta, eps, s.sorted_pos_mass, s.tree, s.groups, sel, cores)
    t_walk = time.perf_counter() - t0
    n_sinks = int(s.groups.count[sel].sum())
    est = t_build + t_walk * (s.groups.n_active / n_sinks)
    what = (f"pre-walk stages single-threaded on all {pm.shape[0]} particles ({t_build:.2f} s) + walk of {len(sel)} of "
            f"{ng} groups (every {stride}th, {n_sinks} sinks) on {cores} threads ({t_walk:.2f} s) scaled by "
            f"{s.groups.n_active}/{n_sinks}")
    return {"value": pm.shape[0] / est, "unit": UNIT, "cores": cores, "kind": "oracle, outer parallel loop over groups",
            "sample": what, "est_full_step_s": est}


def run_reference(args):
    """--impl reference: the oracle, as it stands, on the host cores (rank 0 only)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return 0
    W, n, theta, eps = _workload(args.workload)
    pm = W.plummer(n)
    # each step: the full pre-walk stages (~1.5 s) + a walk sample bounded to ~4 s, so that the default 20 steps end
    # within two minutes
    for _ in range(min(args.warmup, 1)):
        oracle_step_sample(pm, theta, eps, args.ncrit, args.group_mode, args.group_cell, 2.0)
    ests, measured, what, info = [], [], "", {"stride": 1}
    for _ in range(args.steps):
        est, what, info = oracle_step_sample(pm, theta, eps, args.ncrit, args.group_mode, args.group_cell, 4.0)
        ests.append(est)
        measured.append(info["measured_s"])
    est = float(np.mean(ests))
    value = n / est
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": est * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": args.workload, "n": n, "theta": theta, "eps": eps, "nleaf": 16,
                   "ncrit": args.ncrit, "group_mode": args.group_mode, "group_cell": args.group_cell},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        # ms_per_step is an EXTRAPOLATION: each of the `steps` executed every stride-th group's walk (plus all pre-walk
        # stages) in measured_s_per_step seconds of wall clock and scaled it to all sinks
        "sampled": info["stride"] > 1, "stride": info["stride"], "measured_s_per_step": float(np.mean(measured)),
    }
    print(json.dumps(line), flush=True)
    return 0


# ------------------------------------------------------------------------------------------------------
# clocks
# ------------------------------------------------------------------------------------------------------
class ClockSampler:
    """nvidia-smi clocks / throttle reasons of one GPU, sampled every 50 ms while running."""
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.thread = None
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(index), f"--query-gpu={self.FIELDS}", "--format=csv,noheader,nounits",
                 "-lms", "50"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except OSError:
            self.proc = None

    def _read(self):
        for ln in self.proc.stdout:
            self.rows.append((time.perf_counter(), ln.strip()))

    def stop(self, t0: float, t1: float) -> dict:
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        sm, smax, power, reasons = [], [], [], set()
        names = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")
        for t, ln in self.rows:
            if not (t0 - 0.05 <= t <= t1 + 0.15):
                continue
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1])); power.append(float(f[2]))
            except ValueError:
                continue
            for k, nm in enumerate(names):
                if f[3 + k].lower().startswith("active"):
                    reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "power_w_max": max(power) if power else None, "samples": len(sm), "reasons": sorted(reasons)}


# ------------------------------------------------------------------------------------------------------
# the CUDA arm
# ------------------------------------------------------------------------------------------------------
def max_over_ranks(values, world: int, device=None):
    """The timing rule of the bench contract: every rank's device time, reduced with MAX over the ranks.

    With world == 1 (or no process group) the values come back unchanged.  Works on whatever backend the default
    process group uses (nccl in the bench, gloo in the CPU test).
    """
    if world <= 1:
        return [float(v) for v in values]
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(v) for v in values], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(v) for v in t.cpu()]


def aggregate_value(n_per_rank: int, world: int, steps: int, total_ms: float) -> float:
    """Whole-job throughput of N independent replicas: units all ranks processed / max-over-ranks time."""
    return world * n_per_rank * steps / (total_ms * 1e-3)


def run_ours(args):
    import torch
    import torch.distributed as dist

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- libbonsai has no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    from paper_1204_2280_b200 import Bonsai
    from paper_1204_2280_b200.bonsai import measure_fp32_peak
    W, n, theta, eps = _workload(args.workload)
    pm = W.plummer(n)
    peaks = {}
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            peaks = json.load(f)
    except OSError:
        pass

    stream = torch.cuda.Stream(dev)
    b = Bonsai(n, ncrit=args.ncrit, group_mode=args.group_mode, group_cell=args.group_cell, device=dev, stream=stream)
    d_pm = torch.from_numpy(pm).to(dev)
    d_out = torch.zeros((n, 4), dtype=torch.float32, device=dev)
    h_pm = torch.from_numpy(pm).pin_memory()
    h_out = torch.zeros((n, 4), dtype=torch.float32).pin_memory()
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    def flush_l2():
        with torch.cuda.stream(stream):
            flush.fill_(1)

    def one_step():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        flush_l2()
        e0.record(stream)
        b.step(d_pm, theta, eps, None, d_out)
        e1.record(stream)
        return e0, e1

    def one_step_host():
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        flush_l2()
        e0.record(stream)
        b.step_host(h_pm, theta, eps, None, h_out)   # blocking: returns after the D2H copy
        e1.record(stream)
        return e0, e1

    sampler = ClockSampler(local_rank) if rank == 0 else None   # started early: nvidia-smi takes a moment to come up
    b.set_timing(False)
    for _ in range(args.warmup):
        one_step()
        b.sync()
    # ---- timed region: exactly K steps, device-resident inputs, library un-instrumented ----
    barrier()
    launches0 = b.launch_count()
    t_wall0 = time.perf_counter()
    step_ms = []
    for _ in range(args.steps):
        e0, e1 = one_step()
        b.sync()
        step_ms.append(e0.elapsed_time(e1))
    barrier()
    t_wall1 = time.perf_counter()
    launches = b.launch_count() - launches0
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    sum_pp, sum_pc = b.interaction_totals()
    total_ms = float(sum(step_ms))

    # ---- the same K steps with the library's stage events on: per-stage split, walk time of the roofline ----
    b.set_timing(True)
    one_step(); b.sync(); b.stage_ms()
    inst_ms, stage_ms = [], []
    for _ in range(args.steps):
        e0, e1 = one_step()
        b.sync()
        inst_ms.append(e0.elapsed_time(e1))
        stage_ms.append(b.stage_ms())
    b.set_timing(False)

    # ---- end to end through the host-buffer call ----
    for _ in range(min(args.warmup, 2)):
        one_step_host()
    barrier()
    e2e_ms = []
    for _ in range(args.steps):
        e0, e1 = one_step_host()
        torch.cuda.synchronize(dev)
        e2e_ms.append(e0.elapsed_time(e1))
    barrier()
    e2e_total_ms = float(sum(e2e_ms))

    # ---- context only: the same step with the tight particle-box MAC (row f3, R28) ----
    variant = None
    if rank == 0 and world == 1:
        bt = Bonsai(n, ncrit=args.ncrit, group_mode=args.group_mode, group_cell=args.group_cell, device=dev, stream=stream,
                    mac_mode=1)
        for _ in range(3):
            flush_l2(); bt.step(d_pm, theta, eps, None, d_out); bt.sync()
        ms = []
        for _ in range(min(args.steps, 5)):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            flush_l2(); e0.record(stream); bt.step(d_pm, theta, eps, None, d_out); e1.record(stream); bt.sync()
            ms.append(e0.elapsed_time(e1))
        tpp, tpc = bt.interaction_totals()
        variant = {"ms_per_step": float(np.mean(ms)), "value": n / (float(np.mean(ms)) * 1e-3), "pp_per_particle": tpp / n,
                   "pc_per_particle": tpc / n,
                   "note": "mac_mode = 1 (tight particle-box MAC, R28): same theta, force error against direct summation "
                           "within 3 % of the geometric MAC's (tests/test_gpu_mac.py); not the headline configuration"}
        bt.close()

    total_ms, e2e_total_ms = max_over_ranks([total_ms, e2e_total_ms], world, dev)

    if rank == 0:
        ms_per_step = total_ms / args.steps
        value = aggregate_value(n, world, args.steps, total_ms)
        e2e_value = aggregate_value(n, world, args.steps, e2e_total_ms)
        st = {k: float(np.mean([s[k] for s in stage_ms])) for k in stage_ms[0] if k != "integrate"}
        walk_ms = st["walk"]
        flop = FLOP_PP * sum_pp + FLOP_PC * sum_pc
        sm_max = (clocks or {}).get("sm_max_mhz") or peaks.get("sm_max_mhz") or 1965.0
        n_sms = torch.cuda.get_device_properties(dev).multi_processor_count
        peak_tf = n_sms * FP32_LANES_PER_SM * 2 * sm_max * 1e6 / 1e12
        achieved_tf = flop / (walk_ms * 1e-3) / 1e12
        with torch.cuda.stream(stream):
            peak_ffma2 = measure_fp32_peak(True, 40000, stream)
            peak_ffma = measure_fp32_peak(False, 40000, stream)
        peak_meas = max(peak_ffma2, peak_ffma)
        hbm = peaks.get("hbm_gbs", 6650.0)
        hbm_src = "measured" if "hbm_gbs" in peaks else "fallback"
        stages = {}
        for k, v in st.items():
            ent = {"ms": v, "share": v / sum(st.values())}
            if k in ALG_BYTES and v > 0:
                gbs = ALG_BYTES[k](args) * n / (v * 1e-3) / 1e9
                ent.update({"alg_bytes_per_particle": ALG_BYTES[k](args), "alg_gbs": gbs, "hbm_frac": gbs / hbm})
            stages[k] = ent
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "n": n, "theta": theta, "eps": eps, "nleaf": 16,
                       "ncrit": args.ncrit, "group_mode": args.group_mode, "group_cell": args.group_cell},
            "notes": {"parallelism": "replicas only (no data-path collective)",
                      "l2": f"flushed between steps ({L2_FLUSH_BYTES >> 20} MiB fill, outside the event pair)",
                      "paper_context": "GTX480: > 2.8e6 particles/s (PAPER.md:14), other hardware",
                      "groups": "group_mode 2 = runs of 64 sorted particles inside cells of <= group_cell particles: "
                                "full lanes, but more interactions than tree-cell groups (group_mode 0), whose "
                                "survey figure is 88.2 kflop per particle (SURVEY.md 8(d)) against "
                                "roofline.flop_per_particle here; particles/s is the metric, the trade was measured"},
            "clocks": clocks,
            "e2e": {"value": e2e_value, "unit": UNIT, "ms_per_step": e2e_total_ms / args.steps,
                    "h2d_bytes_per_step": 16 * n, "d2h_bytes_per_step": 16 * n},
            "gpu_launches": int(launches),
            "instrumented_ms_per_step": float(np.mean(inst_ms)),
            "roofline": {"kernel": "k_walk", "bound": "alu", "achieved": achieved_tf, "peak": peak_tf,
                         "unit": "TFLOP/s", "frac": achieved_tf / peak_tf,
                         "peak_measured": peak_meas, "frac_of_measured": achieved_tf / peak_meas,
                         "peak_measured_source": f"bonsai_measure_fp32_peak in this process: FFMA2 {peak_ffma2:.2f}, "
                                                 f"FFMA {peak_ffma:.2f} TFLOP/s (64 warps/SM, 8 chains, best of 3)",
                         "traffic": walk_traffic(args),
                         "peak_source": f"derived: {n_sms} SMs x {FP32_LANES_PER_SM} FP32 lanes x 2 flop x "
                                        f"{sm_max:.0f} MHz (clocks.max.sm); no fp32 entry in MEASURED_PEAKS.json",
                         "flop_convention": "20 per p-p, 63 per p-c (FMA = 2, rsqrt = 1)",
                         "flop_per_particle": flop / n, "flop_per_particle_tree_cell_groups_survey": 88.2e3,
                         "walk_ms": walk_ms, "walk_share_of_step": walk_ms / sum(st.values()),
                         "interactions_per_s": (sum_pp + sum_pc) / (walk_ms * 1e-3),
                         "pp_per_particle": sum_pp / n, "pc_per_particle": sum_pc / n,
                         "hbm_peak_gbs": hbm, "hbm_peak_source": hbm_src},
            "stages": stages,
            "variants": {"tight_mac": variant},
        }
        if world == 1 and not args.no_cpu_baseline:
            line["cpu_baseline"] = cpu_baseline(pm, theta, eps, args.ncrit, args.group_mode, args.group_cell)
            line["cpu_baseline_all_cores"] = cpu_baseline_all_cores(pm, theta, eps, args.ncrit, args.group_mode,
                                                                    args.group_cell)
        print(json.dumps(line), flush=True)
    b.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    return 0


# Algorithmic bytes per particle of the HBM-bound stages (SURVEY.md section 8(d) floors):
#   keys: 16 in + 3 key words out; sort: P pair passes (P = 4 up to n = 2^23, 5 up to 2^25, else 6: the library's rule,
#   csrc/sort.cu sort_first_pass) x (8 in + 8 out), minus the index read of the first pass (iota) and the key write of
#   the last; reorder: perm + record in, record + 3 key words out,
#   plus the tie check re-reading the hi and mid words; build: the single-pass floor, 12 (keys once) + 4 (cell
#   records, 0.23 cells x 16 B); groups: positions once + one box per group; multipoles: positions once + 0.23 cells
#   x 48 B out + the children's records re-read by the internal cells (~0.05 x 48 B) = 30.
def sort_passes(a):
    n = _workload(a.workload)[1]
    return 4 if n <= (1 << 23) else 5 if n <= (1 << 25) else 6


ALG_BYTES = {
    "bbox": lambda a: 16, "keys": lambda a: 28, "sort": lambda a: sort_passes(a) * 16 - 8, "reorder": lambda a: 48 + 8,
    "build": lambda a: 16, "groups": lambda a: 16 + 24 / a.ncrit, "multipoles": lambda a: 30,
}


def walk_traffic(args):
    """roofline.traffic: dram__bytes_read.sum + dram__bytes_write.sum of one k_walk launch, from the committed `ncu
    --set full` capture profiles/walk_traffic.json -- valid only for the kernel it was taken from, so it is keyed by
    the SHA-256 of the walk's sources and by the workload; anything else reports null (never a stale number)."""
    import hashlib
    try:
        with open(os.path.join(ROOT, "profiles", "walk_traffic.json")) as f:
            cap = json.load(f)
        h = hashlib.sha256()
        for rel in cap["sources"]:
            with open(os.path.join(ROOT, rel), "rb") as f:
                h.update(f.read())
    except (OSError, KeyError, ValueError):
        return None
    key = [args.workload, args.ncrit, args.group_mode, args.group_cell]
    if h.hexdigest() != cap.get("sources_sha256") or key != cap.get("config"):
        return None
    return cap["dram_bytes_read"] + cap["dram_bytes_write"]


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--workload", default="plummer_4m")
    ap.add_argument("--ncrit", type=int, default=64)
    ap.add_argument("--group-mode", dest="group_mode", type=int, default=2)
    ap.add_argument("--group-cell", dest="group_cell", type=int, default=512)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
