"""Measurements of the BASELINE.json configurations that are not the bench line (python -m paper_1204_2280_b200.report).

  configs[1]  N = 2^18: theta sweep {0.3, 0.5, 0.75, 1.0}, interactions per particle and walk time
  configs[2]  N = 2^20: 8 KDK leapfrog steps (dt = 1/1024, shared step, tree rebuilt every step) at theta = 0.5, 0.75
  configs[4]  N = 2^20: walk of an active subset (N/16, N/256; scattered and clustered) against the full walk,
              with the tree rebuilt and with the tree refreshed (bonsai_refresh_tree)
  scaling     N = 2^15 ... 2^22: time per stage (the paper's Fig. 2 quantity)
  merger      N = 2^20: the second workload (two Plummer spheres on approach) against the single sphere
  mac         N = 2^18: theta-error-cost table of the MAC variants (geometric / tight particle-box MAC, quadrupole /
              monopole-only), the error measured against the library's own theta = 0 walk (= direct summation)

Everything runs through the C-ABI binding on cuda:0 with seeded synthetic Plummer spheres; times are CUDA-event
stage times of the library (median of `--reps`), L2 not flushed between repetitions.  Prints one JSON document.
"""
from __future__ import annotations

import argparse
import json

import numpy as np
import torch

from . import Bonsai
from . import workloads as W


def _median_stage(b: Bonsai, fn, reps: int) -> dict:
    rows = []
    for _ in range(reps):
        fn()
        rows.append(b.stage_ms())
    return {k: float(np.median([r[k] for r in rows])) for k in rows[0]}


def theta_sweep(reps: int) -> dict:
    cfg = W.CONFIGS["plummer_256k"]
    n, eps = cfg["n"], cfg["eps"]
    pm = torch.from_numpy(W.plummer(n)).cuda()
    b = Bonsai(n)
    b.set_timing(True)
    out = {}
    for theta in cfg["theta_sweep"]:
        b.step(pm, theta, eps)
        b.sync()
        st = _median_stage(b, lambda: b.step(pm, theta, eps), reps)
        pp, pc = b.interaction_totals()
        out[str(theta)] = {"pp_per_particle": pp / n, "pc_per_particle": pc / n, "walk_ms": st["walk"],
                           "step_ms": sum(v for k, v in st.items() if k != "integrate")}
    return {"n": n, "eps": eps, "by_theta": out}


def leapfrog(reps: int) -> dict:
    cfg = W.CONFIGS["plummer_1m"]
    n, eps, dt, steps = cfg["n"], cfg["eps"], 1.0 / 1024, 8
    pm_h, vel_h = W.plummer(n, with_velocities=True)
    v4 = np.zeros((n, 4), np.float32)
    v4[:, :3] = vel_h
    res = {}
    for theta in (0.5, 0.75):
        pm, vel = torch.from_numpy(pm_h).cuda(), torch.from_numpy(v4).cuda()
        b = Bonsai(n)
        acc = b.step(pm, theta, eps).clone()
        d0 = b.diagnostics(pm, vel, acc).cpu().numpy()
        b.leapfrog_step(pm, vel, acc, theta, eps, dt)            # warm-up step (counts as step 1 of the run)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        b.sync()
        with torch.cuda.stream(b.stream):
            e0.record()
        for _ in range(steps - 1):
            b.leapfrog_step(pm, vel, acc, theta, eps, dt)
        with torch.cuda.stream(b.stream):
            e1.record()
        b.sync()
        d1 = b.diagnostics(pm, vel, acc).cpu().numpy()
        ms = e0.elapsed_time(e1) / (steps - 1)
        res[str(theta)] = {"ms_per_step": ms, "particle_steps_per_s": n / (ms * 1e-3),
                           "rel_energy_drift_8_steps": float(abs((d1[0] + d1[1]) / (d0[0] + d0[1]) - 1.0))}
    return {"n": n, "eps": eps, "dt": dt, "steps": steps, "by_theta": res}


def block_step(reps: int) -> dict:
    cfg = W.CONFIGS["plummer_1m"]
    n, eps, theta = cfg["n"], cfg["eps"], cfg["theta"]
    pm_h, vel_h = W.plummer(n, with_velocities=True)
    v4 = np.zeros((n, 4), np.float32)
    v4[:, :3] = vel_h
    pm, vel = torch.from_numpy(pm_h).cuda(), torch.from_numpy(v4).cuda()
    b = Bonsai(n)
    b.set_timing(True)
    out = b.step(pm, theta, eps)
    b.sync()
    full = _median_stage(b, lambda: b.step(pm, theta, eps, out=out), reps)
    pre = sum(v for k, v in full.items() if k not in ("walk", "integrate"))
    res = {"n": n, "theta": theta, "full_walk_ms": full["walk"], "full_pre_walk_ms": pre, "subsets": {}}
    for pattern in ("clustered", "scattered"):
        for frac in (16, 256):
            mask = torch.from_numpy(W.active_mask(pm_h, n // frac, pattern)).cuda()
            st = _median_stage(b, lambda: b.step(pm, theta, eps, mask, out=out), reps)
            res["subsets"][f"{pattern}_N/{frac}"] = {
                "walk_ms": st["walk"], "groups_ms": st["groups"], "walk_time_reduction": full["walk"] / st["walk"],
                "ideal": frac}
    # refreshed tree instead of a rebuild: drift a little, refresh, recompute multipoles, walk the clustered N/16 subset
    mask = torch.from_numpy(W.active_mask(pm_h, n // 16, "clustered")).cuda()

    def refreshed():
        b.drift(pm, vel, 1.0 / 1024)
        b.refresh_tree()
        b.compute_multipoles()
        b.walk(theta, eps, mask, out=out)

    st = _median_stage(b, refreshed, reps)
    res["refreshed_clustered_N/16"] = {"reorder_ms": st["reorder"], "groups_ms": st["groups"],
                                       "multipoles_ms": st["multipoles"], "walk_ms": st["walk"],
                                       "step_ms": st["reorder"] + st["groups"] + st["multipoles"] + st["walk"],
                                       "rebuild_step_ms": pre + res["subsets"]["clustered_N/16"]["walk_ms"]}
    return res


def block_ticks(reps: int) -> dict:
    """bonsai_block_tick end to end (R26, R27, R30): ms per tick over one full cycle of
    2^kmax ticks at N = 2^20 with the tree rebuilt every tick, refreshed every tick, or rebuilt when the device says so,
    next to the all-active tick (kmax = 0) -- the tick-time reduction to hold against N / N_active."""
    del reps
    cfg = W.CONFIGS["plummer_1m"]
    n, eps, theta = cfg["n"], cfg["eps"], cfg["theta"]
    eta, dt_max, kmax = 0.3, 1.0 / 32, 4      # rungs 0 (halo) .. 4 (core) all populated on the Plummer sphere
    pm_h, vel_h = W.plummer(n, with_velocities=True)
    v4 = np.zeros((n, 4), np.float32)
    v4[:, :3] = vel_h
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    res = {"n": n, "theta": theta, "eta": eta, "dt_max": dt_max, "kmax": kmax, "modes": {}}
    for label, rebuild in (("all_active_kmax0", 1), ("rebuild", 1), ("refresh", 0), ("device_decides", -1)):
        pm, vel = torch.from_numpy(pm_h).cuda(), torch.from_numpy(v4).cuda()
        b = Bonsai(n)
        acc = b.step(pm, theta, eps).clone()
        km = 0 if label == "all_active_kmax0" else kmax
        rung = b.timestep_rungs(acc, eta, eps, dt_max, km)
        cycle = 1 << km
        n_ticks = 2 * cycle if km else 8
        rows = []
        for tick in range(n_ticks):                      # the first cycle is warm-up (and gives `refresh` its tree)
            n_act = int(b.active_mask(rung, km, tick + 1).sum())         # a host read, outside the event pair
            rb = 1 if (tick == 0 and rebuild == 0) else rebuild
            e0.record()
            b.block_tick(pm, vel, acc, rung, tick, theta, eps, eta, dt_max, km, rebuild=rb)
            e1.record()
            e1.synchronize()
            if tick >= n_ticks // 2:
                rows.append((e0.elapsed_time(e1), n_act))
        ms = [r[0] for r in rows]
        act = [r[1] for r in rows]
        res["modes"][label] = {"ticks_timed": len(rows), "ms_per_tick_mean": float(np.mean(ms)), "ms_per_tick_min": float(min(ms)),
                               "ms_per_tick_max": float(max(ms)), "ticks_per_s": 1e3 * len(ms) / float(sum(ms)),
                               "n_active_mean": float(np.mean(act)), "n_over_n_active": n / max(float(np.mean(act)), 1.0),
                               "ms_by_tick": [round(x, 4) for x in ms], "n_active_by_tick": act}
        if rebuild < 0:
            res["modes"][label]["rebuild_stats"] = b.rebuild_stats()
        b.sync()
        del b
    full = res["modes"]["all_active_kmax0"]["ms_per_tick_mean"]
    for label, d in res["modes"].items():
        d["tick_time_reduction"] = full / d["ms_per_tick_mean"]
    return res


def scaling(reps: int) -> dict:
    rows = {}
    beyond = {"plummer_16m": dict(n=1 << 24, eps=0.0008, theta=0.75)}  # four times the paper's largest N (working set 4x L2)
    for name in ("plummer_32k", "plummer_256k", "plummer_1m", "plummer_4m", "plummer_16m"):
        cfg = W.CONFIGS.get(name) or beyond[name]
        n, eps, theta = cfg["n"], cfg["eps"], cfg["theta"]
        pm = torch.from_numpy(W.plummer(n)).cuda()
        b = Bonsai(n)
        b.set_timing(True)
        b.step(pm, theta, eps)
        b.sync()
        st = _median_stage(b, lambda: b.step(pm, theta, eps), reps)
        pp, pc = b.interaction_totals()
        st.pop("integrate", None)
        total = sum(st.values())
        rows[name] = {"n": n, "stage_ms": st, "step_ms": total, "particles_per_s": n / (total * 1e-3),
                      "walk_share": st["walk"] / total, "pp_per_particle": pp / n, "pc_per_particle": pc / n}
        # the un-instrumented step: replayed CUDA graph (bonsai_step) against kernel-by-kernel launches
        b.set_timing(False)
        out = torch.zeros((n, 4), dtype=torch.float32, device="cuda")
        for tag, bb in (("step_ms_graph", b), ("step_ms_no_graph", Bonsai(n, use_graph=False))):
            for _ in range(3):
                bb.step(pm, theta, eps, None, out)
            bb.sync()
            ms = []
            for _ in range(max(reps, 5)):
                e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                e0.record(bb.stream)
                bb.step(pm, theta, eps, None, out)
                e1.record(bb.stream)
                bb.sync()
                ms.append(e0.elapsed_time(e1))
            rows[name][tag] = float(np.median(ms))
        del b
    return rows


def merger(reps: int) -> dict:
    """Second workload: two Plummer spheres (mass ratio 3) on approach, N = 2^20, against the single sphere."""
    n, eps, theta = 1 << 20, 0.0025, 0.75
    res = {}
    for name, pm_h in (("plummer", W.plummer(n)), ("merger", W.merger(n)[0])):
        pm = torch.from_numpy(pm_h).cuda()
        b = Bonsai(n)
        b.set_timing(True)
        b.step(pm, theta, eps)
        b.sync()
        st = _median_stage(b, lambda: b.step(pm, theta, eps), reps)
        pp, pc = b.interaction_totals()
        st.pop("integrate", None)
        res[name] = {"step_ms": sum(st.values()), "walk_ms": st["walk"], "pp_per_particle": pp / n,
                     "pc_per_particle": pc / n, "n_cells": b.cells(False).n_cells, "n_groups": b.groups().n_groups}
        del b
    return {"n": n, "eps": eps, "theta": theta, "by_workload": res}


def mac_variants(reps: int) -> dict:
    """Row f3 (theta "sets the trade-off between speed and accuracy"): for mac_mode in {geometric, tight} and
    order in {quadrupole, monopole}, the theta sweep of configs[1] at N = 2^18 -- interactions per particle, walk time,
    and the force error of 4096 scattered sinks against the SAME library's theta = 0 walk of those sinks (theta = 0
    opens everything: direct summation through the tree; the parity tests pin it to the oracle's direct sum)."""
    cfg = W.CONFIGS["plummer_256k"]
    n, eps = cfg["n"], cfg["eps"]
    pm_h = W.plummer(n)
    pm = torch.from_numpy(pm_h).cuda()
    mask_h = W.active_mask(pm_h, 4096, "scattered")
    mask = torch.from_numpy(mask_h).cuda()
    sel = torch.from_numpy(np.nonzero(mask_h)[0]).cuda()
    b0 = Bonsai(n)
    exact = b0.step(pm, 0.0, eps, mask)[sel].double()
    b0.sync()
    rows = {}
    for mac_mode, mac_name in ((0, "geometric"), (1, "tight")):
        for order, order_name in ((2, "quadrupole"), (1, "monopole")):
            b = Bonsai(n, mac_mode=mac_mode, order=order)
            b.set_timing(True)
            by_theta = {}
            for theta in cfg["theta_sweep"]:
                out = b.step(pm, theta, eps)
                b.sync()
                st = _median_stage(b, lambda: b.step(pm, theta, eps), reps)
                pp, pc = b.interaction_totals()
                got = out[sel].double()
                err = (torch.linalg.norm(got[:, :3] - exact[:, :3], dim=1) / torch.linalg.norm(exact[:, :3], dim=1)).cpu().numpy()
                by_theta[str(theta)] = {"acc_err_median": float(np.median(err)), "acc_err_p99": float(np.quantile(err, 0.99)),
                                        "pp_per_particle": pp / n, "pc_per_particle": pc / n, "walk_ms": st["walk"],
                                        "multipoles_ms": st["multipoles"]}
            rows[f"{mac_name}/{order_name}"] = by_theta
            del b
    return {"n": n, "eps": eps, "sinks_compared": 4096, "error_reference": "theta = 0 walk of the same library",
            "variants": rows}


def parity_summary(path: str) -> None:
    """`--parity FILE`: the figures the `-m gpu` tests recorded (tests/test_gpu_parity.record -> gpurun_out/parity_r3.jsonl)
    as markdown tables on stdout.  Needs no GPU."""
    rows = [json.loads(ln) for ln in open(path) if ln.strip()]
    walk = [r for r in rows if "count_frac" in r]
    iso = [r for r in rows if r["test"] == "walk on the GPU's cell records"]
    mp = [r for r in rows if r["test"] == "multipoles"]
    print("# Parity figures measured by the `-m gpu` tests (CUDA path vs the CPU oracle)\n")
    print(f"Command: `python -m pytest tests -m gpu -q && python -m paper_1204_2280_b200.report --parity {path}`; {len(rows)} records.\n")
    print("## Walk: full-size configurations and named cases (sinks compared = N: every sink of the configuration)\n")
    print("| case | N | theta | sinks compared | counts identical | mismatches (all borderline) | acc max | acc median | pot max | pot median |")
    print("|---|---|---|---|---|---|---|---|---|---|")
    for r in walk:
        if r["test"] in ("check_walk", "check_walk_sampled"):
            continue
        print(f"| {r['test']} | {r['n']} | {r.get('theta', '')} | {r.get('sinks_sampled', r.get('n_checked'))} | "
              f"{r['count_frac']:.6f} | {r['n_borderline_mismatch']} | {r['acc_max']:.2e} | {r['acc_med']:.2e} | "
              f"{r['pot_max']:.2e} | {r['pot_med']:.2e} |")
    deep = [r for r in walk if r.get("deep_tree")]
    walk = [r for r in walk if not r.get("deep_tree")]
    rest = [r for r in walk if r["test"] in ("check_walk", "check_walk_sampled")]
    if deep:
        print(f"\nClumps far below the 13th level (sort-pass tests, {len(deep)} calls, trees up to 26 levels deep): one "
              f"ulp(fp32) of a centre-of-mass coordinate is 1e-3 of a cell side there, so opening tests outside the oracle's "
              f"borderline margin may flip; required end to end: counts identical for >= 98 % of the sinks (lowest "
              f"{min(r['count_frac'] for r in deep):.5f}, {sum(r['n_borderline_mismatch'] for r in deep)} mismatching "
              f"sinks in total) and every mismatching sink within 1e-2 of the oracle.")
    if iso:
        print(f"\nThe walk in isolation (oracle walking the GPU's exported cell records, {len(iso)} calls, "
              f"{sum(r['sinks'] for r in iso)} sinks): {sum(r['count_mismatches'] for r in iso)} count mismatches, worst acc max "
              f"{max(r['acc_max'] for r in iso):.2e}.")
    if rest:
        print(f"\nAll other walk comparisons ({len(rest)} calls, N = {min(r['n'] for r in rest)} .. {max(r['n'] for r in rest)}): "
              f"lowest identical-count fraction {min(r['count_frac'] for r in rest):.5f}, "
              f"{sum(r['n_borderline_mismatch'] for r in rest)} mismatching sinks in total (every one in an oracle-flagged "
              f"borderline group), worst acc max {max(r['acc_max'] for r in rest):.2e}, worst acc median "
              f"{max(r['acc_med'] for r in rest):.2e}, worst pot max {max(r['pot_max'] for r in rest):.2e}.")
    if mp:
        print("\n## Multipoles: <= 1 ulp(fp32); fraction of values that differ at all\n")
        print("| N | M, COM | delta | second moments | largest difference (ulp) |")
        print("|---|---|---|---|---|")
        seen = set()
        for r in sorted(mp, key=lambda r: -r["n"]):
            if r["n"] in seen or r["n"] < 30000:
                continue
            seen.add(r["n"])
            print(f"| {r['n']} | {r['com_m_frac_differing']:.2e} | {r['delta_frac_differing']:.2e} | "
                  f"{r['quad_frac_differing']:.2e} | {max(r['com_m_max_ulp'], r['delta_max_ulp'], r['quad_max_ulp'])} |")
        print(f"\nOver all {len(mp)} multipole comparisons: largest difference "
              f"{max(max(r['com_m_max_ulp'], r['delta_max_ulp']) for r in mp)} ulp on M / COM / delta; second moments above "
              f"the fp64 noise floor <= 1 ulp (diagonal) or within 1e-7 of the largest diagonal moment (off-diagonal).")
    bt = [r for r in rows if r["test"] == "block_ticks"]
    if bt:
        print("\n## Block time-steps: 8 ticks, both sides independent\n")
        for r in bt:
            print(f"* rebuild every {r['rebuild_every']} tick(s): rung arrays differ for {r['rung_flips_after_8_ticks']:.2e} "
                  f"of the particles after 8 ticks; |dx| median {r['dx_median']:.1e}, max {r['dx_max']:.1e}; "
                  f"|dv|/v_rms median {r['dv_median_over_vrms']:.1e}, max {r['dv_max_over_vrms']:.1e}")



def markdown(doc: dict) -> str:
    """The tables of profiles/r2_configs.md from the dictionary main() prints (`--markdown FILE`)."""
    o = ["# The BASELINE.json configurations that are not the bench line\n",
         "Command: `python -m paper_1204_2280_b200.report --markdown FILE > FILE.json`.  One B200, seeded Plummer spheres, "
         "CUDA-event stage times of the library (median of 5), L2 not flushed between repetitions.\n"]
    if "theta_sweep" in doc:
        d = doc["theta_sweep"]
        o += [f"## configs[1]: N = {d['n']}, eps = {d['eps']}, theta sweep\n",
              "| theta | p-p per particle | p-c per particle | walk ms | step ms |", "|---|---|---|---|---|"]
        o += [f"| {th} | {r['pp_per_particle']:.0f} | {r['pc_per_particle']:.0f} | {r['walk_ms']:.3f} | {r['step_ms']:.3f} |"
              for th, r in d["by_theta"].items()]
        o.append("")
    if "leapfrog" in doc:
        d = doc["leapfrog"]
        o += [f"## configs[2]: N = {d['n']}, eps = {d['eps']}, {d['steps']} KDK steps, dt = {d['dt']}, tree rebuilt every step "
              "(bonsai_leapfrog_step, graph replay)\n",
              "| theta | ms per step | particle-steps per s | relative energy drift over the run |", "|---|---|---|---|"]
        o += [f"| {th} | {r['ms_per_step']:.3f} | {r['particle_steps_per_s']:.3e} | {r['rel_energy_drift_8_steps']:.2e} |"
              for th, r in d["by_theta"].items()]
        o.append("")
    if "block_step" in doc:
        d = doc["block_step"]
        o += [f"## configs[4]: N = {d['n']}, theta = {d['theta']}, full rebuild, walk of an active subset (P:L32)\n",
              f"Full walk {d['full_walk_ms']:.3f} ms; stages before the walk {d['full_pre_walk_ms']:.3f} ms.\n",
              "| subset | walk ms | groups stage ms | walk-time reduction | N / N_active |", "|---|---|---|---|---|"]
        o += [f"| {k} | {r['walk_ms']:.4f} | {r['groups_ms']:.3f} | {r['walk_time_reduction']:.1f} x | {r['ideal']} |"
              for k, r in d["subsets"].items()]
        r = d.get("refreshed_clustered_N/16")
        if r:
            o.append(f"\nRefreshed tree (bonsai_refresh_tree, R25) instead of a rebuild, clustered N/16: reorder "
                     f"{r['reorder_ms']:.3f} + groups {r['groups_ms']:.3f} + multipoles {r['multipoles_ms']:.3f} + walk "
                     f"{r['walk_ms']:.3f} = {r['step_ms']:.3f} ms against {r['rebuild_step_ms']:.3f} ms with a rebuild.")
        o.append("")
    if "scaling" in doc:
        names = ("bbox", "keys", "sort", "reorder", "build", "groups", "multipoles", "walk")
        o += ["## Scaling with N (the paper's Fig. 2 quantity, P:L48), theta = 0.75\n",
              "| N | " + " | ".join(names) + " | stage sum ms | step ms, graph replay | step ms, kernel by kernel | "
              "particles/s (graph) | walk share |", "|---|" + "---|" * (len(names) + 5)]
        for r in doc["scaling"].values():
            o.append(f"| {r['n']} | " + " | ".join(f"{r['stage_ms'][k]:.3f}" for k in names) +
                     f" | {r['step_ms']:.3f} | {r['step_ms_graph']:.3f} | {r.get('step_ms_no_graph', float('nan')):.3f} | "
                     f"{r['n'] / r['step_ms_graph'] * 1e3:.3e} | {100 * r['walk_share']:.0f} % |")
        o.append("")
    if "merger" in doc:
        d = doc["merger"]["by_workload"]
        m, pl = d["merger"], d["plummer"]
        o += [f"## Second workload (row f4): two Plummer spheres, mass ratio 3, on approach, N = {doc['merger']['n']}\n",
              f"merger {m['step_ms']:.3f} ms per step ({m['n_cells']} cells, {m['n_groups']} groups, {m['pp_per_particle']:.0f} p-p + "
              f"{m['pc_per_particle']:.0f} p-c per particle) against {pl['step_ms']:.3f} ms for the single sphere "
              f"({pl['n_cells']} cells, {pl['n_groups']} groups).\n"]
    if "mac" in doc:
        d = doc["mac"]
        o += [f"## Row f3: MAC variants, N = {d['n']} (error of {d['sinks_compared']} sinks against: {d['error_reference']})\n",
              "| variant | theta | median force error | 99th percentile | p-p per particle | p-c per particle | walk ms |",
              "|---|---|---|---|---|---|---|"]
        for name, by in d["variants"].items():
            o += [f"| {name} | {th} | {r['acc_err_median']:.2e} | {r['acc_err_p99']:.2e} | {r['pp_per_particle']:.0f} | "
                  f"{r['pc_per_particle']:.0f} | {r['walk_ms']:.3f} |" for th, r in by.items()]
        o.append("")
    if "block_ticks" in doc:
        d = doc["block_ticks"]
        o += [f"## bonsai_block_tick end to end, N = {d['n']}, kmax = {d['kmax']} (one cycle of {1 << d['kmax']} ticks, after one warm-up cycle)\n",
              "| tree per tick | ms per tick (mean) | min | max | ticks/s | mean N_active | N / N_active | tick-time reduction vs all-active |",
              "|---|---|---|---|---|---|---|---|"]
        o += [f"| {k} | {r['ms_per_tick_mean']:.3f} | {r['ms_per_tick_min']:.3f} | {r['ms_per_tick_max']:.3f} | {r['ticks_per_s']:.0f} | "
              f"{r['n_active_mean']:.0f} | {r['n_over_n_active']:.1f} | {r['tick_time_reduction']:.2f} |" for k, r in d["modes"].items()]
        o.append("")
    return "\n".join(o)


def main() -> None:
    ap = argparse.ArgumentParser(description=__doc__, formatter_class=argparse.RawDescriptionHelpFormatter)
    ap.add_argument("--reps", type=int, default=5)
    ap.add_argument("--only", choices=("theta_sweep", "leapfrog", "block_step", "block_ticks", "scaling", "merger", "mac"), default=None)
    ap.add_argument("--markdown", default=None, help="also write the tables as markdown to this file")
    ap.add_argument("--from-json", dest="from_json", default=None,
                    help="render --markdown from an earlier JSON output instead of measuring (needs no GPU)")
    ap.add_argument("--parity", default=None, metavar="JSONL",
                    help="summarise the parity records of a `pytest -m gpu` run as markdown on stdout (needs no GPU)")
    args = ap.parse_args()
    if args.parity:
        parity_summary(args.parity)
        return
    if args.from_json:
        with open(args.from_json) as f:
            text = f.read()
        with open(args.markdown, "w") as f:
            f.write(markdown(json.loads(text[text.index("{"):])))
        return
    if not torch.cuda.is_available():
        raise SystemExit("report: no CUDA device -- libbonsai has no CPU fallback")
    parts = {"theta_sweep": theta_sweep, "leapfrog": leapfrog, "block_step": block_step, "block_ticks": block_ticks,
             "scaling": scaling,
             "merger": merger, "mac": mac_variants}
    doc = {k: f(args.reps) for k, f in parts.items() if args.only in (None, k)}
    print(json.dumps(doc, indent=1))
    if args.markdown:
        with open(args.markdown, "w") as f:
            f.write(markdown(doc))


if __name__ == "__main__":
    main()
