#!/usr/bin/env python
"""Benchmark of the hybrid symplectic step on B200 (contract: see DESIGN.md "Measurement").

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference] [--config 1]

A step = one full time step of BASELINE.json configs[1] (2048 massive bodies, order 2,
dt = 6 d): critical radii, kick + precheck, Sun kick, Kepler drift, encounter search,
grouping, Bulirsch-Stoer on the groups, Sun kick, kick.  Prints ONE JSON line.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402

METRIC = "fp64_pair_interactions_per_s"
UNIT = "ordered pair interactions/s"
FLOP_PER_INTERACTION = 20.0        # Nyland et al. convention, DESIGN.md "Rooflines"
FP64_NOMINAL_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12   # SMs x DFMA/clk/SM x 2 flop x max clock


def workload(cfg_id, rank=0, world=1, order=None):
    """The configuration of BASELINE.json; under world > 1 the particle and multi-system modes take a global
    workload world times as large (weak scaling) and this rank's shard of it (workloads.shard: no collective);
    the massive mode runs replicas."""
    if world > 1 and cfg_id == 2:
        w = workloads.shard(workloads.config2(n_test=1_000_000 * world), rank, world)
    elif world > 1 and cfg_id == 3:
        w = workloads.shard(workloads.config3(n_systems=4096 * world), rank, world)
    else:
        w = workloads.CONFIGS[cfg_id]()
    if order is not None:
        w = dict(w, order=int(order))
    name = {0: "cfg0 massive N=15", 1: "cfg1 planetesimal disc N=2048 massive, order 2, dt=6d",
            2: "cfg2 8 massive + 1e6 test particles", 3: "cfg3 4096 systems x 16",
            4: "cfg4 annulus N=2048 order %d, dt=2d" % w["order"]}[cfg_id]
    return w, name


def interactions_per_step(w, merged=True):
    # force evaluations the library makes per step: 2 per map, adjacent kicks of the substeps of one step merged
    # (modes 0 and 2): 2, 4, 8 for orders 2, 4, 6; the particle mode keeps them apart
    maps = {2: 1, 4: 3, 6: 7}[w["order"]]
    nm, evals = w["n_massive"], (2 * maps if (w["mode"] == 1 or not merged) else maps + 1)   # the oracle never merges
    if w["mode"] == 2:
        per = w["n_systems"] * nm * (nm - 1)
    else:
        # the massive bodies are replicated on every rank of a sharded run: counted once, on rank 0
        per = (nm * (nm - 1) if w.get("shard", (0,))[0] == 0 else 0) + w["n_test"] * nm
    return per * evals, evals


# --------------------------------------------------------------------------- clocks
class ClockSampler:
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.p, self.index = [], None, index

    def start(self):
        try:
            self.p = subprocess.Popen(["nvidia-smi", "--query-gpu=" + self.Q, "--format=csv,noheader,nounits",
                                       "-lms", "20", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.p = None

    def _read(self):
        for line in self.p.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.p:
            self.p.terminate()
        sm = [float(r[1]) for r in self.rows if len(r) >= 9 and r[1].replace(".", "").isdigit()]
        mx = [float(r[2]) for r in self.rows if len(r) >= 9 and r[2].replace(".", "").isdigit()]
        reasons = set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            if len(r) >= 9:
                for k, nm in enumerate(names):
                    if r[5 + k].lower().startswith("active"):
                        reasons.add(nm)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# --------------------------------------------------------------------------- reference arm
def oracle_rate(w, budget_s, max_steps):
    """Time the oracle as it stands on one host core; returns (interactions/s, steps, seconds)."""
    import oracle
    sim = oracle.Sim(w, cap=200000)
    per_step, _ = interactions_per_step(w, merged=False)
    sim.step(1)
    t0 = time.perf_counter()
    n = 0
    while n < max_steps:
        sim.step(1)
        n += 1
        if time.perf_counter() - t0 > budget_s:
            break
    dt = time.perf_counter() - t0
    return per_step * n / dt, n, dt


def lib_evals(w):
    """full force evaluations (all-pairs loops) the library makes per step: 2 per map in the particle mode; adjacent kicks
    of the maps of a step are one evaluation (modes 0, 2); in massive mode with N > 32 the opening kick of a step is
    none either (S2': it adds the sums the previous closing kick stored)"""
    maps = {2: 1, 4: 3, 6: 7}[w["order"]]
    if w["mode"] == 1:
        return 2 * maps
    return maps if (w["mode"] == 0 and w["n_massive"] > 32) else maps + 1


def timed_chunk(w):
    """steps per timed call: 1, except where the library runs all the steps of a call in ONE launch (multi-system mode and
    massive mode with N <= 16, multi_persist.cuh): there a timed call is 16 steps, L2 flushed between the calls"""
    return 16 if (w["mode"] == 2 or (w["mode"] == 0 and w["n_massive"] <= 16)) else 1


def config_dict(w, name, evals, world=1):
    """the `config` object of the JSON line: the benchmark configuration, the same object on both arms"""
    evals = lib_evals(w)
    return {"workload": name, "n_massive": w["n_massive"], "order": w["order"], "dt_days": w["dt"] / workloads.DAY,
            "force_evals_per_step": evals, "steps_per_timed_call": timed_chunk(w),
            "l2": "flushed (512 MiB fill) before every timed step",
            "parallelism": ("1 gpu" if world == 1 else "replicas only" if w["mode"] == 0 else
                            "particles sharded, massive bodies replicated, no collective" if w["mode"] == 1
                            else "systems sharded, no collective")}


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, name = workload(args.config, order=args.order)
    import oracle
    sim = oracle.Sim(w, cap=200000)
    sim.step(max(args.warmup, 0))                       # W untimed warm-up steps, as given
    per_step, evals = interactions_per_step(w, merged=False)
    t0 = time.perf_counter()
    n = 0
    while n < args.steps:                               # K timed steps, bounded to a few minutes
        sim.step(1)
        n += 1
        if time.perf_counter() - t0 > 240.0:
            break
    secs = time.perf_counter() - t0
    rate = per_step * n / secs
    sample = "%d full steps of %s (%.1f s) after %d warm-up steps" % (n, name, secs, args.warmup)
    cfg = config_dict(w, name, interactions_per_step(w)[1])      # the benchmark configuration: the CUDA arm's keys and values
    line = {
        "impl": "reference", "metric": METRIC, "value": rate, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "steps_timed": n, "ms_per_step": 1e3 * secs / n, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": cfg,
        "steps_per_s": n / secs,
        "cpu_baseline": {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "reference_arm": {"l2": "n/a (host cores)", "cores": 1, "force_evals_per_step": evals,
                          "note": "the oracle as it stands: single-threaded, never merges adjacent kicks"},
    }
    print(json.dumps(line))


# --------------------------------------------------------------------------- multi-rank glue
def reduce_max_and_sum(elapsed_s, units, backend_device):
    """max over ranks of the elapsed time, sum over ranks of the units (replicas, no data exchange)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()):
        return elapsed_s, units
    t = torch.tensor([elapsed_s], dtype=torch.float64, device=backend_device)
    u = torch.tensor([float(units)], dtype=torch.float64, device=backend_device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(u, op=dist.ReduceOp.SUM)
    return float(t.item()), float(u.item())


def pinned(torch, a):
    t = torch.empty(a.shape, dtype=torch.float64).pin_memory().numpy()
    t[...] = a
    return t


def measure(torch, G, dev, cfg_id, order, steps, warmup, rank, world, clocks=None, e2e_steps=200):
    """One configuration: K timed steps (L2 flushed between), the back-to-back run, the end-to-end leg through the host
    calls, the per-phase profile of a step and the rooflines of its dominant kernels.  Returns the JSON object."""
    w, name = workload(cfg_id, rank, world, order)
    per_step, evals = interactions_per_step(w)
    g = G.from_workload(w, device=str(dev))
    dt, order = w["dt"], w["order"]
    flush = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device=dev)   # > 126 MB L2

    def barrier():
        if world > 1:
            torch.distributed.barrier()
        torch.cuda.synchronize(dev)

    # ---- warm-up (also instantiates the CUDA graphs)
    g.step(max(warmup, 3), dt, order)
    g.step(16, dt, order)
    if clocks is not None:
        tw = time.perf_counter()
        while not clocks.rows and time.perf_counter() - tw < 3.0:      # keep the GPU busy until the sampler delivers (nvidia-smi
            g.fp64_probe()                                             # needs ~0.3 s to start); the probe leaves the state alone
    assert g.status() == 0
    c0 = g.counters()

    # ---- timed: K steps, timed with events on the library's stream, L2 flushed between the timed calls (timed_chunk)
    chunk = timed_chunk(w)
    steps = max(chunk, steps // chunk * chunk)
    barrier()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps // chunk)]
    with torch.cuda.stream(g.stream):
        for k in range(steps // chunk):
            flush.fill_(k & 255)               # evicts the state from L2; outside the timed events
            ev[k][0].record(g.stream)
            g.step(chunk, dt, order)
            ev[k][1].record(g.stream)
    barrier()
    ms = [a.elapsed_time(b) for a, b in ev]
    elapsed = sum(ms) * 1e-3
    c1 = g.counters()
    status = g.status()
    trace = g.bs_trace()                       # the groups of the last substep: the longest chain sets the step time
    # pair interactions the library evaluated per step (its own count of full force evaluations: adjacent kicks merged,
    # the opening kick of a step taken from the stored sums of the previous closing kick)
    evals = (c1["force_evals"] - c0["force_evals"]) / steps
    per_step = (c1["interactions"] - c0["interactions"]) / steps
    if w.get("shard", (0,))[0] != 0 and w["mode"] == 1:      # the replicated massive bodies are counted once, on rank 0
        per_step -= w["n_massive"] * (w["n_massive"] - 1) * evals

    # ---- back-to-back (state resident in L2, 16-step graphs): the production loop
    nres = max(16, (steps // 16) * 16)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(g.stream)
    g.step(nres, dt, order)
    e1.record(g.stream)
    barrier()
    resident_s = e0.elapsed_time(e1) * 1e-3
    if clocks is not None:
        tw = time.perf_counter()
        while len(clocks.rows) < 4 and time.perf_counter() - tw < 2.0:  # short runs: keep the load on until a few samples are in
            g.step(16, dt, order)
            g.fp64_probe()

    # ---- the phases of a step (plain launches with an event at every phase boundary), from the state the timed steps left
    c2 = g.counters()
    nprof = min(steps, 32)
    phases = g.profile_step(nprof, dt, order)
    c3 = g.counters()
    del flush

    # ---- end to end through the C-ABI with HOST buffers (pinned), copies inside the timed region
    xh, vh = pinned(torch, w["x"]), pinned(torch, w["v"])
    m0h, mh, rh = pinned(torch, w["m0"]), pinned(torch, w["m"]), pinned(torch, w["radius"])
    for _ in range(3):
        g.set_state_host(m0h, mh, rh, xh, vh); g.step(1, dt, order); g.get_state_host(xh, vh)
    ne2e = min(steps, e2e_steps)
    barrier()
    t0 = time.perf_counter()
    for _ in range(ne2e):
        g.set_state_host(m0h, mh, rh, xh, vh)
        g.step(1, dt, order)
        g.get_state_host(xh, vh)
    barrier()
    e2e_s = time.perf_counter() - t0
    h2d = 8 * (len(m0h) + 2 * g.ntot + 6 * g.ntot)
    d2h = 8 * 6 * g.ntot

    # ---- dominant kernels in isolation (CUDA events inside the library, on its stream)
    g.set_state(w["m0"], w["m"], w["radius"], w["x"], w["v"])
    peak_probe = g.fp64_probe()
    pk = os.path.join(ROOT, "MEASURED_PEAKS.json")
    hbm_peak = json.load(open(pk)).get("hbm_gbs") if os.path.exists(pk) else None
    hbm_src = "MEASURED_PEAKS.json hbm_gbs (measured copy bandwidth)" if hbm_peak else "fallback of B200_PROFILING.md"
    hbm_peak = hbm_peak or 6650.0
    tpath = os.path.join(ROOT, "profiles", "traffic.json")
    tab = json.load(open(tpath)) if os.path.exists(tpath) else {}
    maps = {2: 1, 4: 3, 6: 7}[order]
    nsteps_prof = c3["steps"] - c2["steps"]
    groups_ps = (c3["groups"] - c2["groups"]) / max(nsteps_prof, 1)
    acc_ps = (c3["bs_steps"] - c2["bs_steps"]) / max(nsteps_prof, 1)
    rej_ps = (c3["bs_rejects"] - c2["bs_rejects"]) / max(nsteps_prof, 1)
    # Bulirsch-Stoer (S7; "group-steps/s and FP64 pipe utilisation, no peak target"): the phase that sets
    # the step time.  in_step_ms = all Bulirsch-Stoer launches of a step, from the event profile.
    bs = {"kernel": "k_bs_warp + k_bs_cluster (+ k_bs_block / k_tp_bs / k_bs_multi)", "bound": "latency (dependent FP64 chains)",
          "in_step_ms": phases["bs"], "share_of_step": phases["bs"] / phases["total"] if phases["total"] else None,
          "groups_per_step": groups_ps, "accepted_steps_per_step": acc_ps, "rejected_attempts_per_step": rej_ps,
          "group_steps_per_s": acc_ps / (phases["bs"] * 1e-3) if phases["bs"] > 0 else None,
          "longest_chain": ({"group_size": int(trace[np.argmax(trace[:, 4]), 0]), "accepted": int(trace[np.argmax(trace[:, 4]), 2]),
                             "rejected": int(trace[np.argmax(trace[:, 4]), 3]), "us": float(trace[:, 4].max()) / 1965.0,
                             "note": "last substep of the timed run (genga_bs_trace), SM cycles at 1965 MHz"} if len(trace) else None),
          "fp64_pipe_pct_ncu": tab.get("fp64_pipe_pct", {}).get("bs"),
          "note": "time = the longest dependent chain of one group, not arithmetic: ncu's FP64-pipe share (profiles/) is the utilisation figure"}
    if w["mode"] == 0:
        kick_ms = g.time_kernel(0, 200, dt)
        inter = w["n_massive"] * (w["n_massive"] - 1)
        achieved = FLOP_PER_INTERACTION * inter / (kick_ms * 1e-3) / 1e12
        nk = maps + 1                                            # kick launches per step: `maps` full ones + the near-pair one of S2' (N > 32)
        kin = phases["kick"] / nk
        roof = {"bound": "alu", "kernel": "k_kick", "achieved": achieved, "peak": peak_probe,
                "unit": "TFLOP/s", "frac": achieved / peak_probe, "traffic": tab.get("k_kick"),
                "peak_source": "DFMA probe measured in this run (genga_fp64_probe); nominal %.1f = 148 SM x 64 DFMA/clk x 2 x 1.965 GHz" % FP64_NOMINAL_TFLOPS,
                "ms_per_launch": kick_ms, "interactions_per_launch": inter,
                "interactions_per_s": inter / (kick_ms * 1e-3),
                "flop_per_interaction": FLOP_PER_INTERACTION,
                "convention": "frac = 20 flop (Nyland et al., PAPER.md L242) x interactions / time / DFMA peak; the kernel issues 16 FP64 "
                              "instructions per interaction, fp64_issue_frac is its share of the FP64 issue slots",
                "fp64_issue_frac": 16.0 * 2.0 * inter / (kick_ms * 1e-3) / 1e12 / peak_probe,
                "fp64_pipe_pct_ncu": tab.get("fp64_pipe_pct", {}).get("k_kick"),
                # the same kernel as it runs inside a step: candidates recorded, exact pass writing the list, real h
                "in_step": {"ms_per_launch": kin, "launches_per_step": nk,
                            "frac": FLOP_PER_INTERACTION * inter / (kin * 1e-3) / 1e12 / peak_probe if kin > 0 else None,
                            "note": "from genga_profile_step (events around the kick launches of real steps, record = 1)"}}
        drift_ms = g.time_kernel(1, 200, dt)
        roof["drift"] = {"kernel": "k_drift", "ms_per_launch": drift_ms, "bodies": g.ntot,
                         "algorithmic_bytes": 144 * g.ntot,
                         "gbs": 144 * g.ntot / (drift_ms * 1e-3) / 1e9,
                         "note": "launch-latency bound at N = 2048 (295 KB)"}
        if w["n_massive"] <= 32:
            roof["note"] = ("N <= 32: the step runs k_tiny_front / k_tiny_back (one warp per half map) and is launch-latency "
                            "bound; k_kick and k_drift are timed alone here for reference only")
    elif w["mode"] == 1:
        # dominant kernel: k_tp_mid, ONE pass over the particle per step (closing half, opening half, drift, encounter search).
        # It is bound by FP64 issue, as SURVEY 8(d) predicts for a fused particle step; both rooflines are reported.
        nt = w["n_test"]
        mid_ms = g.time_kernel(5, 50, dt)
        front_ms = g.time_kernel(3, 50, dt)
        back_ms = g.time_kernel(4, 50, dt)
        step_ms = 1e3 * elapsed / steps
        FP64_PER_PARTICLE = 528.0          # FP64 instructions per particle of k_tp_mid (profiles/r2_ncu_full_cfg2_cfg3.md: pipe cycles / 2)
        ach = 2.0 * FP64_PER_PARTICLE * nt / (mid_ms * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": "k_tp_mid", "achieved": ach, "peak": peak_probe, "unit": "TFLOP/s",
                "frac": ach / peak_probe, "traffic": tab.get("k_tp_mid"),
                "peak_source": "DFMA probe measured in this run (genga_fp64_probe)",
                "ms_per_launch": mid_ms, "fp64_instructions_per_particle": FP64_PER_PARTICLE,
                "convention": "achieved = 2 flop x FP64 instructions the kernel issues (528 per particle by ncu's pipe cycles) / time: the share of the FP64 issue slots",
                "hbm": {"algorithmic_bytes_per_launch": 112.0 * nt, "gbs": 112.0 * nt / (mid_ms * 1e-3) / 1e9, "peak": hbm_peak,
                        "frac": 112.0 * nt / (mid_ms * 1e-3) / 1e9 / hbm_peak, "peak_source": hbm_src,
                        "note": "56 B read + 56 B written per particle (state + rc); not the binding roofline"},
                "front": {"kernel": "k_tp_front", "ms_per_launch": front_ms, "note": "first map of a call"},
                "back": {"kernel": "k_tp_back", "ms_per_launch": back_ms, "algorithmic_bytes_per_launch": 104.0 * nt,
                         "gbs": 104.0 * nt / (back_ms * 1e-3) / 1e9, "frac_hbm": 104.0 * nt / (back_ms * 1e-3) / 1e9 / hbm_peak,
                         "traffic": tab.get("k_tp_back"), "note": "last map of a call: the HBM-bound one"},
                # the step as a whole against SURVEY 8(d)'s unit
                "step": {"algorithmic_bytes_per_step": 96.0 * nt, "unit": "96 B per particle per step",
                         "gbs": 96.0 * nt / (step_ms * 1e-3) / 1e9, "frac_hbm": 96.0 * nt / (step_ms * 1e-3) / 1e9 / hbm_peak,
                         "traffic_per_step": tab.get("cfg2_step_dram_bytes")}}
    else:
        kick_ms = g.time_kernel(2, 200, dt)
        inter = w["n_systems"] * w["n_massive"] * (w["n_massive"] - 1)
        achieved = FLOP_PER_INTERACTION * inter / (kick_ms * 1e-3) / 1e12
        roof = {"bound": "alu", "kernel": "k_kick_multi", "achieved": achieved, "peak": peak_probe, "unit": "TFLOP/s",
                "frac": achieved / peak_probe, "traffic": tab.get("k_kick_multi"), "ms_per_launch": kick_ms,
                "interactions_per_launch": inter, "flop_per_interaction": FLOP_PER_INTERACTION,
                "peak_source": "DFMA probe measured in this run (genga_fp64_probe)",
                "note": "the pair loop timed alone; inside a step it runs within the fused multi-system kernels"}
    roof["bs"] = bs

    # ---- aggregate over ranks (replicas: no data-path collective)
    tmax, units = reduce_max_and_sum(elapsed, per_step * steps, dev)
    e2e_max, e2e_units = reduce_max_and_sum(e2e_s, per_step * ne2e, dev)
    res_max, res_units = reduce_max_and_sum(resident_s, per_step * nres, dev)
    line = {
        "metric": METRIC, "value": units / tmax, "unit": UNIT, "n_gpus": world, "steps": steps,
        "value_note": "pair interactions EVALUATED per second (force evaluations counted by the library: one per second-order step in "
                      "massive mode, the opening kick comes from stored sums, PAPER.md L266-274); round 1 counted two per step",
        "interactions_applied_per_s": units / tmax * ({2: 2, 4: 4, 6: 8}[w["order"]] / evals if w["mode"] != 1 and evals else 1.0),
        "warmup": max(warmup, 3), "ms_per_step": 1e3 * tmax / steps, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": config_dict(w, name, evals, world),
        "steps_per_s": steps * (world if w["mode"] == 0 else 1) / tmax,     # replicas step independently
        "resident": {"steps_per_s": nres * (world if w["mode"] == 0 else 1) / res_max, "value": res_units / res_max,
                     "ms_per_step": 1e3 * res_max / nres,
                     "note": "16-step CUDA graphs back to back, state resident in L2 (no flush)"},
        "e2e": {"value": e2e_units / e2e_max, "unit": UNIT, "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h,
                "steps": ne2e, "ms_per_step": 1e3 * e2e_max / ne2e},
        "gpu_launches": c1["launches"] - c0["launches"],
        "status": status,
        "phases_ms": phases,
        "encounters": {"groups_per_step": (c1["groups"] - c0["groups"]) / steps,
                       "bs_steps_per_step": (c1["bs_steps"] - c0["bs_steps"]) / steps,
                       "bs_rejects_per_step": (c1["bs_rejects"] - c0["bs_rejects"]) / steps,
                       "max_group": c1["max_group"]},
        "roofline": roof,
    }
    g.close()
    return line, w


def run_gpu(args):
    import torch
    import paper_1404_2324_b200 as G

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)

    clocks = ClockSampler(local)
    clocks.start()                      # nvidia-smi needs ~0.1 s to deliver its first sample: started before the warm-up
    line, w = measure(torch, G, dev, args.config, args.order, args.steps, args.warmup, rank, world, clocks)
    line["clocks"] = clocks.stop()

    # ---- the other configurations of BASELINE.json, short legs (1 GPU, default run only)
    if world == 1 and args.config == 1 and args.order is None and not args.no_configs:
        legs = []
        for cfg_id, order in ((0, None), (2, None), (3, None), (4, 4), (4, 6)):
            cs = ClockSampler(local)
            cs.start()
            leg, _ = measure(torch, G, dev, cfg_id, order, {0: 200, 2: 50, 3: 100, 4: 30}[cfg_id], 3, 0, 1, cs, e2e_steps=30)
            leg["clocks"] = cs.stop()
            legs.append({k: leg[k] for k in ("config", "value", "ms_per_step", "steps", "steps_per_s", "resident", "e2e", "gpu_launches",
                                             "status", "phases_ms", "encounters", "roofline", "clocks")})
        line["configs"] = legs

    if rank == 0:
        if world == 1 and not args.no_cpu:
            rate, n, secs = oracle_rate(w, budget_s=15.0, max_steps=10000)
            line["cpu_baseline"] = {"value": rate, "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": "%d full steps of the same workload in %.1f s (1 of %d cores; the oracle is single-threaded by design)" % (n, secs, os.cpu_count())}
        print(json.dumps(line))
    if world > 1:
        torch.distributed.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--order", type=int, default=None, help="override the configuration's order (2, 4, 6)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-configs", action="store_true", help="default run: skip the short legs of the other configurations")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_gpu(args)


if __name__ == "__main__":
    main()
