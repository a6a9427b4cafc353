#!/usr/bin/env python
"""bench.py -- headline benchmark of the flatspin hot path on B200 (contract: see the task prompt).

Default line: BASELINE.json config 5 (square ASI 500x500, 501,000 spins, neighbor_distance 10,
~621 neighbours/spin; "full field recompute plus switching scan repeated"), the configuration the
metric "spin-neighbor field updates/s (GB/s vs HBM peak)" is quoted on.  One step = one pass of the
field path: fs_update_fields (A3 full gather) + fs_scan (A4-A7 fused total field + astroid + arg-max).
The same JSON line carries a "relax" object: the 2M-spin sweep of config 4 (flips/s, us/flip, sweep
wall time), the second half of the metric, unless --no-relax.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--no-relax]

Multi-GPU: the path does not shard (replicas only); under torchrun every rank
runs an independent replica of the workload, value = sum over ranks / max time.
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
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2002_11401_b200 import workloads as W  # noqa: E402

METRIC = "spin_neighbor_field_updates_per_s"
UNIT = "interactions/s"


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        d = json.load(open(path))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def kernel_source_hash():
    """sha256 of the CUDA sources: measured ncu figures stored under profiles/ are tied to the code they were taken on."""
    import hashlib
    h = hashlib.sha256()
    d = os.path.join(ROOT, "paper_2002_11401_b200", "csrc")
    for f in sorted(os.listdir(d)):
        h.update(open(os.path.join(d, f), "rb").read())
    return h.hexdigest()[:16]


def stored_traffic(kernel, N, K):
    """dram__bytes_read + dram__bytes_write per launch from the committed ncu capture (profiles/traffic.json), or None
    if the capture was taken on other kernel sources or another workload size (a stale figure is not reported)."""
    path = os.path.join(ROOT, "profiles", "traffic.json")
    if not os.path.exists(path):
        return None, "no capture"
    d = json.load(open(path))
    e = d.get(kernel)
    if not e or e.get("source_hash") != kernel_source_hash() or (e.get("N"), e.get("K")) != (N, K):
        return None, "capture is stale for these sources / this size (see profiles/traffic.json)"
    return e["traffic_bytes"], e.get("source", "profiles/traffic.json")


class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True); self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 2 + k and r[2 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": reasons, "samples": len(sm)}


# ------------------------------------------------------------------------------------------------ CPU oracle legs
def oracle_field_sample(w, budget_s=12.0, chunk=256, seed=123):
    """Tier A as it stands (direct evaluation of Eq. 3 per pair + Eq. 5/6 per spin, nothing cached) on a bounded
    random sample of the workload's spins.  Returns (interactions/s, n_spins, n_interactions, seconds)."""
    from oracle import Oracle
    orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=w.spins)
    hx, hy = w.fields[0]
    orc.set_field(hx, hy, 0)
    rng = np.random.default_rng(seed)
    orc.neighbors_of(0)                       # builds the cell grid outside the timed region
    n_sp = n_int = 0
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < budget_s:
        for i in rng.integers(0, w.N, chunk):
            n_int += len(orc.neighbors_of(int(i)))
            orc.key_one(int(i))               # total field (Eq. 2,3) + astroid margin (Eq. 5,6)
            n_sp += 1
    dt = time.perf_counter() - t0
    return n_int / dt, n_sp, n_int, dt


CFG5_K = 632                       # maximum degree of config 5 (316 + 316), asserted against the library in run_ours
L2_NOTE = ("GPU arm: flushed before every timed step (256 MiB fill, untimed), step time = sum of per-step CUDA-event "
           "intervals; reference arm: the 6.2 GB coupling list is streamed from host DRAM every pass")


def workload_config(w, K, I):
    """The `config` object of the JSON line, the same for the GPU arm and the reference arm: what is computed, on which
    input.  How each arm ran it (kernel variant, lattice tables, launch details) goes under `run`."""
    return {"workload": w.name, "N": int(w.N), "K": None if K is None else int(K), "interactions": int(I),
            "neighbor_distance": float(w.params["neighbor_distance"]),
            "step": "full dipolar-field gather over every spin + switching scan (fs_update_fields + fs_scan)", "l2": L2_NOTE}


def cpu_field_workload(scale=None, need_gb=10.0):
    """Config 5 itself (501,000 spins, 311,247,284 interactions: ~7 GB of host memory for the oracle's precomputed
    couplings) when the host can hold it, else the same recipe at 160 x 160 under a name that says so."""
    import psutil
    if scale is None and psutil.virtual_memory().available < need_gb * 2**30:
        w = W.config("5", scale=160)
        w.name = "cfg5_recipe_160x160_sample"
        return w
    return W.config("5", scale=scale)


class OracleFieldPass:
    """The oracle's precomputed-neighbour-list field pass and switching scan (SURVEY.md 8(d) legs (i), (ii)), as it
    stands: couplings built once (untimed), then one pass = gather_cached (h_dip = sum_j s_j w_ij over the list) +
    scan_cached (Eq. 2, 5, 6 per spin, arg-max), single-threaded or with OpenMP over spins on all host cores."""

    def __init__(self, w):
        from oracle import Oracle
        self.w = w
        self.orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=w.spins)
        hx, hy = w.fields[0]
        self.orc.set_field(hx, hy, 0)
        t0 = time.perf_counter(); self.orc.build_weights(); self.t_build = time.perf_counter() - t0
        self.I = self.orc.num_interactions
        self.cores = os.cpu_count() or 1
        self.sample = (f"{w.name}: {w.N} spins, {self.I} interactions, couplings precomputed (untimed, {self.t_build:.1f} s); "
                       "each repetition = one gather over the whole list + one switching scan")

    def one_pass(self):
        a = time.perf_counter(); self.orc.gather_cached(); b = time.perf_counter(); self.orc.scan_cached(); c = time.perf_counter()
        return b - a, c - b

    def leg(self, threads, reps, warm=1):
        self.orc.set_threads(threads)
        for _ in range(warm):
            self.one_pass()
        tg = ts = 0.0
        for _ in range(reps):
            g, sc = self.one_pass(); tg += g; ts += sc
        return {"threads": threads, "repetitions": reps, "interactions_per_s": self.I * reps / (tg + ts),
                "gather_interactions_per_s": self.I * reps / tg, "scan_spins_per_s": self.w.N * reps / ts,
                "s_per_pass": (tg + ts) / reps}


def oracle_cached_legs(scale=None, reps=3):
    """Both legs on the full config 5 (or the named sample if the host cannot hold it): `reps` passes with 1 thread and
    with all cores ("Config 5 ... over 3 repetitions")."""
    fp = OracleFieldPass(cpu_field_workload(scale))
    out = {"sample": fp.sample, "workload": fp.w.name, "N": fp.w.N, "interactions": fp.I, "host_cores": fp.cores}
    out["threads_1"] = fp.leg(1, reps)
    out["threads_all"] = fp.leg(fp.cores, reps)
    return out


def oracle_relax_sample(scale=400):
    """Tier B oracle on a reduced config 4 (same recipe, n=scale): whole sweep, flips/s."""
    from oracle import Oracle
    w = W.config("4", scale=scale)
    orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=w.spins)
    orc.set_thermal(w.sigma_th, w.thermal_seed)
    orc.build_neighbors()
    t0 = time.perf_counter(); flips = 0
    for t, (hx, hy) in enumerate(w.fields):
        orc.set_field(hx, hy, t)
        flips += orc.relax_B(cap=1)[0]
    dt = time.perf_counter() - t0
    return {"flips_per_s": flips / dt, "flips": flips, "seconds": dt, "N": w.N,
            "sample": f"config 4 recipe at {scale}x{scale} ({w.N} spins), all {len(w.fields)} steps, Tier B oracle, 1 thread"}


def run_reference(args, rank, world):
    """The oracle as it stands on the host cores, on the GPU arm's workload: config 5 at full size, the precomputed-list
    gather + scan with OpenMP over all cores (the stronger of its two field tiers).  One step = one whole pass (gather
    + scan) over the 311 M interactions; the couplings are built once before the timed region, as fs_create builds the
    GPU arm's tables before its timed region."""
    if rank != 0:
        return
    fp = OracleFieldPass(cpu_field_workload(args.scale))
    fp.orc.set_threads(fp.cores)
    for _ in range(max(args.warmup, 1)):
        fp.one_pass()
    tot = 0.0
    for _ in range(args.steps):
        g, sc = fp.one_pass(); tot += g + sc
    value = fp.I * args.steps / tot
    one = fp.leg(1, min(args.steps, 3))
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": max(args.warmup, 1), "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(fp.w, CFG5_K if fp.w.N == 501000 else None, fp.I),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": fp.cores, "kind": "oracle", "sample": fp.sample,
                             "threads_1": one},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ GPU arm
def relax_sweep(B, torch, which="4", scale=None, sequential=False):
    """Whole-sweep wall time and flips/s of config 4 (2,002,000 spins, thermal ramp, 201 steps).  Pass 1 (timed as the
    headline): every step enqueued without a host round trip.  Pass 2 (statistics): the same sweep with the flip count
    read back after every step, for the per-step us/flip distribution."""
    w = W.config(which, scale=scale)
    t0 = time.perf_counter()
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    torch.cuda.synchronize(); t_create = time.perf_counter() - t0
    if sequential:
        sim.set_batch(0)

    def reset():
        sim.set_spins(w.spins)
        if w.sigma_th:
            sim.set_thermal(w.sigma_th, w.thermal_seed)
        sim.update_fields(); sim.counters(reset=True); torch.cuda.synchronize()

    reset()
    l0 = B.kernel_launches()
    t0 = time.perf_counter()
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t)
        sim.relax(sync=False)                      # no host round trip per step
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    launches = B.kernel_launches() - l0
    total, _ = sim.counters()
    flips = int(total.sum())
    s = sim.get_spins()
    st = sim.batch_stats()
    out = {"workload": w.name, "N": w.N, "steps": len(w.fields), "flips": flips, "sweep_wall_s": wall,
           "flips_per_s": flips / wall, "us_per_flip_whole_sweep": 1e6 * wall / max(flips, 1), "create_s": t_create,
           "gpu_launches": launches, "all_reversed": bool((s == -1).all().item()),
           "mode": "one flip per dependent chain (k_relax only)" if sequential else
                   "exact batched flips (k_relax_batch on all SMs) + k_relax for the tails",
           "batched": {"max_seeds": st["max_seeds"], "flips_committed": st["flips"], "rounds": st["rounds"],
                       "mean_committed_prefix": st["flips"] / max(st["rounds"], 1), "seq_threshold": st["seq_threshold"]}}
    # pass 2: per-step flips and device time
    reset()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(len(w.fields) + 1)]
    per = []
    ev[0].record()
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t)
        per.append(sim.relax())
        ev[t + 1].record()
    torch.cuda.synchronize()
    per = np.array(per); step_ms = np.array([ev[t].elapsed_time(ev[t + 1]) for t in range(len(w.fields))])
    quiet = float(np.median(step_ms[per == 0])) if (per == 0).any() else float(step_ms.min())
    busy = per >= 100
    out["quiet_step_ms_median"] = quiet
    out["max_step_ms"] = float(step_ms.max()); out["max_step_flips"] = int(per.max())
    if busy.any():
        upf = 1e3 * np.maximum(step_ms[busy] - quiet, 0.0) / per[busy]
        out["us_per_flip_mean"] = float(1e3 * np.maximum(step_ms[busy] - quiet, 0.0).sum() / per[busy].sum())
        out["us_per_flip_median_over_steps"] = float(np.median(upf))
        out["us_per_flip_p10_p90_over_steps"] = [float(np.percentile(upf, 10)), float(np.percentile(upf, 90))]
        out["steps_with_100_or_more_flips"] = int(busy.sum())
    # scan share: the fused scan alone at this size (thermal field included), times the number of steps
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    sim.scan_async(); torch.cuda.synchronize()
    e0.record()
    for _ in range(20):
        sim.scan_async()
    e1.record(); torch.cuda.synchronize()
    scan_ms = e0.elapsed_time(e1) / 20
    out["scan_ms"] = scan_ms
    out["scan_share_of_sweep"] = scan_ms * 1e-3 * len(w.fields) / wall
    out["flip_loop_share_of_sweep"] = 1.0 - out["scan_share_of_sweep"]
    sim.close()
    return out


def anneal_ensemble(B, torch, R=592):
    """PAPER.md:196-206 (IV.B): R replicas of the 50 x 50 square ASI (neighbor distance 10, b = 0.4, h_k = 0.186)
    annealed by an exponentially decreasing thermal field, whole protocol in one launch (one CTA per replica), then the
    spin-spin correlation by separation and the vertex populations of every replica on the device."""
    w = W.paper_square_anneal(50, replicas=R)
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    out = {"workload": w.name, "replicas": R, "N": w.N, "K": sim.K, "steps": len(w.fields)}
    for _ in range(2):
        sim.set_spins(np.tile(w.spins, (R, 1))); sim.set_thermal(0.0, w.thermal_seed); sim.update_fields(); sim.counters(reset=True)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        sim.sweep(w.fields, step0=0, per_step=False, sync=False, sigma=w.extra["sigma"])
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
    flips = int(sim.counters()[0].sum())
    t0 = time.perf_counter()
    sm, cnt = sim.correlation(0.5, 24)
    vp = sim.vertex_populations(w.extra["vertices"])
    torch.cuda.synchronize(); dt_red = time.perf_counter() - t0
    cnt = cnt.cpu().numpy().astype(np.float64); sm = sm.cpu().numpy().astype(np.float64).mean(axis=0)
    corr = np.where(cnt > 0, sm / np.maximum(cnt, 1), 0.0)
    vp = vp.cpu().numpy().astype(np.float64).mean(axis=0)
    out.update({"anneal_wall_s": dt, "flips": flips, "flips_per_s": flips / dt, "replica_anneals_per_s": R / dt,
                "reductions_wall_s": dt_red,
                "correlation_by_separation": {f"{0.5 * b:.1f}": round(float(corr[b]), 4) for b in range(24) if cnt[b] > 0},
                "vertex_fractions_I_II_III_IV": [round(float(x / vp.sum()), 4) for x in vp]})
    sim.close()
    return out


def protocol_sweeps(B, torch, cpu=True):
    """Whole-sweep wall time of configs 1-3 (BASELINE.json metric (3)): the stepwise path (fs_set_field +
    fs_relax per field value, asynchronous) and fs_sweep (whole protocol in one launch), with the Tier B
    oracle on the host beside them; plus an ensemble of config-1 replicas."""
    out = []
    for which in ("1", "2", "3"):
        w = W.config(which)
        sim = B.Sim(w.pos, w.angle, w.hc, w.params)
        row = {"workload": w.name, "N": w.N, "K": sim.K, "steps": len(w.fields)}
        for mode in ("stepwise", "one_launch"):
            sim.set_spins(w.spins); sim.update_fields(); sim.counters(reset=True)
            torch.cuda.synchronize(); t0 = time.perf_counter()
            if mode == "stepwise":
                for t, (hx, hy) in enumerate(w.fields):
                    sim.set_field(hx, hy, t); sim.relax(sync=False)
            else:
                sim.sweep(w.fields, step0=0, per_step=False, sync=False)
            torch.cuda.synchronize(); dt = time.perf_counter() - t0
            flips = int(sim.counters()[0].sum())
            row[mode] = {"wall_s": dt, "flips": flips, "flips_per_s": flips / dt}
        sim.close()
        if cpu:
            from oracle import Oracle
            orc = Oracle(w.pos, w.angle, w.hc, w.params, spins=w.spins)
            orc.build_neighbors()
            stride = 1 if which != "3" else 4
            t0 = time.perf_counter(); flips = 0
            for t, (hx, hy) in list(enumerate(w.fields))[::stride]:
                orc.set_field(hx, hy, t); flips += orc.relax_B(cap=1)[0]
            dt = time.perf_counter() - t0
            row["cpu_oracle_tier_b"] = {"wall_s": dt, "flips": flips, "cores": 1,
                                        "sample": "whole protocol" if stride == 1 else f"every {stride}th field value"}
        out.append(row)
    # ensemble: R replicas of config 1 (different disorder), whole protocol in one launch, one CTA per replica
    w = W.config("1")
    R = 4736                                           # 32 replicas per SM
    hc = W.coercive_fields(w.N, seed=1000, replicas=R)
    sim = B.Sim(w.pos, w.angle, hc, w.params)
    for _ in range(2):                                 # second pass timed (first one warms the instruction caches)
        sim.set_spins(np.ones((R, w.N), np.int8)); sim.update_fields(); sim.counters(reset=True)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        sim.sweep(w.fields, step0=0, per_step=False, sync=False)
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
    flips = int(sim.counters()[0].sum())
    sim.close()
    ens = {"workload": w.name, "replicas": R, "N": w.N, "steps": len(w.fields), "wall_s": dt, "flips": flips,
           "flips_per_s": flips / dt, "replica_sweeps_per_s": R / dt}
    return out, ens


def paper_workloads(B, torch):
    """The two timings the paper itself prints besides Fig. 9, on its own parameter set
    (section IV.C; the field range is not printed, workloads.paper_pinwheel_reversal states the choice):
    one reversal of the 25 x 25 pinwheel ASI (1250 magnets, K = 2500 field values; paper: ~6 s including
    result storage) and of the 708 x 708 pinwheel ASI (1,002,528 magnets; paper: "several days")."""
    out = []
    for n, paper in ((25, "approximately 6 seconds (PAPER.md:286)"), (708, "several days (PAPER.md:288)")):
        w = W.paper_pinwheel_reversal(n, 0.0)
        t0 = time.perf_counter()
        sim = B.Sim(w.pos, w.angle, w.hc, w.params); torch.cuda.synchronize(); tc = time.perf_counter() - t0
        sim.set_spins(w.spins); sim.update_fields(); torch.cuda.synchronize()
        t0 = time.perf_counter()
        for t, (hx, hy) in enumerate(w.fields):
            sim.set_field(hx, hy, t); sim.relax(sync=False)
        torch.cuda.synchronize(); dt = time.perf_counter() - t0
        flips = int(sim.counters()[0].sum())
        s = sim.get_spins()
        row = {"workload": w.name, "N": w.N, "K_neighbors": sim.K, "field_values": len(w.fields), "create_s": tc,
               "reversal_wall_s": dt, "flips": flips, "reversed": bool((s == -torch.as_tensor(w.spins, device=s.device)).all().item()),
               "paper": paper + ", Tesla V100, other hardware and includes I/O: context, not a target"}
        if n == 25:
            sim.set_spins(w.spins); sim.update_fields(); torch.cuda.synchronize(); t0 = time.perf_counter()
            sim.sweep(w.fields, per_step=False, sync=False); torch.cuda.synchronize()
            row["one_launch_wall_s"] = time.perf_counter() - t0
        sim.close()
        out.append(row)
    return out


def phase_profile():
    """Per-phase budgets of the two relax kernels from an instrumented build of the same sources (see build.build_profile):
    config 4, k_relax_batch rounds (ns per phase, CTA 0) and k_relax alone (cycles per flip and phase)."""
    import ctypes as C
    import tempfile
    import torch
    from paper_2002_11401_b200 import binding as B, build as bld
    lib = bld.build_profile(tempfile.mkdtemp(prefix="fs_profile_"))
    L = B.load_library(lib); B._lib = L
    L.fs_debug_batch_profile.argtypes = [C.c_void_p, C.c_void_p]
    L.fs_debug_relax_profile.argtypes = [C.c_void_p, C.c_int]
    out = {}
    w = W.config("4")
    for mode in ("batched", "sequential"):
        sim = B.Sim(w.pos, w.angle, w.hc, w.params); sim.set_thermal(w.sigma_th, w.thermal_seed)
        if mode == "sequential":
            sim.set_batch(0)
        sim.update_fields()
        z = (C.c_longlong * 16)(); L.fs_debug_relax_profile(z, 1)
        torch.cuda.synchronize(); t0 = time.perf_counter()
        for t, (hx, hy) in enumerate(w.fields):
            sim.set_field(hx, hy, t); sim.relax(sync=False)
        torch.cuda.synchronize(); wall = time.perf_counter() - t0
        st = sim.batch_stats()
        row = {"sweep_wall_s": wall, "batch": st}
        if mode == "batched":
            p = (C.c_longlong * 12)(); L.fs_debug_batch_profile(sim.h, p)
            names = ["1 threshold (histogram over the candidate list, theta)", "2 seeds (compaction)", "3 claims", "4 conflict edges",
                     "5 components (labels)", "6 local relaxation (CTA 0's own warps)", "6b wait for the slowest component",
                     "7 cut, commit / undo", "8 merged order -> flip log"]
            row["us_per_round"] = {n: p[k] / 1e3 / max(st["rounds"], 1) for k, n in enumerate(names)}
        r = (C.c_longlong * 16)(); L.fs_debug_relax_profile(r, 1)
        nfl = max(r[15], 1)
        if mode == "sequential":
            row["k_relax_cycles_per_flip"] = {"flips": int(r[15]), "top arg-max (+ prefetch engines)": r[0] / nfl, "update (row, state, margins)": r[1] / nfl,
                                              "wait at the update barrier (thread 0)": r[2] / nfl, "leaf repair + groups + supergroups": r[3] / nfl,
                                              "of which: own leaf rescan": r[5] / nfl, "wait for the other warps' rescans": r[6] / nfl,
                                              "groups + wait": r[7] / nfl, "supergroups": r[8] / nfl, "wait at the last barrier": r[4] / nfl}
        out[mode] = row
        sim.close()
    print(json.dumps({"phase_profile": out, "workload": w.name, "source_hash": kernel_source_hash()}), flush=True)


def scan_probe():
    """The fused scan alone at config-4 size (2,002,000 spins, thermal field on: Philox + Box-Muller per spin), L2 flushed
    before every launch: the command `ncu -k regex:k_scan` is pointed at."""
    import torch
    from paper_2002_11401_b200 import binding as B
    w = W.config("4")
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    sim.set_spins(w.spins); sim.set_thermal(w.sigma_th, w.thermal_seed)
    hx, hy = w.fields[100]
    sim.set_field(hx, hy, 100); sim.update_fields()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    for _ in range(3):
        sim.scan_async()
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(2)] for _ in range(10)]
    for a, b in ev:
        flush.fill_(1); a.record(); sim.scan_async(); b.record()
    torch.cuda.synchronize()
    ms = np.array([a.elapsed_time(b) for a, b in ev])
    n_sw, best, bestL = sim.scan()
    peak, _ = measured_peaks()
    print(json.dumps({"scan_probe": {"workload": w.name, "N": w.N, "thermal": True, "scan_us_mean": 1e3 * float(ms.mean()),
                                     "scan_us_min": 1e3 * float(ms.min()), "algorithmic_bytes": 49 * w.N,
                                     "hbm_frac": 49 * w.N / (float(ms.mean()) * 1e-3) / 1e9 / peak,
                                     "n_switchable": n_sw, "best_index": best, "source_hash": kernel_source_hash()}}), flush=True)
    sim.close()


def max_over_ranks(dist, values_ms, device):
    """Replicas only: every rank times its own replica; the job's time is the slowest rank's."""
    import torch
    t = torch.tensor(list(values_ms), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(units_per_rank_step, steps, world, ms):
    """Whole-job throughput: every rank processed `units_per_rank_step` per step (weak scaling, no collective
    on the data path), all ranks finished within `ms` (max over ranks)."""
    return world * units_per_rank_step * steps / (ms * 1e-3)


def run_ours(args, rank, world, local_rank):
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the flatspin path has no CPU fallback")
    from paper_2002_11401_b200 import binding as B
    dist = None
    if world > 1:
        import torch.distributed as dist
        torch.cuda.set_device(local_rank)
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    dev = f"cuda:{local_rank}"
    torch.cuda.set_device(local_rank)

    w = W.config("5") if args.scale is None else W.config("5", scale=args.scale)
    t0 = time.perf_counter()
    sim = B.Sim(w.pos, w.angle, w.hc, w.params, device=dev)
    torch.cuda.synchronize(); t_create = time.perf_counter() - t0
    lat = sim.lattice()
    sim.set_gather_variant(args.gather)
    use_stencil = lat["active"] and args.gather != B.GATHER_ELL_F64
    sim.set_spins(w.spins)
    hx, hy = w.fields[0]
    sim.set_field(hx, hy, 0)
    I, N, K = sim.n_interactions, sim.N, sim.K
    assert N != 501000 or K == CFG5_K, K                   # the reference arm states config 5's K without a neighbour build of its own
    ell_bytes = I * 20.0 + N * 17.0     # idx + weight pair per interaction; s read + h_dip written per spin
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > L2 (126 MB)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(n, split=False):
        """n steps of (gather, scan); L2 flushed (untimed) before every step.  Returns per-step ms of the whole step and
        of the gather kernel, from CUDA events on the launching stream.  split=False (the timed region of the headline):
        events at the step boundaries only, so that the scan can be launched programmatically dependent on the gather (an
        event record between the two would serialise them); split=True: a third event between gather and scan."""
        e = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n)]
        for k in range(n):
            flush.fill_(k & 0xff)
            e[k][0].record(); sim.update_fields()
            if split:
                e[k][1].record()
            sim.scan_async(); e[k][2].record()
        barrier()
        return (np.array([a.elapsed_time(c) for a, b, c in e]),
                np.array([a.elapsed_time(b) for a, b, c in e]) if split else None)

    for _ in range(max(args.warmup, 3)):
        sim.update_fields(); sim.scan_async()
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    l0 = B.kernel_launches()
    step_ms, _ = timed_steps(args.steps)
    launches = B.kernel_launches() - l0
    # the dominant kernel's own duration: the same steps again with an event between gather and scan
    split_ms, g_ms = timed_steps(args.steps, split=True)
    # the timed region lasts a few milliseconds, less than one nvidia-smi sampling period: keep the sampler
    # running over an untimed replay of the same loop (~1 s) so that the clocks are read under this load
    t_rep = time.perf_counter()
    while time.perf_counter() - t_rep < 1.0:
        for _ in range(50):
            sim.update_fields(); sim.scan_async()
        torch.cuda.synchronize()
    clocks = sampler.stop()
    clocks["note"] = "sampled from the start of the timed steps through a 1 s untimed replay of the same loop"
    ms = float(step_ms.sum())
    gather_ms = float(g_ms.mean())
    n_sw, best, bestL = sim.scan()
    ell = None
    if use_stencil and not args.no_ell:
        # the general-geometry ELL gather on the same workload, for the HBM roofline (inputs 6.2 GB > L2)
        sim.set_gather_variant(B.GATHER_ELL_F64)
        for _ in range(3):
            sim.update_fields()
        _, eg = timed_steps(min(args.steps, 10), split=True)
        sim.set_gather_variant(args.gather)
        ell = float(eg.mean())

    f32 = None
    if use_stencil and not args.no_ell:
        # the optional fp32 field path (north_star: reported separately, fields at 1e-5, no flip-order claim)
        try:
            sim.set_gather_variant(B.GATHER_STENCIL_F32)
            for _ in range(3):
                sim.update_fields()
            _, fg = timed_steps(min(args.steps, 10), split=True)
            f32 = float(fg.mean())
        except Exception:
            f32 = None
        sim.set_gather_variant(args.gather)
        sim.update_fields()

    # end to end through the host-buffer C-ABI call: H2D spins + gather + scan + D2H fields every step
    s_host = torch.as_tensor(w.spins).pin_memory()
    h_host = torch.empty((N, 2), dtype=torch.float64).pin_memory()
    for _ in range(2):
        sim.step_host(s_host, h_host)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sim.step_host(s_host, h_host)
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0
    # the same call returning only the scan's summary (24 B) to the host: what a relaxation driven from the host needs
    for _ in range(2):
        sim.step_host(s_host, None)
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        sim.step_host(s_host, None)
    torch.cuda.synchronize()
    e2e_sum_s = time.perf_counter() - t0

    ms, e2e_ms, e2e_sum_ms = max_over_ranks(dist, [ms, e2e_s * 1e3, e2e_sum_s * 1e3], dev)
    value = whole_job_value(I, args.steps, world, ms)
    e2e_value = whole_job_value(I, args.steps, world, e2e_ms)

    peak, peak_src = measured_peaks()
    if use_stencil:
        dfma_peak = B.measure_fp64_peak()                     # DFMA/s, measured in this run
        achieved = 2.0 * 2.0 * I / (gather_ms * 1e-3) / 1e12    # 2 DFMA (4 flop) per interaction
        roofline = {"bound": "alu", "kernel": "k_gather_stencil", "achieved": achieved, "peak": 2.0 * dfma_peak / 1e12,
                    "unit": "TFLOP/s", "frac": achieved / (2.0 * dfma_peak / 1e12),
                    "traffic": stored_traffic("k_gather_stencil", N, K)[0], "traffic_source": stored_traffic("k_gather_stencil", N, K)[1],
                    "inversion_pairs": bool(lat.get("inversion_pairs")),
                    "peak_source": "fp64 DFMA-chain kernel (fs_measure_fp64_peak) measured in this run; "
                                   "nominal 148 SM x 64 DFMA/clk x 1.965 GHz = 37.2 TFLOP/s",
                    "algorithmic_flops_per_launch": 4.0 * I, "kernel_ms": gather_ms, "source_hash": kernel_source_hash(),
                    "share_of_step": gather_ms / float(split_ms.mean()),
                    "kernel_ms_note": "CUDA events around fs_update_fields in a second pass over the same steps (an event between "
                                      "gather and scan would serialise the programmatically dependent scan of the timed pass); "
                                      "share_of_step is relative to that pass's step time",
                    "step_ms_with_split_events": float(split_ms.mean())}
    else:
        achieved = ell_bytes / (gather_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "k_gather", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": ell_bytes, "kernel_ms": gather_ms,
                    "share_of_step": gather_ms / float(split_ms.mean())}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": workload_config(w, K, I),
        "run": {"gather": ("lattice stencil" + (", inversion-paired" if lat.get("inversion_pairs") and args.gather != 3 else "")) if use_stencil else "ELL fp64",
                "lattice": lat, "parallelism": "replicas only" if world > 1 else "1 GPU", "create_s": t_create,
                "n_switchable": n_sw, "best_index": best},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(N), "d2h_bytes_per_step": int(16 * N + 24),
                "ms_per_step": e2e_ms / args.steps, "call": "fs_step_host (pinned host spins in, host total fields out)",
                "summary_only": {"value": whole_job_value(I, args.steps, world, e2e_sum_ms), "ms_per_step": e2e_sum_ms / args.steps,
                                 "h2d_bytes_per_step": int(N), "d2h_bytes_per_step": 24,
                                 "call": "fs_step_host with h_host_out = NULL (spins in; number of switchable spins, arg-max and its margin out)"}},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "paper_context": {"v100_field_calcs_per_s": 1e8, "v100_interactions_per_s": 8e8,
                          "source": "PAPER.md:274-282, Tesla V100, 8-neighbourhood; other hardware, context only"},
    }
    if ell is not None:
        a = ell_bytes / (ell * 1e-3) / 1e9
        line["roofline_ell"] = {"bound": "hbm", "kernel": "k_gather (general-geometry ELL path, same workload)",
                                "achieved": a, "peak": peak, "unit": "GB/s", "frac": a / peak,
                                "traffic": stored_traffic("k_gather", N, K)[0], "traffic_source": stored_traffic("k_gather", N, K)[1],
                                "peak_source": peak_src, "algorithmic_bytes_per_launch": ell_bytes, "kernel_ms": ell,
                                "interactions_per_s": I / (ell * 1e-3)}
    if f32 is not None:
        ffma = B.measure_fp32_peak()
        a32 = 4.0 * I / (f32 * 1e-3) / 1e12
        line["roofline_f32"] = {"bound": "alu", "kernel": "k_gather_stencil<float> (optional fp32 field path, reported separately)",
                                "achieved": a32, "peak": 2.0 * ffma / 1e12, "unit": "TFLOP/s", "frac": a32 / (2.0 * ffma / 1e12),
                                "kernel_ms": f32, "interactions_per_s": I / (f32 * 1e-3),
                                "peak_source": "fp32 FFMA-chain kernel (fs_measure_fp32_peak) measured in this run",
                                "accuracy": "fields within 1e-5 of the fp64 oracle relative to max|h| (tests/test_gpu_parity.py); no flip-order claim"}
    sim.close()
    if rank == 0 and not args.no_cpu:
        legs = oracle_cached_legs(scale=args.scale, reps=3)
        v, n_sp, n_int, dt = oracle_field_sample(w, budget_s=min(args.cpu_budget, 6.0))
        line["cpu_baseline"] = {"value": legs["threads_all"]["interactions_per_s"], "unit": UNIT, "cores": legs["host_cores"],
                                "kind": "oracle", "sample": legs["sample"],
                                "threads_1": legs["threads_1"], "threads_all": legs["threads_all"],
                                "tier_a_direct": {"interactions_per_s": v, "cores": 1,
                                                  "sample": f"{n_sp} random spins of {w.name} ({n_int} interactions, {dt:.1f} s): "
                                                            "direct Eq. 3 per pair + Eq. 5/6 per spin, nothing cached"}}
    if rank == 0 and not args.no_relax:
        try:
            line["relax"] = relax_sweep(B, torch, "4", scale=args.relax_scale)
            line["relax_sequential"] = relax_sweep(B, torch, "4", scale=args.relax_scale, sequential=True)
            line["relax"]["speedup_over_sequential"] = line["relax_sequential"]["sweep_wall_s"] / line["relax"]["sweep_wall_s"]
            if not args.no_cpu:
                line["relax"]["cpu_baseline"] = oracle_relax_sample()
        except Exception as e:   # never lose the headline line
            line["relax"] = {"error": repr(e)}
        try:
            line["sweeps"], line["ensemble"] = protocol_sweeps(B, torch, cpu=not args.no_cpu)
        except Exception as e:
            line["sweeps"] = {"error": repr(e)}
        try:
            line["anneal_ensemble"] = anneal_ensemble(B, torch)
        except Exception as e:
            line["anneal_ensemble"] = {"error": repr(e)}
        try:
            line["paper_workloads"] = paper_workloads(B, torch)
        except Exception as e:
            line["paper_workloads"] = {"error": repr(e)}
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank == 0:
        print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--gather", type=int, default=0, help="FS_GATHER_* variant (0 auto, 1 ELL fp64, 2 lattice stencil, 3 stencil without inversion pairing)")
    ap.add_argument("--no-ell", action="store_true", help="skip the side measurement of the ELL gather")
    ap.add_argument("--scale", type=int, default=None, help="debug: lattice size override for config 5")
    ap.add_argument("--relax-scale", type=int, default=None, help="debug: lattice size override for config 4")
    ap.add_argument("--no-relax", action="store_true")
    ap.add_argument("--phase-profile", action="store_true", help="instrumented build: per-phase budgets of k_relax_batch / k_relax on config 4")
    ap.add_argument("--scan-probe", action="store_true", help="k_scan alone at config-4 size with the thermal field (ncu target)")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.phase_profile:
        if rank == 0:
            phase_profile()
    elif args.scan_probe:
        if rank == 0:
            scan_probe()
    elif args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
