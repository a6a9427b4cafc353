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
    """The oracle as it stands (Tier A direct evaluation of Eq. 3 + Eq. 5/6 per spin) on a bounded random
    sample of the workload's spins.  Returns (interactions/s, n_spins, n_interactions, seconds)."""
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
    if rank != 0:
        return
    w = W.config("5")
    budget = 3.0
    for _ in range(args.warmup):
        oracle_field_sample(w, budget_s=0.5)
    vals = []; t0 = time.perf_counter()
    for k in range(args.steps):
        v, n_sp, n_int, dt = oracle_field_sample(w, budget_s=budget, seed=1000 + k)
        vals.append((n_int, dt))
    tot_int = sum(a for a, _ in vals); tot_t = sum(b for _, b in vals)
    value = tot_int / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": w.name, "N": w.N, "neighbor_distance": 10.0},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle",
                             "sample": f"each step: {budget:.0f} s of random spins of config 5, direct Eq. 3 + Eq. 5/6 per spin"},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------ GPU arm
def relax_sweep(B, torch, which="4", scale=None):
    """Whole-sweep wall time and flips/s of config 4 (2,002,000 spins, thermal ramp, 201 steps)."""
    w = W.config(which, scale=scale)
    t0 = time.perf_counter()
    sim = B.Sim(w.pos, w.angle, w.hc, w.params)
    torch.cuda.synchronize(); t_create = time.perf_counter() - t0
    sim.set_spins(w.spins)
    if w.sigma_th:
        sim.set_thermal(w.sigma_th, w.thermal_seed)
    sim.update_fields()
    ev = [torch.cuda.Event(enable_timing=True) for _ in range(len(w.fields) + 1)]
    l0 = B.kernel_launches()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    ev[0].record()
    for t, (hx, hy) in enumerate(w.fields):
        sim.set_field(hx, hy, t)
        sim.relax(sync=False)                      # no host round trip per step
        ev[t + 1].record()
    torch.cuda.synchronize()
    wall = time.perf_counter() - t0
    launches = B.kernel_launches() - l0
    total, _ = sim.counters()
    flips = int(total.sum())
    step_ms = np.array([ev[t].elapsed_time(ev[t + 1]) for t in range(len(w.fields))])
    s = sim.get_spins()
    out = {"workload": w.name, "N": w.N, "steps": len(w.fields), "flips": flips, "sweep_wall_s": wall,
           "flips_per_s": flips / wall, "create_s": t_create, "gpu_launches": launches,
           "all_reversed": bool((s == -1).all().item()), "max_step_ms": float(step_ms.max()),
           "quiet_step_ms_median": float(np.median(step_ms))}
    busy = step_ms > 4 * np.median(step_ms)
    if busy.any() and flips:
        # per-flip latency inside the avalanches: time of the busy steps beyond a quiet step / flips
        out["us_per_flip"] = float(1e3 * (step_ms[busy] - np.median(step_ms)).sum() / flips)
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
    ell_bytes = I * 20.0 + N * 17.0     # idx + weight pair per interaction; s read + h_dip written per spin
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)      # > L2 (126 MB)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def timed_steps(n):
        """n steps of (gather, scan); L2 flushed (untimed) before every step.  Returns per-step ms of the
        whole step and of the gather kernel, from CUDA events on the launching stream."""
        e = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(n)]
        for k in range(n):
            flush.fill_(k & 0xff)
            e[k][0].record(); sim.update_fields(); e[k][1].record(); sim.scan_async(); e[k][2].record()
        barrier()
        return (np.array([a.elapsed_time(c) for a, b, c in e]), np.array([a.elapsed_time(b) for a, b, c in e]))

    for _ in range(max(args.warmup, 3)):
        sim.update_fields(); sim.scan_async()
    barrier()
    sampler = ClockSampler(local_rank); sampler.start()
    l0 = B.kernel_launches()
    step_ms, g_ms = timed_steps(args.steps)
    launches = B.kernel_launches() - l0
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
        _, eg = timed_steps(min(args.steps, 10))
        sim.set_gather_variant(args.gather)
        ell = float(eg.mean())

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

    ms, e2e_ms = max_over_ranks(dist, [ms, e2e_s * 1e3], dev)
    value = whole_job_value(I, args.steps, world, ms)
    e2e_value = whole_job_value(I, args.steps, world, e2e_ms)

    peak, peak_src = measured_peaks()
    if use_stencil:
        dfma_peak = B.measure_fp64_peak()                     # DFMA/s, measured in this run
        achieved = 2.0 * 2.0 * I / (gather_ms * 1e-3) / 1e12    # 2 DFMA (4 flop) per interaction
        roofline = {"bound": "alu", "kernel": "k_gather_stencil", "achieved": achieved, "peak": 2.0 * dfma_peak / 1e12,
                    "unit": "TFLOP/s", "frac": achieved / (2.0 * dfma_peak / 1e12),
                    # dram__bytes_read+write of one launch at full config-5 size, from the committed ncu capture
                    "traffic": 3310848 if (N, K) == (501000, 632) else None, "traffic_source": "profiles/r01_ncu_full.md",
                    "peak_source": "fp64 DFMA-chain kernel (fs_measure_fp64_peak) measured in this run; "
                                   "nominal 148 SM x 64 DFMA/clk x 1.965 GHz = 37.2 TFLOP/s",
                    "algorithmic_flops_per_launch": 4.0 * I, "kernel_ms": gather_ms,
                    "share_of_step": gather_ms / (ms / args.steps)}
    else:
        achieved = ell_bytes / (gather_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": "k_gather", "achieved": achieved, "peak": peak, "unit": "GB/s",
                    "frac": achieved / peak, "traffic": None, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": ell_bytes, "kernel_ms": gather_ms,
                    "share_of_step": gather_ms / (ms / args.steps)}
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "N": N, "K": K, "interactions": I, "neighbor_distance": w.params["neighbor_distance"],
                   "step": "fs_update_fields + fs_scan", "gather": "lattice stencil" if use_stencil else "ELL fp64",
                   "lattice": lat,
                   "l2": "flushed before every timed step (256 MiB fill, untimed); step time = sum of per-step CUDA-event intervals",
                   "parallelism": "replicas only" if world > 1 else "1 GPU", "create_s": t_create,
                   "n_switchable": n_sw, "best_index": best},
        "clocks": clocks,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(N), "d2h_bytes_per_step": int(16 * N + 24),
                "ms_per_step": e2e_ms / args.steps, "call": "fs_step_host (pinned host spins in, host total fields out)"},
        "gpu_launches": int(launches),
        "roofline": roofline,
        "paper_context": {"v100_field_calcs_per_s": 1e8, "v100_interactions_per_s": 8e8,
                          "source": "PAPER.md:274-282, Tesla V100, 8-neighbourhood; other hardware, context only"},
    }
    if ell is not None:
        a = ell_bytes / (ell * 1e-3) / 1e9
        line["roofline_ell"] = {"bound": "hbm", "kernel": "k_gather (general-geometry ELL path, same workload)",
                                "achieved": a, "peak": peak, "unit": "GB/s", "frac": a / peak,
                                "traffic": 6271733000 if (N, K) == (501000, 632) else None,
                                "traffic_source": "profiles/r01_ncu_full.md",
                                "peak_source": peak_src, "algorithmic_bytes_per_launch": ell_bytes, "kernel_ms": ell,
                                "interactions_per_s": I / (ell * 1e-3)}
    sim.close()
    if rank == 0 and not args.no_cpu:
        v, n_sp, n_int, dt = oracle_field_sample(w, budget_s=args.cpu_budget)
        line["cpu_baseline"] = {"value": v, "unit": UNIT, "cores": 1, "kind": "oracle",
                                "sample": f"{n_sp} random spins of {w.name} ({n_int} interactions, {dt:.1f} s): direct Eq. 3 + Eq. 5/6 per spin"}
    if rank == 0 and not args.no_relax:
        try:
            line["relax"] = relax_sweep(B, torch, "4", scale=args.relax_scale)
            if not args.no_cpu:
                line["relax"]["cpu_baseline"] = oracle_relax_sample()
        except Exception as e:   # never lose the headline line
            line["relax"] = {"error": repr(e)}
        try:
            line["sweeps"], line["ensemble"] = protocol_sweeps(B, torch, cpu=not args.no_cpu)
        except Exception as e:
            line["sweeps"] = {"error": repr(e)}
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
    ap.add_argument("--gather", type=int, default=0, help="FS_GATHER_* variant (0 auto, 1 ELL fp64, 2 lattice stencil)")
    ap.add_argument("--no-ell", action="store_true", help="skip the side measurement of the ELL gather")
    ap.add_argument("--scale", type=int, default=None, help="debug: lattice size override for config 5")
    ap.add_argument("--relax-scale", type=int, default=None, help="debug: lattice size override for config 4")
    ap.add_argument("--no-relax", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--cpu-budget", type=float, default=12.0)
    args = ap.parse_args()
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
