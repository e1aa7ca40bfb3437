#!/usr/bin/env python
"""bench.py -- headline measurement of the PAKR hot path on B200 (contract: see DESIGN.md "Measurement").

A "step" is one pass of the whole hot path: one pakr_plan call (AO-x replanning around the batched
expansion iteration, every row of SURVEY.md 8(a)) on BASELINE.json configs[1] (C2: 3D double
integrator, 32 boxes, B=1024, K=8, cap 2^20, 20 replans) with planner seed = step index.
metric = expanded nodes/s = children propagated and checked per second (B*K*iterations / time).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl reference]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2607_03987_b200 import replicas, workloads as wl  # noqa: E402

WORKLOAD = "C2"
METRIC = "expanded nodes/s"
UNIT = "nodes/s"
# dram__bytes_read.sum + dram__bytes_write.sum of one pakr_loop_kernel launch on this workload, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists for the current kernel).
NCU_TRAFFIC_BYTES_PER_LAUNCH = 1222656  # profiles/r01_s3_ncu_bench.md


def algorithmic_ops(problem, nn_pairs: int, children: int) -> dict:
    """Algorithmic fp32 lane-operations of one launch: the NN scan evaluates
    nn_pairs (query, node) pairs at D sub + D fma + compare + select each (+ D mul if weighted, +2 on an
    angle dim); a child costs S steps of (8 D integrator ops + F dynamics ops + 2 per bounded dim + the
    obstacle broad phase: cell index and header, 10 ops, plus ONE obstacle test -- not one per obstacle,
    because the grid culls the rest exactly)."""
    D = problem.state_dim
    weighted = not np.all(problem.nn_weight == 1.0)
    n_angle = int((problem.dim_kind == 1).sum())
    nn_per_pair = 2 * D + 2 + (D if weighted else 0) + 2 * n_angle
    f_dyn = {wl.DYN_DOUBLE_INTEGRATOR: 0, wl.DYN_UNICYCLE2: 25, wl.DYN_QUADROTOR: 140, wl.DYN_DUBINS_AIRPLANE: 50,
             wl.DYN_UNICYCLE1: 24, wl.DYN_QUADROTOR_BODY: 170}[problem.dynamics_id]
    stages = 4 if problem.integrator == wl.INT_RK4 else 1
    integ = 8 * D if problem.integrator == wl.INT_RK4 else 2 * D
    n_bounded = int((np.isfinite(problem.state_lo) & (problem.dim_kind == 0)).sum())
    c_obs = 2 * problem.pos_dim if problem.obstacle_type == wl.OBS_AABB else 5
    per_child = problem.steps_per_edge * (stages * f_dyn + integ + 2 * n_bounded + 10 + c_obs)
    return dict(nn=nn_pairs * nn_per_pair, prop=children * per_child, nn_per_pair=nn_per_pair, per_child=per_child)


class ClockSampler(threading.Thread):
    """Samples nvidia-smi clocks and throttle reasons during the timed region (B200_PROFILING.md)."""

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._halt = index, [], threading.Event()

    def run(self):
        q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")
        while not self._halt.is_set():
            try:
                out = subprocess.run(["nvidia-smi", f"--query-gpu={q}", "--format=csv,noheader,nounits", "-i",
                                      str(self.index)], capture_output=True, text=True, timeout=5).stdout.strip()
                if out:
                    self.rows.append([c.strip() for c in out.split(",")])
            except Exception:
                pass
            self._halt.wait(0.2)

    def finish(self) -> dict:
        self._halt.set()
        self.join(timeout=6)
        sm = [float(r[0]) for r in self.rows if r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if r[1].replace(".", "").isdigit()]
        reasons = set()
        for r in self.rows:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(self.rows)}


def oracle_sample(problem, cfg, seed: int) -> dict:
    """The CPU oracle as it stands on a bounded sample of the workload: replan 0 (first solution) of the
    same config and seed, one thread."""
    from oracle import pakr_oracle as orc
    op = orc.OracleProblem(problem)
    t0 = time.perf_counter()
    res = orc.plan(op, seed, cfg.B, cfg.K, cfg.tree_capacity, 1)
    dt = time.perf_counter() - t0
    return dict(value=res["children"] / dt, seconds=dt, children=res["children"], iterations=res["iterations"],
                first_solution_ms=res["first_solution_ms"], cost=res["cost"])


def run_reference(args, problem, cfg):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    for i in range(args.warmup):
        oracle_sample(problem, cfg, 1000 + i) if i == 0 else None  # one untimed pass warms the library
    t_total, children, firsts = 0.0, 0, []
    for i in range(args.steps):
        r = oracle_sample(problem, cfg, i)
        t_total += r["seconds"]
        children += r["children"]
        firsts.append(r["first_solution_ms"])
    value = children / t_total
    sample = f"replan 0 (first solution) of {WORKLOAD} per step, planner seeds 0..{args.steps - 1}"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / args.steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": WORKLOAD, "dynamics": problem.name, "B": cfg.B, "K": cfg.K,
                       "tree_capacity": cfg.tree_capacity, "n_replans": cfg.n_replans,
                       "sampled": "replan 0 only (the oracle needs ~3 s per replan-0, minutes for all 20)"},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "first_solution_ms_median": statistics.median(firsts)}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    problem, cfg = wl.CONFIGS[WORKLOAD]()
    if args.impl == "reference":
        if args.steps > 8:
            args.steps = 8  # ~10 s of CPU per step: keep the whole run within minutes
        return run_reference(args, problem, cfg)

    import torch
    import torch.distributed as dist
    from paper_2607_03987_b200 import pakr

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    pakr.lib()  # fails loudly if the CUDA extension is missing
    pl = pakr.Planner(problem, local)
    ws = pl.workspace(cfg.B, cfg.K, cfg.tree_capacity)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}")  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # replicas only: rank r plans seeds r, r + world, ...
    seeds = replicas.replica_seeds(rank, world, args.warmup + args.steps)
    for s in seeds[:max(args.warmup, 3)]:
        pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    results, wall = [], []
    barrier()
    for i, s in enumerate(seeds[args.warmup:]):
        flush.fill_(i & 0xFF)  # L2 flush between timed steps (outside the events)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ev[i][0].record()
        res = pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)  # HOST result buffers filled inside
        ev[i][1].record()
        torch.cuda.synchronize()
        wall.append(time.perf_counter() - t0)
        results.append(res)
    barrier()
    clocks = sampler.finish()
    dev_ms = [a.elapsed_time(b) for a, b in ev]
    kern_ms = [r["device_ms"] for r in results]
    agg = replicas.aggregate(sum(dev_ms), sum(wall) * 1e3, float(sum(r["children"] for r in results)),
                             dist=dist if world > 1 else None, device=f"cuda:{local}")
    value, e2e = agg["value"], agg["e2e"]
    ms_per_step = agg["device_ms"] / args.steps

    if rank == 0:
        # roofline of the one kernel (ALU-bound: DESIGN.md "Roofline")
        ops = [algorithmic_ops(problem, r["nn_pairs"], r["children"]) for r in results]
        alg = sum(o["nn"] + o["prop"] for o in ops)
        launch_s = sum(kern_ms) * 1e-3
        sm_max = clocks["sm_max_mhz"] or 1965.0
        peak = 148 * 128 * sm_max * 1e6 / 1e12
        achieved = alg / launch_s / 1e12
        first = [r["first_solution_ms"] for r in results if r["first_solution_ms"] >= 0]
        # best cost at 100 ms (BASELINE metric, part 3): unlimited replans under a device time budget
        best100 = [pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, 4096, time_budget_ms=100.0)["cost"] for s in range(5)]
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": WORKLOAD, "dynamics": problem.name, "B": cfg.B, "K": cfg.K,
                       "tree_capacity": cfg.tree_capacity, "n_replans": cfg.n_replans,
                       "seeds": f"rank + {world} * step", "l2": "flushed between timed steps (256 MiB fill)",
                       "parallelism": f"replicas x{world}"},
            "clocks": clocks,
            "e2e": {"value": e2e, "unit": UNIT, "h2d_bytes_per_step": 4 * pl.Dp + 4,
                    "d2h_bytes_per_step": int(np.mean([1700 + 4 * r["path_len"] * (1 + pl.D + pl.m) for r in results]))},
            "gpu_launches": args.steps,
            "roofline": {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlaneop/s (fp32 lane-instructions)",
                         "frac": achieved / peak, "traffic": NCU_TRAFFIC_BYTES_PER_LAUNCH,
                         "kernel": "pakr_loop_kernel<DI3,BOX>", "avg_launch_ms": 1e3 * launch_s / args.steps,
                         "algorithmic_ops_per_launch": alg / args.steps,
                         "nn_share_of_ops": sum(o["nn"] for o in ops) / alg,
                         "nn_fma_pipe_frac": sum(r["nn_pairs"] for r in results) * 2 * problem.state_dim / launch_s / 1e12 / peak,
                         "peak_basis": f"148 SM x 4 schedulers x 32 lanes x {sm_max:.0f} MHz issue slots (= FMA-pipe lane-ops/s)",
                         "frac_at_measured_clock": (achieved / (148 * 128 * clocks['sm_mhz'] * 1e6 / 1e12))
                         if clocks["sm_mhz"] else None},
            "first_solution_ms_median": statistics.median(first) if first else None,
            "best_cost_at_100ms_median": statistics.median(best100),
            "final_cost_median": statistics.median(r["cost"] for r in results),
            "iterations_per_step": float(np.mean([r["iterations"] for r in results])),
            "phase_share": {k: sum(r["phase_ms"][i] for r in results) / sum(kern_ms)
                            for i, k in enumerate(("nn_tail_scan", "propagate_and_nn_lookahead", "insert_and_fused_tail"))},
            "inserted_nodes_per_s": sum(r["inserted"] for r in results) / (sum(dev_ms) * 1e-3),
            "solved": sum(r["outcome"] for r in results),
        }
        if not args.no_cpu_baseline and world == 1:
            cb = oracle_sample(problem, cfg, 0)
            line["cpu_baseline"] = {"value": cb["value"], "unit": UNIT, "cores": 1, "kind": "oracle",
                                    "sample": f"replan 0 (first solution) of {WORKLOAD}, planner seed 0: "
                                              f"{cb['iterations']} iterations, {cb['children']} children in {cb['seconds']:.1f} s",
                                    "first_solution_ms": cb["first_solution_ms"]}
        print(json.dumps(line), flush=True)
    pl.close()
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
