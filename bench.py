#!/usr/bin/env python
"""bench.py -- measurements of the PAKR hot path on B200 (contract: DESIGN.md "Measurement").

Default mode (`--what bench`): a "step" is one pass of the whole hot path, i.e. one pakr_plan call (AO-x
replanning around the batched expansion iteration, every row of SURVEY.md 8(a)) on the LARGEST single-GPU
config of BASELINE.json, configs[3] = C4 (12-D quadrotor, 128 cylinders, B=4096, K=16, cap 2^22, 30 replans),
planner seed = step index.  metric = expanded nodes/s = children propagated and checked per second
(B*K*iterations / time).  The other configs (C1-C3 and one C5 point) are reported as extra keys of the same line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference]
  python bench.py --what peak                 measured FFMA / FFMA2 rates (the ALU roofline's denominators)
  python bench.py --what phases [--only nn|filter|stream|prop] [--quick]   single phases through pakr_expand_step
  python bench.py --what sweep|c5|pathlen [--seeds N]                  BASELINE metrics over seeds, config 5 sweep
  python bench.py --what oracle-c5            the oracle on config 5's small points: ns per (query, node) pair / child step

With --gpus N > 1 and no RANK in the environment it starts the N ranks itself (torch.distributed.run, one
planner replica per GPU, NCCL only for the timing harness' scalar reductions).
"""
from __future__ import annotations

import argparse
import dataclasses
import json
import multiprocessing as mp
import os
import socket
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

from paper_2607_03987_b200 import peak, replicas, workloads as wl  # noqa: E402

WORKLOAD = "C4"
METRIC = "expanded nodes/s"
UNIT = "nodes/s"
C5_POINT = (4096, 16)  # the fixed config-5 point reported beside the headline
# dram__bytes_read.sum + dram__bytes_write.sum of one pakr_loop_kernel launch on WORKLOAD, from the
# `ncu --set full` capture summarised in profiles/ (None until a capture exists for the current kernel).
NCU_TRAFFIC_BYTES_PER_LAUNCH = 79737088  # profiles/r03_ncu_c4_bench.md: 1,630,720 read + 78,106,368 written
NOMINAL_LANES = 148 * 4 * 32  # SMs x schedulers x lanes: issue slots per clock = fp32 FMA lanes per clock

# Arithmetic of one evaluation of f(x, u), counted on the formulas of DESIGN.md "Readings" Q / P33 / P34 with every
# multiply-add fused (one lane-op each), a sine/cosine pair as 2, a reciprocal as 1 (DESIGN.md "Measurement" has
# the count line by line).
F_DYN = {wl.DYN_DOUBLE_INTEGRATOR: 0, wl.DYN_UNICYCLE2: 4, wl.DYN_QUADROTOR: 37, wl.DYN_DUBINS_AIRPLANE: 8,
         wl.DYN_UNICYCLE1: 4, wl.DYN_QUADROTOR_BODY: 59, wl.DYN_ACROBOT: 24}


def nn_ops_per_pair(problem) -> int:
    """D sub + D fma + compare + select per (query, node) pair (+ D mul if weighted, +2 per angle
    dim for the wrap)."""
    D = problem.state_dim
    weighted = not np.all(problem.nn_weight == 1.0)
    return 2 * D + 2 + (D if weighted else 0) + 2 * int((problem.dim_kind == 1).sum())


def prop_ops_per_child(problem) -> int:
    """S steps of: stages * f + integrator combination (RK4: 7 fused ops per dim; Euler: 1) + closed-box test
    (2 compares + 1 combine per bounded dim) + obstacle broad phase (cell index and header: 10) + ONE obstacle
    test (the exact grid culls the rest)."""
    D = problem.state_dim
    rk4 = problem.integrator == wl.INT_RK4
    n_bounded = int((np.isfinite(problem.state_lo) & (problem.dim_kind == 0)).sum())
    c_obs = 2 * problem.pos_dim if problem.obstacle_type == wl.OBS_AABB else 5
    per_step = (4 if rk4 else 1) * F_DYN[problem.dynamics_id] + (7 if rk4 else 1) * D + 3 * n_bounded + 10 + c_obs
    return problem.steps_per_edge * per_step


def algorithmic_ops(problem, nn_pairs: int, children: int) -> dict:
    a, b = nn_ops_per_pair(problem), prop_ops_per_child(problem)
    return dict(nn=nn_pairs * a, prop=children * b, nn_per_pair=a, per_child=b)


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


# ---------------------------------------------------------------------------------------------------------
# CPU oracle, timed as it stands (BASELINE.md "CPU-baseline plan"): single-threaded fp64
# C++, one process PINNED to one core for latency, expansions/s and per-phase shares, plus a seed fan-out over
# every core the process may run on (count read at run time) for the aggregate rate.  Child processes are
# spawned (never forked: the parent may hold a CUDA context) and import only numpy + the oracle.
# ---------------------------------------------------------------------------------------------------------
def _workload(name: str):
    if name == "C5":
        return wl.config5(B=C5_POINT[0], K=C5_POINT[1])
    return wl.CONFIGS[name]()


def _oracle_worker(job):
    name, seed, budget_ms, core = job
    if core is not None:
        try:
            os.sched_setaffinity(0, {core})
        except OSError:
            core = None
    from oracle import pakr_oracle as orc
    problem, cfg = _workload(name)
    op = orc.OracleProblem(problem)
    t0 = time.perf_counter()
    # replan 0 (first solution) under a wall-clock cap: the oracle checks the cap between iterations
    res = orc.plan(op, seed, cfg.B, cfg.K, cfg.tree_capacity, 1, time_budget_ms=budget_ms)
    dt = time.perf_counter() - t0
    return dict(seconds=dt, children=res["children"], iterations=res["iterations"], solved=res["outcome"],
                nodes=int(res["replan_nodes"][0]), first_solution_ms=res["first_solution_ms"], cost=res["cost"],
                phase_ms=res["phase_ms"], core=core)


def oracle_baseline(name: str, budget_s: float, fanout: bool, seed: int = 0) -> dict:
    """-> cpu_baseline object for workload `name`."""
    from oracle import pakr_oracle as orc
    orc.build()  # before the children race to build it
    cores = sorted(os.sched_getaffinity(0))
    ctx = mp.get_context("spawn")
    with ctx.Pool(1) as pool:
        one = pool.map(_oracle_worker, [(name, seed, budget_s * 1e3, cores[0])])[0]
    ph = one["phase_ms"]
    tot = sum(ph) or 1.0
    how = ("to its first solution" if one["solved"] else f"cut off by the {budget_s:.0f} s cap")
    out = {"value": one["children"] / one["seconds"], "unit": UNIT, "cores": 1, "kind": "oracle",
           "pinned_core": one["core"],
           "sample": f"replan 0 of {name}, planner seed {seed}, {how}: {one['iterations']} iterations, "
                     f"{one['children']} children, tree {one['nodes']} nodes in {one['seconds']:.1f} s",
           "phase_share": {"nn": ph[0] / tot, "propagate_validity_prune": ph[1] / tot, "insert": ph[2] / tot},
           "first_solution_ms": one["first_solution_ms"] if one["solved"] else None}
    if fanout and len(cores) > 1:
        t0 = time.perf_counter()
        with ctx.Pool(len(cores)) as pool:
            rows = pool.map(_oracle_worker, [(name, seed + 1 + i, budget_s * 1e3, c) for i, c in enumerate(cores)], 1)
        wall = time.perf_counter() - t0
        out["all_cores"] = {"cores": len(cores), "value": sum(r["children"] for r in rows) / max(r["seconds"] for r in rows),
                            "unit": UNIT, "sample": f"{len(cores)} pinned single-thread replicas, planner seeds "
                                                    f"{seed + 1}..{seed + len(cores)}, same cap; wall {wall:.1f} s"}
    return out


def _oracle_c5_worker(job):
    """Replan 0 of config 5 at (B, K) driven iteration by iteration, so the (query, node) pairs each NN call really
    scored are known: -> oracle ns per pair and per child step.  Stops at the first solution or the wall-clock cap."""
    B, K, seed, budget_s, core = job
    if core is not None:
        try:
            os.sched_setaffinity(0, {core})
        except OSError:
            pass
    from oracle import pakr_oracle as orc
    problem, cfg = wl.config5(B=B, K=K)
    op = orc.OracleProblem(problem)
    tree = orc.OracleTree(op, cfg.tree_capacity)
    tree.reset()
    pairs = children = it = 0
    ph = [0.0, 0.0, 0.0]
    solved = False
    t0 = time.perf_counter()
    while time.perf_counter() - t0 < budget_s and tree.n < cfg.tree_capacity:
        pairs += B * tree.n
        out = orc.expand_iteration(op, tree, seed, 0, it, B, K)
        children += B * K
        it += 1
        for i in range(3):
            ph[i] += out["phase_ms"][i]
        if out["goal"]:
            solved = True
            break
    return dict(B=B, K=K, seed=seed, seconds=time.perf_counter() - t0, iterations=it, nodes=tree.n, solved=solved,
                pairs=pairs, children=children, nn_ms=ph[0], prop_ms=ph[1], insert_ms=ph[2],
                steps_per_edge=problem.steps_per_edge, D=problem.state_dim)


def run_oracle_c5(args):
    """--what oracle-c5: SURVEY.md 8(d) / BASELINE.md's CPU plan for config 5 -- the oracle as it stands on B in {256,
    1024} x K in {1, 4}, 3 planner seeds, one pinned core, with its cost per (query, node) pair and per child step, so
    the figures for C4 / the large C5 points are stated extrapolations instead of implied ones."""
    from oracle import pakr_oracle as orc
    orc.build()
    core = sorted(os.sched_getaffinity(0))[0]
    ctx = mp.get_context("spawn")
    rows = []
    with ctx.Pool(1) as pool:
        for B in (256, 1024):
            for K in (1, 4):
                for seed in range(3):
                    r = pool.map(_oracle_c5_worker, [(B, K, seed, 10.0, core)])[0]
                    r["ns_per_pair"] = 1e6 * r["nn_ms"] / max(1, r["pairs"])
                    r["ns_per_child_step"] = 1e6 * r["prop_ms"] / max(1, r["children"] * r["steps_per_edge"])
                    r["nodes_per_s"] = r["children"] / r["seconds"]
                    rows.append(r)
                    print(json.dumps({"what": "oracle-c5", **r}), flush=True)
    pp = statistics.median(r["ns_per_pair"] for r in rows if r["pairs"] > 1e6)
    pc = statistics.median(r["ns_per_child_step"] for r in rows)
    # extrapolation to the headline: per-plan totals of C4 from the GPU's own counters are not available here, so the
    # statement is per unit: a (query, node) pair of D = 6 costs pp ns, a child step pc ns; C4 (D = 12, RK4) scales the
    # pair cost by ~2 and is measured directly by the cpu_baseline leg.
    print(json.dumps({"what": "oracle-c5-summary", "median_ns_per_pair_D6": pp, "median_ns_per_child_step": pc,
                      "cores": 1, "cap_s_per_run": 10.0, "runs": len(rows),
                      "example": "C5 B=4096 K=16 iteration on a 100 k-node tree = 4.1e8 pairs -> %.1f s of NN alone" % (4.096e8 * pp * 1e-9)}),
          flush=True)


def run_reference(args):
    """--impl reference: the oracle on the box's host cores, same metric and config (tier rule)."""
    if int(os.environ.get("RANK", "0")) != 0:
        return
    problem, cfg = _workload(args.workload)
    budget_s = 12.0
    steps = max(1, min(args.steps, 8))  # ~12 s of CPU per step: the whole run stays within minutes
    ctx = mp.get_context("spawn")
    cores = sorted(os.sched_getaffinity(0))
    from oracle import pakr_oracle as orc
    orc.build()
    rows = []
    with ctx.Pool(1) as pool:
        for i in range(min(args.warmup, 1)):
            pool.map(_oracle_worker, [(args.workload, 1000 + i, 2e3, cores[0])])  # one short untimed pass
        for i in range(steps):
            rows += pool.map(_oracle_worker, [(args.workload, i, budget_s * 1e3, cores[0])])
    t_total = sum(r["seconds"] for r in rows)
    value = sum(r["children"] for r in rows) / t_total
    sample = (f"per step: replan 0 of {args.workload} under a {budget_s:.0f} s wall-clock cap, planner seed = step; "
              f"one pinned core")
    firsts = [r["first_solution_ms"] for r in rows if r["solved"]]
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": steps, "warmup": args.warmup, "ms_per_step": 1e3 * t_total / steps,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": args.workload, "dynamics": problem.name, "B": cfg.B, "K": cfg.K,
                       "tree_capacity": cfg.tree_capacity, "n_replans": cfg.n_replans, "sampled": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "first_solution_ms_median": statistics.median(firsts) if firsts else None,
            "solved": len(firsts)}
    print(json.dumps(line), flush=True)


# ---------------------------------------------------------------------------------------------------------
def time_plans(torch, pl, cfg, seeds, flush, n_replans=None):
    """Times one pakr_plan per seed: CUDA events on the launching stream (device) and the host clock around the
    same call (end to end: HOST buffers in, HOST result out).  L2 is flushed between steps, outside the events."""
    R = cfg.n_replans if n_replans is None else n_replans
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in seeds]
    results, wall = [], []
    for i, s in enumerate(seeds):
        flush.fill_(i & 0xFF)
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        ev[i][0].record()
        res = pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, R)
        ev[i][1].record()
        torch.cuda.synchronize()
        wall.append(time.perf_counter() - t0)
        results.append(res)
    return results, [a.elapsed_time(b) for a, b in ev], wall


def roofline_of(problem, results, dev_ms, sm_max_mhz, measured_peak) -> dict:
    """ALU roofline of the launch.  `achieved` / `frac` count the fp32 lane-ops the kernel's own method EXECUTES:
    (query, node) distances actually evaluated (pakr_stats.nn_pairs_evaluated: all B*n under the scan tiers, the
    rows of opened tiles under the NN index, the rescored rows under the filter) x ops per pair + children x ops per
    child.  Box-bound tests, Morton keys and the radix sort of the index are NOT counted, so frac is a lower bound of
    the utilisation and can never exceed 1.  The brute-force B*n-pair count of SURVEY.md 8(d) is kept beside it as
    `algorithmic_equiv_*`: how fast a plain scan would have had to run to match (it may exceed 1)."""
    ops = [algorithmic_ops(problem, r["nn_pairs"], r["children"]) for r in results]
    alg = sum(o["nn"] + o["prop"] for o in ops)
    launch_s = sum(dev_ms) * 1e-3
    peak = NOMINAL_LANES * sm_max_mhz * 1e6 / 1e12
    ev = sum(r.get("nn_pairs_evaluated", r["nn_pairs"]) for r in results)
    tot = sum(r["nn_pairs"] for r in results)
    exe_ops = ev * ops[0]["nn_per_pair"] + sum(o["prop"] for o in ops)
    achieved = exe_ops / launch_s / 1e12
    alg_achieved = alg / launch_s / 1e12
    out = {"bound": "alu", "achieved": achieved, "peak": peak, "unit": "Tlaneop/s (fp32 lane-instructions)",
           "frac": achieved / peak, "traffic": None,
           "counts": "executed: distances actually evaluated x ops/pair + children x ops/child",
           "algorithmic_equiv_achieved": alg_achieved, "algorithmic_equiv_frac": alg_achieved / peak,
           "nn_pairs_evaluated_share": ev / tot if tot else 1.0,
           "avg_launch_ms": 1e3 * launch_s / len(results), "kernel_ms_by_globaltimer": float(np.mean([r["device_ms"] for r in results])),
           "executed_ops_per_launch": exe_ops / len(results),
           "algorithmic_ops_per_launch": alg / len(results), "nn_ops_per_pair": ops[0]["nn_per_pair"],
           "prop_ops_per_child": ops[0]["per_child"], "nn_share_of_ops": sum(o["nn"] for o in ops) / alg,
           "peak_basis": f"nominal: 148 SM x 4 schedulers x 32 lanes x {sm_max_mhz:.0f} MHz (clocks.max.sm)"}
    if measured_peak:
        out["peak_measured_ffma"] = measured_peak["ffma_lane_ops_per_s"] / 1e12
        out["frac_vs_measured_ffma"] = achieved / out["peak_measured_ffma"]
    return out


def summarize(results, dev_ms, wall):
    first = [r["first_solution_ms"] for r in results if r["first_solution_ms"] >= 0]
    kern = sum(r["device_ms"] for r in results)
    return {"first_solution_ms_median": statistics.median(first) if first else None,
            "final_cost_median": statistics.median(r["cost"] for r in results),
            "iterations_per_step": float(np.mean([r["iterations"] for r in results])),
            "replans_solved_per_step": float(np.mean([r["replans_solved"] for r in results])),
            "replans_run_per_step": float(np.mean([r["replans_run"] for r in results])),
            "phase_share": {k: sum(r["phase_ms"][i] for r in results) / kern
                            for i, k in enumerate(("nn_phases", "propagate_and_nn_lookahead", "insert_phases",
                                                   "nn_index_rebuilds"))},
            "inserted_nodes_per_s": sum(r["inserted"] for r in results) / (sum(dev_ms) * 1e-3),
            "solved": sum(r["outcome"] for r in results)}


def run_bench(args):
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
    problem, cfg = _workload(args.workload)
    pl = pakr.Planner(problem, local)
    ws = pl.workspace(cfg.B, cfg.K, cfg.tree_capacity)  # noqa: F841  (allocated before the timed region)
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=f"cuda:{local}")  # > 126 MB L2

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # replicas only: rank r plans seeds r, r + world, ...
    W = max(args.warmup, 3)
    seeds = replicas.replica_seeds(rank, world, W + args.steps)
    for s in seeds[:W]:
        pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    sampler = ClockSampler(local)
    barrier()
    sampler.start()
    barrier()
    results, dev_ms, wall = time_plans(torch, pl, cfg, seeds[W:], flush)
    barrier()
    clocks = sampler.finish()
    agg = replicas.aggregate(sum(dev_ms), sum(wall) * 1e3, float(sum(r["children"] for r in results)),
                             dist=dist if world > 1 else None, device=f"cuda:{local}")

    if rank == 0:
        sm_max = clocks["sm_max_mhz"] or 1965.0
        measured = peak.measure_fp32_peak(local)
        roof = roofline_of(problem, results, dev_ms, sm_max, measured)
        roof["traffic"] = NCU_TRAFFIC_BYTES_PER_LAUNCH
        roof["traffic_source"] = ("constant: dram read + written bytes of one launch in the ncu --set full capture "
                                  "profiles/r03_ncu_c4_bench.md, not measured in this run")
        roof["kernel"] = f"pakr_loop_kernel ({problem.name})"
        if clocks["sm_mhz"]:
            roof["frac_at_sampled_clock"] = roof["achieved"] / (NOMINAL_LANES * clocks["sm_mhz"] * 1e6 / 1e12)
        # best cost at 100 ms (BASELINE metric, part 3): unlimited replans under a device time budget
        best100 = [pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, 4096, time_budget_ms=100.0)["cost"] for s in range(5)]
        line = {
            "metric": METRIC, "value": agg["value"], "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": W, "ms_per_step": agg["device_ms"] / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
            "config": {"workload": args.workload, "dynamics": problem.name, "B": cfg.B, "K": cfg.K,
                       "tree_capacity": cfg.tree_capacity, "n_replans": cfg.n_replans,
                       "seeds": f"rank + {world} * step", "l2": "flushed between timed steps (256 MiB fill)",
                       "parallelism": f"replicas x{world}"},
            "clocks": clocks,
            "e2e": {"value": agg["e2e"], "unit": UNIT,  # bytes as counted by pakr_plan itself (pakr_stats)
                    "h2d_bytes_per_step": int(np.mean([r["h2d_bytes"] for r in results])),
                    "d2h_bytes_per_step": int(np.mean([r["d2h_bytes"] for r in results]))},
            "gpu_launches": args.steps,
            "roofline": roof,
            "best_cost_at_100ms_median": statistics.median(best100),
        }
        line.update(summarize(results, dev_ms, wall))
        # "PAKR without AO-x": one replan, ends at the first solution.  first_solution_ms_host is
        # SURVEY.md 8(d)'s definition -- host clock from pakr_plan entry to its return (memsets, cooperative launch, the
        # loop, the result copy) -- beside the device figure, which starts at kernel start.
        if not args.no_extras:
            r0, dev0, wall0 = time_plans(torch, pl, cfg, list(range(100, 105)), flush, n_replans=1)
            line["replan0"] = {"value": sum(r["children"] for r in r0) / (sum(dev0) * 1e-3), "unit": UNIT, "steps": 5,
                               "ms_per_step": sum(dev0) / 5, "solved": sum(r["outcome"] for r in r0),
                               "first_solution_ms_device_median": statistics.median(r["first_solution_ms"] for r in r0),
                               "first_solution_ms_host_median": 1e3 * statistics.median(wall0),
                               "iterations_per_step": float(np.mean([r["iterations"] for r in r0]))}
        pl.close()
        if not args.no_extras and world == 1:
            line["other_workloads"] = {}
            for name in ("C1", "C2", "C3", "C5"):
                p2, c2 = _workload(name)
                pl2 = pakr.Planner(p2, local)
                pl2.plan(999, c2.B, c2.K, c2.tree_capacity, c2.n_replans)
                res2, dev2, wall2 = time_plans(torch, pl2, c2, list(range(3)), flush)
                sm = summarize(res2, dev2, wall2)
                rf = roofline_of(p2, res2, dev2, sm_max, measured)
                # kept short on purpose: the driver records only the tail of this line
                row = {"B": c2.B, "K": c2.K, "n_replans": c2.n_replans,
                       "value": sum(r["children"] for r in res2) / (sum(dev2) * 1e-3),
                       "e2e": sum(r["children"] for r in res2) / sum(wall2), "ms_per_step": sum(dev2) / 3,
                       "first_solution_ms_median": sm["first_solution_ms_median"], "final_cost_median": sm["final_cost_median"],
                       "replans_solved_per_step": sm["replans_solved_per_step"],
                       "roofline_frac": rf["frac"],  # executed lane-ops / peak
                       "algorithmic_equiv_frac": rf["algorithmic_equiv_frac"]}
                if not args.no_cpu_baseline:
                    row["cpu_value"] = oracle_baseline(name, 4.0, fanout=False)["value"]  # oracle, 1 pinned core, 4 s cap
                line["other_workloads"]["C5 (B=%d, K=%d)" % C5_POINT if name == "C5" else name] = row
                pl2.close()
            # HBM-bound regime of the NN scan: B = 8 queries share one pass over n = 2^23 rows, D = 6
            p6, _ = wl.config2()
            pl6 = pakr.Planner(p6, local)
            n6 = 1 << 23
            ms6 = measure_phase(torch, pl6, p6, n6, 8, 1, 3, flush, nn_mode=pakr.NN_SCAN)[0]
            hbm = measured_hbm_gbs()
            line["stream_tier"] = {"D": 6, "B": 8, "n": n6, "ms": ms6, "algorithmic_GBps": 4 * 6 * n6 / (ms6 * 1e-3) / 1e9,
                                   "hbm_peak_GBps": hbm, "hbm_frac": 4 * 6 * n6 / (ms6 * 1e-3) / (hbm * 1e9)}
            pl6.close()
        if not args.no_cpu_baseline and world == 1:
            line["cpu_baseline"] = oracle_baseline(args.workload, 12.0, fanout=True)
        print(json.dumps(line), flush=True)
    else:
        pl.close()
    if world > 1:
        dist.destroy_process_group()


def run_peak(args):
    """Measured fp32 peaks: the denominators beside the nominal one in `roofline`."""
    from paper_2607_03987_b200 import pakr
    m = peak.measure_fp32_peak(0)
    nominal = NOMINAL_LANES * m["sm_clock_mhz"] * 1e6
    print(json.dumps({"what": "peak", "nominal_lane_ops_per_s": nominal, **m,
                      "ffma_frac_of_nominal": m["ffma_lane_ops_per_s"] / nominal,
                      "ffma2_frac_of_nominal": m["ffma2_lane_ops_per_s"] / nominal,
                      "scan_mix_frac_of_nominal": m["scan_mix_lane_ops_per_s"] / nominal,
                      "mma_f16_mac_per_clk_per_sm": m["mma_f16_mac_per_s"] / (m["sm_clock_mhz"] * 1e6) / m["sm_count"],
                      "mma_f16_minfold_mac_per_clk_per_sm": m["mma_f16_minfold_mac_per_s"] / (m["sm_clock_mhz"] * 1e6) / m["sm_count"]}),
          flush=True)


# ---------------------------------------------------------------------------------------------------------
# --what phases: one pakr_expand_step on a synthetic tree of n uniform-in-bounds nodes is one iteration whose
# phases the kernel times itself (pakr_read_stats: phase_ms[0] = NN scan of the whole tree, [1] = propagate
# (+ insert when B*K is small), [2] = insert as a phase of its own; each includes its grid barrier, ~1.2 us).
# ---------------------------------------------------------------------------------------------------------
def measure_phase(torch, pl, problem, n, B, K, reps, flush, nn_mode=0):
    host = wl.random_tree(problem, n, seed=n % 1000 + B, flat=True)
    cap = n + B * K
    tree = pl.new_tree(cap, host)
    ws = pl.workspace(B, K, cap)
    out = []
    for rep in range(reps + 1):
        tree["n_nodes"][0] = n
        if flush is not None:
            flush.fill_(rep)  # tree out of L2
        torch.cuda.synchronize()
        pl.expand_step(tree, 0, 0, rep, B, K, debug=False, workspace=ws, nn_mode=nn_mode)
        st = pl.read_stats(B, K, cap, workspace=ws)
        if rep:  # first call is the warm-up
            out.append(st["phase_ms"])
    return np.median(np.array(out), axis=0)


def measured_hbm_gbs() -> float:
    """Measured HBM copy bandwidth of this pool's B200s (driver-written MEASURED_PEAKS.json), else round 1's figure."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["hbm_gbs"])
    except Exception:
        return 6446.3


def run_phases(args):
    import torch
    from paper_2607_03987_b200 import pakr
    pakr.lib()
    peak = NOMINAL_LANES * 1.965e9
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    hbm_peak_gbs = measured_hbm_gbs()
    reps = 3 if args.quick else 7
    nn_points = [("C2", 1 << 16, 1024), ("C2", 1 << 20, 1024), ("C5", 1 << 20, 16384), ("C3", 1 << 20, 2048),
                 ("C4", 1 << 18, 4096), ("C4", 1 << 22, 4096)]
    if args.quick:
        nn_points = nn_points[1:3] + nn_points[5:]
    for name, n, B in (nn_points if args.only in ("", "nn", "filter") else []):
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        ops = nn_ops_per_pair(p)
        heavy_angles = float(p.nn_weight[p.dim_kind == 1].sum()) > 0.1  # such problems keep the fp32 scan (pakr.h)
        tiers = [("fp32 scan", pakr.NN_SCAN)] if args.only != "filter" else []
        if args.only in ("", "filter") and not heavy_angles:
            tiers.append(("tensor-core filter + exact rescoring", pakr.NN_FILTER))
        for tier, mode in tiers:
            ph = measure_phase(torch, pl, p, n, B, 1, reps, None, nn_mode=mode)
            t = (ph[0] + ph[3]) * 1e-3  # [3]: the filter's rescoring phase (0 for the scan)
            row = {"phase": "nn", "tier": tier, "workload": name, "D": p.state_dim, "n": n, "B": B, "ms": ph[0] + ph[3],
                   "pairs_per_s": B * n / t, "alg_lane_ops_per_pair": ops, "alu_frac": B * n * ops / t / peak,
                   "fma_pipe_frac": B * n * 2 * p.state_dim / t / peak, "tree_GBps": 4 * p.state_dim * n / t / 1e9}
            if mode == pakr.NN_FILTER:
                K = 32 if 3 * (p.state_dim + int((p.dim_kind == 1).sum()) + 1) <= 32 else 48
                row.update({"rescoring_ms": ph[3], "filter_K": K,
                            # tensor roofline of the first phase: K multiply-accumulates per pair against the measured
                            # mma.sync rate with the min-fold epilogue (bench.py --what peak)
                            "mma_mac_per_s": B * n * K / (ph[0] * 1e-3)})
            print(json.dumps(row), flush=True)
        pl.close()
    # HBM-bound regime: few queries share one pass over a tree > L2.  Algorithmic bytes = 4 * D * n.
    for name, B in ((("C2", 4), ("C2", 8), ("C4", 4), ("C4", 8)) if args.only in ("", "stream") else ()):
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        n = 1 << 23
        ph = measure_phase(torch, pl, p, n, B, 1, reps, flush, nn_mode=pakr.NN_SCAN)
        t = ph[0] * 1e-3
        print(json.dumps({"phase": "stream", "workload": name, "D": p.state_dim, "n": n, "B": B, "ms": ph[0],
                          "algorithmic_GBps": 4 * p.state_dim * n / t / 1e9,
                          "hbm_frac_of_measured": 4 * p.state_dim * n / t / (hbm_peak_gbs * 1e9), "hbm_peak_GBps": hbm_peak_gbs,
                          "alu_frac": B * n * nn_ops_per_pair(p) / t / peak,
                          "row_bytes_in_memory": 4 * p.state_dim, "l2": "flushed before every call"}), flush=True)
        pl.close()
    for name, B, K in ((("C2", 1024, 8), ("C3", 2048, 8), ("C4", 4096, 16), ("C5", 16384, 64)) if args.only in ("", "prop", "prop1") else ()):
        if (args.quick and name in ("C3",)) or (args.only == "prop1" and name != "C4"):
            continue
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        # tree of 4096 nodes: the launch also scans 4096 rows; tree of 1 node (--only prop1): the launch is the
        # propagate + insert alone, which is what an ncu capture of the executed instructions per child needs
        n_tree = 1 if args.only == "prop1" else 4096
        ph = measure_phase(torch, pl, p, n_tree, B, K, reps, None, nn_mode=pakr.NN_SCAN)
        t = ph[1] * 1e-3
        ops = prop_ops_per_child(p)
        print(json.dumps({"phase": "prop", "workload": name, "children": B * K, "tree_nodes": n_tree, "ms": ph[1], "insert_ms": ph[2],
                          "children_per_s": B * K / t, "alg_lane_ops_per_child": ops,
                          "alu_frac": B * K * ops / t / peak}), flush=True)
        pl.close()


# ---------------------------------------------------------------------------------------------------------
# --what sweep | c5 | pathlen: BASELINE.json metrics over planner seeds (medians), one JSON line per row.
# ---------------------------------------------------------------------------------------------------------
def med(v):
    v = [x for x in v if x is not None]
    return statistics.median(v) if v else None


def run_sweep_configs(pakr, seeds, path_length=False):
    for name in (("C1", "C2") if path_length else ("C1", "C2", "C3", "C4", "N1", "N2", "N3", "N4")):
        p, cfg = wl.CONFIGS[name]()
        if path_length:  # the paper's convergence metric (Table II, Fig. 2: cost = distance travelled)
            p = dataclasses.replace(p, cost_mode=wl.COST_PATH_LENGTH, heuristic_speed=1.0, name=p.name + "-pathlen")
        pl = pakr.Planner(p)
        pl.plan(1000, cfg.B, cfg.K, cfg.tree_capacity, 1)  # warm-up
        first, nodes1, cost1, costf, ms_all, iters, solved, rate = [], [], [], [], [], [], 0, []
        curve_c, curve_t = [], []
        for s in range(seeds):
            r = pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
            solved += r["outcome"]
            if r["first_solution_ms"] >= 0:
                k = int((r["replan_cost"] < float("inf")).argmax())
                first.append(r["first_solution_ms"])
                nodes1.append(int(r["replan_nodes"][k]))
                cost1.append(float(r["replan_cost"][k]))
            costf.append(r["cost"])
            curve_c.append([float(v) if v < float("inf") else None for v in r["replan_cost"]])
            curve_t.append([float(v) for v in r["replan_end_ms"]])
            ms_all.append(r["device_ms"])
            iters.append(r["iterations"])
            rate.append(r["children"] / (r["device_ms"] * 1e-3))
        best100 = [pl.plan(s, cfg.B, cfg.K, cfg.tree_capacity, 4096, time_budget_ms=100.0)["cost"]
                   for s in range(min(seeds, 10))]
        print(json.dumps({"row": "config", "workload": p.name if path_length else name, "B": cfg.B, "K": cfg.K,
                          "replans": cfg.n_replans, "seeds": seeds, "solved": solved,
                          "first_solution_ms_median": med(first), "first_solution_nodes_median": med(nodes1),
                          "first_cost_median": med(cost1), "final_cost_median": med(costf),
                          "all_replans_ms_median": med(ms_all), "iterations_median": med(iters),
                          "expanded_nodes_per_s_median": med(rate), "best_cost_at_100ms_median": med(best100),
                          # cost-vs-time curve of AO-x (Table II, Fig. 2): median over seeds of c_best
                          # and of the device time at the end of each replan
                          "cost_after_replan_median": [med(c) for c in zip(*curve_c)],
                          "ms_at_end_of_replan_median": [med(t) for t in zip(*curve_t)]}), flush=True)
        pl.close()


def run_sweep_c5(pakr, seeds):
    """BASELINE config 5: expansions/s, NN-scan HBM GB/s and time-to-first-solution at every (B, K)."""
    p, _ = wl.config5()
    pl = pakr.Planner(p)
    for B in (256, 1024, 4096, 16384):
        for K in (1, 4, 16, 64):
            cap = 1 << 23 if B * K >= (1 << 18) else 1 << 21
            pl.plan(1000, B, K, cap, 1)
            first, nodes, iters, rate, nn_share, gbps, solved = [], [], [], [], [], [], 0
            for s in range(seeds):
                r = pl.plan(s, B, K, cap, 1)
                solved += r["outcome"]
                if r["outcome"]:
                    first.append(r["first_solution_ms"])
                nodes.append(r["final_tree_nodes"])
                iters.append(r["iterations"])
                rate.append(r["children"] / (r["device_ms"] * 1e-3))
                nn_ms = r["phase_ms"][0] + r["phase_ms"][1]
                nn_share.append(nn_ms / r["device_ms"])
                # every iteration's NN reads its snapshot once: sum_i 4 D n_i = 4 D nn_pairs / B algorithmic bytes
                gbps.append(4 * p.state_dim * r["nn_pairs"] / B / (nn_ms * 1e-3) / 1e9 if nn_ms > 0 else None)
            print(json.dumps({"row": "c5", "B": B, "K": K, "children_per_iter": B * K, "tree_capacity": cap,
                              "seeds": seeds, "solved": solved, "first_solution_ms_median": med(first),
                              "iterations_median": med(iters), "nodes_median": med(nodes),
                              "expanded_nodes_per_s_median": med(rate),
                              "nn_scan_tree_GBps_median": med(gbps),
                              "share_of_time_in_scan_and_propagate_phases": med(nn_share)}), flush=True)
    pl.close()


def run_sweep(args):
    from paper_2607_03987_b200 import pakr
    pakr.lib()
    if args.what == "sweep":
        run_sweep_configs(pakr, args.seeds)
    elif args.what == "pathlen":
        run_sweep_configs(pakr, args.seeds, path_length=True)
    elif args.what == "c5":
        run_sweep_c5(pakr, args.seeds)


def spawn_ranks(args) -> int:
    """`python bench.py --gpus N` started by hand: launch the N ranks exactly as the driver would."""
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
           "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
    return subprocess.call(cmd)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--what", default="bench", choices=["bench", "peak", "phases", "sweep", "c5", "pathlen", "oracle-c5"])
    ap.add_argument("--workload", default=WORKLOAD, choices=["C1", "C2", "C3", "C4", "C5"],
                    help="headline workload of --what bench (default: the largest single-GPU config)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extras", action="store_true", help="skip the other_workloads rows")
    ap.add_argument("--seeds", type=int, default=10, help="--what sweep|c5|pathlen: planner seeds per row")
    ap.add_argument("--quick", action="store_true", help="--what phases: fewer points and repetitions")
    ap.add_argument("--only", default="", help="--what phases: nn | filter | stream | prop | prop1")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    if args.what == "oracle-c5":
        return run_oracle_c5(args)
    if args.what == "peak":
        return run_peak(args)
    if args.what == "phases":
        return run_phases(args)
    if args.what in ("sweep", "c5", "pathlen"):
        return run_sweep(args)
    if args.gpus > 1 and "RANK" not in os.environ:
        sys.exit(spawn_ranks(args))
    return run_bench(args)


if __name__ == "__main__":
    main()
