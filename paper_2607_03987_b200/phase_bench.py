#!/usr/bin/env python
"""Per-phase measurements of the PAKR iteration on one B200.

One `pakr_expand_step` on a synthetic tree of n uniform-in-bounds nodes (workloads.random_tree, flat) is
one iteration whose three phases are timed on the device by the kernel itself (`pakr_read_stats`:
phase_ms[0] = NN scan of the whole tree, [1] = propagate (+ insert when B*K is small), [2] = insert as a phase
of its own; each includes its grid barrier, about 1.2 us).  Prints one JSON line per point:

  nn     B x n (query, node) pairs: pairs/s, algorithmic fp32 lane-ops/s against the issue-slot peak,
         and the DRAM-side GB/s the scan would need if the tree were streamed once (4*Dp*n bytes)
  stream the regime where HBM binds: B = 8 queries, n = 2^23 (tree 268-403 MB > 126 MB L2)
  prop   B*K children: children/s and algorithmic lane-ops/s of propagate + validity + prune

  python -m paper_2607_03987_b200.phase_bench [--quick] [--only nn|stream|prop]
"""
from __future__ import annotations

import argparse
import json
import os
import sys

import numpy as np

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_2607_03987_b200 import workloads as wl  # noqa: E402

PEAK_LANE_OPS = 148 * 4 * 32 * 1.965e9  # issue slots: 148 SMs x 4 schedulers x 32 lanes x clocks.max.sm


def nn_ops_per_pair(problem) -> int:
    D = problem.state_dim
    weighted = not np.all(problem.nn_weight == 1.0)
    return 2 * D + 2 + (D if weighted else 0) + 2 * int((problem.dim_kind == 1).sum())


def prop_ops_per_child(problem) -> int:
    D = problem.state_dim
    f_dyn = {wl.DYN_DOUBLE_INTEGRATOR: 0, wl.DYN_UNICYCLE2: 25, wl.DYN_QUADROTOR: 140, wl.DYN_DUBINS_AIRPLANE: 50,
             wl.DYN_UNICYCLE1: 24, wl.DYN_QUADROTOR_BODY: 170}[problem.dynamics_id]
    stages = 4 if problem.integrator == wl.INT_RK4 else 1
    integ = 8 * D if problem.integrator == wl.INT_RK4 else 2 * D
    n_bounded = int((np.isfinite(problem.state_lo) & (problem.dim_kind == 0)).sum())
    c_obs = 2 * problem.pos_dim if problem.obstacle_type == wl.OBS_AABB else 5
    # obstacle term: broad-phase cell lookup (10 ops) + one obstacle test; the grid culls the rest exactly
    return problem.steps_per_edge * (stages * f_dyn + integ + 2 * n_bounded + 10 + c_obs)


def measure(pl, problem, n, B, K, reps, flush):
    import torch
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
        pl.expand_step(tree, 0, 0, rep, B, K, debug=False, workspace=ws)
        st = pl.read_stats(B, K, cap, workspace=ws)
        if rep:  # first call is the warm-up
            out.append(st["phase_ms"])
    return np.median(np.array(out), axis=0)


def main():
    import torch
    from paper_2607_03987_b200 import pakr
    ap = argparse.ArgumentParser()
    ap.add_argument("--quick", action="store_true")
    ap.add_argument("--only", default="", help="nn | stream | prop: run that phase's points only (ncu captures)")
    args = ap.parse_args()
    pakr.lib()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")
    reps = 3 if args.quick else 7
    nn_points = [("C2", 1 << 16, 1024), ("C2", 1 << 20, 1024), ("C5", 1 << 20, 16384), ("C3", 1 << 20, 2048),
                 ("C4", 1 << 18, 4096), ("C4", 1 << 22, 4096)]
    if args.quick:
        nn_points = nn_points[1:3] + nn_points[5:]
    for name, n, B in (nn_points if args.only in ("", "nn") else []):
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        ph = measure(pl, p, n, B, 1, reps, None)
        t = ph[0] * 1e-3
        ops = nn_ops_per_pair(p)
        print(json.dumps({"phase": "nn", "workload": name, "D": p.state_dim, "n": n, "B": B, "ms": ph[0],
                          "pairs_per_s": B * n / t, "alg_lane_ops_per_pair": ops,
                          "alu_frac": B * n * ops / t / PEAK_LANE_OPS,
                          "fma_pipe_frac": B * n * 2 * p.state_dim / t / PEAK_LANE_OPS,
                          "tree_GBps": 4 * p.state_stride * n / t / 1e9}), flush=True)
        pl.close()
    for name, B in ((("C2", 8), ("C4", 8), ("C4", 4)) if args.only in ("", "stream") else ()):  # HBM-bound regime: few queries share one pass over a tree > L2
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        n = 1 << 23
        ph = measure(pl, p, n, B, 1, reps, flush)
        t = ph[0] * 1e-3
        print(json.dumps({"phase": "stream", "workload": name, "D": p.state_dim, "n": n, "B": B, "ms": ph[0],
                          "tree_GBps": 4 * p.state_stride * n / t / 1e9, "hbm_frac_of_measured_6446": 4 * p.state_stride * n / t / 6446.3e9,
                          "l2": "flushed before every call"}),
              flush=True)
        pl.close()
    for name, B, K in ((("C2", 1024, 8), ("C3", 2048, 8), ("C4", 4096, 16), ("C5", 16384, 64)) if args.only in ("", "prop") else ()):
        if args.quick and name in ("C3",):
            continue
        p, _ = wl.CONFIGS[name]()
        pl = pakr.Planner(p)
        ph = measure(pl, p, 4096, B, K, reps, None)
        t = ph[1] * 1e-3
        ops = prop_ops_per_child(p)
        print(json.dumps({"phase": "prop", "workload": name, "children": B * K, "ms": ph[1], "insert_ms": ph[2],
                          "children_per_s": B * K / t, "alg_lane_ops_per_child": ops,
                          "alu_frac": B * K * ops / t / PEAK_LANE_OPS}), flush=True)
        pl.close()


if __name__ == "__main__":
    main()
