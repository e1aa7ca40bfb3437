#!/usr/bin/env python
"""BASELINE.json metrics over seeds: expanded nodes/s, median ms to first solution, best cost at 100 ms.

  configs  C1-C4 at their BASELINE sizes (and the NEXT-2 workloads N1-N3): first-solution time (replan 0, device clock), cost after all
           replans, best cost under a 100 ms device budget; medians over planner seeds 0..N-1
  c5       BASELINE config 5: the B x K scaling sweep on the 6D double integrator with 128 boxes
           (first solution only, like the paper's Table IV)

One JSON line per row.  Every plan comes back through pakr_plan (C ABI); nothing here computes.

  pathlen  C1, C2 with cost = path length (the paper's Table II metric): AO-x cost-vs-time curve

  python -m paper_2607_03987_b200.sweep [--seeds N] [--what configs|c5|all|pathlen]
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys

sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))

from paper_2607_03987_b200 import workloads as wl  # noqa: E402


def med(v):
    v = [x for x in v if x is not None]
    return statistics.median(v) if v else None


def run_configs(pakr, seeds, path_length=False):
    import dataclasses
    for name in (("C1", "C2") if path_length else ("C1", "C2", "C3", "C4", "N1", "N2", "N3")):
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
        print(json.dumps({"row": "config", "workload": p.name if path_length else name, "B": cfg.B, "K": cfg.K, "replans": cfg.n_replans,
                          "seeds": seeds, "solved": solved, "first_solution_ms_median": med(first),
                          "first_solution_nodes_median": med(nodes1), "first_cost_median": med(cost1),
                          "final_cost_median": med(costf), "all_replans_ms_median": med(ms_all),
                          "iterations_median": med(iters), "expanded_nodes_per_s_median": med(rate),
                          "best_cost_at_100ms_median": med(best100),
                          # cost-vs-time curve of AO-x (Table II, Fig. 2): median over seeds of c_best
                          # and of the device time at the end of each replan
                          "cost_after_replan_median": [med(c) for c in zip(*curve_c)],
                          "ms_at_end_of_replan_median": [med(t) for t in zip(*curve_t)]}), flush=True)
        pl.close()


def run_c5(pakr, seeds):
    p, _ = wl.config5()
    pl = pakr.Planner(p)
    for B in (256, 1024, 4096, 16384):
        for K in (1, 4, 16, 64):
            cap = 1 << 23 if B * K >= (1 << 18) else 1 << 21
            pl.plan(1000, B, K, cap, 1)
            first, nodes, iters, rate, nn_share, solved = [], [], [], [], [], 0
            for s in range(seeds):
                r = pl.plan(s, B, K, cap, 1)
                solved += r["outcome"]
                if r["outcome"]:
                    first.append(r["first_solution_ms"])
                nodes.append(r["final_tree_nodes"])
                iters.append(r["iterations"])
                rate.append(r["children"] / (r["device_ms"] * 1e-3))
                nn_share.append((r["phase_ms"][0] + r["phase_ms"][1]) / r["device_ms"])
            print(json.dumps({"row": "c5", "B": B, "K": K, "children_per_iter": B * K, "tree_capacity": cap,
                              "seeds": seeds, "solved": solved, "first_solution_ms_median": med(first),
                              "iterations_median": med(iters), "nodes_median": med(nodes),
                              "expanded_nodes_per_s_median": med(rate),
                              "share_of_time_in_scan_and_propagate_phases": med(nn_share)}), flush=True)
    pl.close()


def main():
    from paper_2607_03987_b200 import pakr
    ap = argparse.ArgumentParser()
    ap.add_argument("--seeds", type=int, default=10)
    ap.add_argument("--what", default="all", choices=["configs", "c5", "all", "pathlen"])
    args = ap.parse_args()
    pakr.lib()
    if args.what in ("configs", "all"):
        run_configs(pakr, args.seeds)
    if args.what == "pathlen":
        run_configs(pakr, args.seeds, path_length=True)
    if args.what in ("c5", "all"):
        run_c5(pakr, args.seeds)


if __name__ == "__main__":
    main()
