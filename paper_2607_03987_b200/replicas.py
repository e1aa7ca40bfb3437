"""Multi-GPU form of the PAKR hot path: replicas only.

One tree's iteration does not shard (every query needs the whole snapshot, iterations are tens of
microseconds long), so N GPUs run N independent planners on disjoint planner seeds -- the coarse-grained
parallel form the paper cites (independent planner instances).  There is no data-path
collective; the only communication is the timing harness: a barrier and two scalar all-reduces.
This module holds that host logic so that it can be tested with the gloo backend on CPU.
"""
from __future__ import annotations

from typing import Sequence


def replica_seeds(rank: int, world: int, count: int, first: int = 0) -> list[int]:
    """Planner seeds of one rank: first + rank, first + rank + world, ...  Disjoint across ranks and, over
    all ranks, exactly first .. first + world*count - 1."""
    if not (0 <= rank < world) or count < 0:
        raise ValueError("need 0 <= rank < world and count >= 0")
    return [first + rank + world * i for i in range(count)]


def aggregate(device_ms: float, wall_ms: float, units: float, dist=None, device=None) -> dict:
    """Whole-job numbers from per-rank totals: time = MAX over ranks (device and wall clock), units = SUM over
    ranks.  `dist` is torch.distributed (initialised) or None for a single process."""
    import torch
    t = torch.tensor([device_ms, wall_ms, units], dtype=torch.float64, device=device)
    tmax, tsum = t.clone(), t.clone()
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
        dist.all_reduce(tsum, op=dist.ReduceOp.SUM)
    dev, wall, tot = float(tmax[0]), float(tmax[1]), float(tsum[2])
    return {"device_ms": dev, "wall_ms": wall, "units": tot,
            "value": tot / (dev * 1e-3) if dev > 0 else 0.0,
            "e2e": tot / (wall * 1e-3) if wall > 0 else 0.0}


def best_of_replicas(costs: Sequence[float], dist=None, device=None) -> float:
    """First/best solution wins: the minimum cost over all replicas' results."""
    import torch
    local = min(costs) if len(costs) else float("inf")
    t = torch.tensor([local], dtype=torch.float64, device=device)
    if dist is not None and dist.is_initialized() and dist.get_world_size() > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MIN)
    return float(t[0])


def shared_bound_rounds(plan_fn, rounds: int, dist=None, device=None) -> dict:
    """Replicas that share the cost bound between rounds (C-FOREST-style).

    plan_fn(bound, round) -> (cost, payload) runs this rank's planner for one round under `bound` (+inf = none;
    with the CUDA library: pakr_plan(..., initial_cost_bound=bound), a different seed per rank and round) and
    returns the cost it found (+inf if nothing cheaper) with anything describing the plan.  After every round
    one scalar MIN all-reduce makes the best cost of ANY replica the bound of ALL replicas for the next round:
    4-8 bytes per round over NCCL / NVLink, latency-bound, never on the per-iteration path.
    Returns {"cost": global best, "payload": this rank's plan for its own best cost, "owner": whether this rank
    holds a plan achieving the global best, "history": global best after each round}."""
    bound = float("inf")
    my_cost, my_payload, history = float("inf"), None, []
    for rnd in range(rounds):
        cost, payload = plan_fn(bound, rnd)
        if cost < my_cost:
            my_cost, my_payload = cost, payload
        bound = min(bound, best_of_replicas([my_cost], dist=dist, device=device))
        history.append(bound)
    return {"cost": bound, "payload": my_payload, "owner": my_cost == bound and my_payload is not None,
            "history": history}
