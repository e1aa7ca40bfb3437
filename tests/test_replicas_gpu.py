"""NEXT-4 on real processes (C-FOREST-style sharing of the cost bound): two planner PROCESSES on
cuda:0, each running pakr_plan through the C ABI, exchange their best cost between rounds with one scalar MIN
all-reduce (gloo here; NCCL on a multi-GPU node).  The second round of every replica must run under the global best
of the first.  The two processes take turns on the GPU (a barrier between their launches): a persistent cooperative
kernel owns every SM while it runs, so two of them are never in flight together."""
import os
import socket

import numpy as np
import pytest

pytestmark = pytest.mark.gpu


def _worker(rank, world, port, q):
    import torch
    import torch.distributed as dist
    from paper_2607_03987_b200 import pakr, replicas, workloads as wl
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    torch.cuda.set_device(0)
    p, cfg = wl.config1()
    pl = pakr.Planner(p, 0)
    log = []

    def plan_fn(bound, rnd):
        out = None
        for turn in range(world):  # one process on the GPU at a time
            if turn == rank:
                seed = replicas.replica_seeds(rank, world, rnd + 1, first=100)[rnd]
                out = pl.plan(seed, cfg.B, cfg.K, cfg.tree_capacity, 2,
                              initial_cost_bound=0.0 if np.isinf(bound) else bound)
                torch.cuda.synchronize()
            dist.barrier()
        log.append(dict(bound=bound, cost=out["cost"], outcome=out["outcome"], replan_cost=out["replan_cost"].tolist(),
                        path_states=out["path_states"], path_controls=out["path_controls"]))
        return (out["cost"], out) if out["outcome"] else (float("inf"), None)

    shared = replicas.shared_bound_rounds(plan_fn, 2, dist=dist)
    dist.barrier()
    q.put((rank, log, shared["history"], shared["cost"], shared["owner"]))
    pl.close()
    dist.destroy_process_group()


def test_two_processes_share_the_cost_bound(orc):
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    import torch.multiprocessing as mp
    from paper_2607_03987_b200 import workloads as wl
    world = 2
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        port = s.getsockname()[1]
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for pr in procs:
        pr.start()
    res = sorted((q.get(timeout=300) for _ in range(world)), key=lambda t: t[0])
    for pr in procs:
        pr.join(timeout=60)
        assert pr.exitcode == 0
    p, _ = wl.config1()
    op = orc.OracleProblem(p)
    round0 = [log[0]["cost"] for _, log, *_ in res]
    assert all(np.isfinite(c) for c in round0)          # C1 is solved by every seed without a bound
    best0 = min(round0)
    owners = 0
    for rank, log, history, cost, owner in res:
        assert np.isinf(log[0]["bound"])                 # round 0: Alg. 1 l.1, c_best = inf
        assert log[1]["bound"] == best0 == history[0]    # round 1 runs under the GLOBAL best of round 0
        # under that bound a replica reports only strictly cheaper plans, and every replan's c_best stays <= it
        assert np.all(np.array(log[1]["replan_cost"]) <= np.float32(best0))
        if log[1]["outcome"]:
            assert log[1]["cost"] < best0
        for entry in log:                                # every plan any replica returned is valid for the oracle
            if entry["outcome"]:
                code, c, err = op.validate_plan(entry["path_states"], entry["path_controls"], per_edge=False)
                assert code == 0 and c == pytest.approx(entry["cost"], rel=1e-4)
        assert history[1] == cost == min(best0, *(l[1]["cost"] for _, l, *_ in res))
        owners += owner
    assert owners >= 1
