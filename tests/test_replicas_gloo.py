"""Multi-GPU host logic (replicas only) on CPU: two gloo ranks."""
import os
import socket

import pytest
import torch
import torch.distributed as dist
import torch.multiprocessing as mp

from paper_2607_03987_b200 import replicas


def test_replica_seeds_partition():
    for world in (1, 2, 8):
        all_seeds = sorted(s for r in range(world) for s in replicas.replica_seeds(r, world, 5, first=3))
        assert all_seeds == list(range(3, 3 + 5 * world))
    with pytest.raises(ValueError):
        replicas.replica_seeds(2, 2, 1)


def test_aggregate_single_process():
    out = replicas.aggregate(10.0, 20.0, 1000.0)
    assert out["value"] == pytest.approx(1e5) and out["e2e"] == pytest.approx(5e4)


def _worker(rank, world, port, q):
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    seeds = replicas.replica_seeds(rank, world, 3)
    # rank r "takes" (r+1)*10 ms on the device and (r+1)*12 ms wall for 100*(r+1) units
    out = replicas.aggregate(10.0 * (rank + 1), 12.0 * (rank + 1), 100.0 * (rank + 1), dist=dist)
    best = replicas.best_of_replicas([5.0 - rank, 9.0], dist=dist)
    # NEXT-4: the bound found by one replica prunes the others from the next round on
    table = {0: [9.0, 7.0, 7.5], 1: [8.0, 8.5, 6.0]}[rank]
    seen = []

    def plan_fn(bound, rnd):
        seen.append(bound)
        c = table[rnd]
        return (c, (rank, rnd)) if c < bound else (float("inf"), None)

    shared = replicas.shared_bound_rounds(plan_fn, 3, dist=dist)
    dist.barrier()
    q.put((rank, seeds, out, best, shared, seen))
    dist.destroy_process_group()


def test_two_rank_gloo_aggregation():
    world = 2
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    port = s.getsockname()[1]
    s.close()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    res = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    assert res[0][1] == [0, 2, 4] and res[1][1] == [1, 3, 5]
    for rank, _, _, _, shared, seen in res:
        assert seen == [float("inf"), 8.0, 7.0]          # bounds handed to the planner: global best so far
        assert shared["history"] == [8.0, 7.0, 6.0] and shared["cost"] == 6.0
        assert shared["owner"] == (rank == 1) and shared["payload"] == ((0, 1) if rank == 0 else (1, 2))
    for _, _, out, best, _, _ in res:  # identical on every rank: max time, summed units, min cost
        assert out["device_ms"] == 20.0 and out["wall_ms"] == 24.0 and out["units"] == 300.0
        assert out["value"] == pytest.approx(300.0 / 0.020)
        assert best == 4.0
