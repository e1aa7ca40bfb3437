"""End-to-end GPU tests of pakr_plan (Alg. 1 whole): every returned plan is re-propagated by the
oracle, the tree left in the workspace satisfies the invariants, c_best decreases strictly,
runs are deterministic, and the ABI reports errors instead of launching."""
import ctypes as C

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pakr():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_03987_b200 import pakr as mod
    mod.lib()
    return mod


def _check_plan(orc, p, res, edge_exact=True):
    op = orc.OracleProblem(p)
    assert res["outcome"] == 1 and res["path_len"] >= 2
    # per-edge form: every edge restarts from the stored node (tree invariant)
    code, cost, err = op.validate_plan(res["path_states"], res["path_controls"], per_edge=True)
    assert code == 0 and err < 1e-4
    assert cost == pytest.approx(res["cost"], rel=1e-4)
    # one continuous roll-out from the start: collision-free, ends in the goal, same cost
    code, cost, err = op.validate_plan(res["path_states"], res["path_controls"], per_edge=False)
    assert code == 0, code
    assert cost == pytest.approx(res["cost"], rel=1e-4)
    np.testing.assert_array_equal(res["path_states"][0], p.start)
    assert res["path_nodes"][0] == 0 and np.all(np.diff(res["path_nodes"]) > 0)
    # admissibility along the path: g + h <= g(goal)  (P15)
    edge = p.steps_per_edge * float(np.float32(p.dt))
    g = np.arange(res["path_len"]) * edge
    h = np.array([op.heuristic(x) for x in res["path_states"].astype(np.float64)])
    assert np.all(g + h <= res["cost"] + 1e-3)
    return op


def _check_tree(orc, op, p, tree, cap, n_samples=300):
    n = len(tree["parents"])
    par, cost = tree["parents"], tree["costs"]
    assert n <= cap and par[0] == -1
    assert np.all(par[1:] >= 0) and np.all(par[1:] < np.arange(1, n))  # every parent precedes its child
    edge = np.float32(p.steps_per_edge) * np.float32(p.dt)
    np.testing.assert_allclose(cost[1:], cost[par[1:]] + edge, rtol=1e-6)  # costs grow along every path
    rng = np.random.default_rng(0)
    for i in rng.integers(1, n, min(n_samples, n - 1)):
        x = tree["states"][i].astype(np.float64)
        assert op.bounds_margin(x) >= -1e-5 and op.obstacle_margin(x) > -1e-5
        xr, fl, fb, mm, ec = op.propagate(tree["states"][par[i]].astype(np.float64), tree["actions"][i].astype(np.float64))
        assert (fl & 1) or mm < 1e-5
        d = np.abs(xr - x)
        ang = p.dim_kind == 1
        d[ang] = np.minimum(d[ang], 2 * np.pi - d[ang])
        assert d.max() < 1e-4


@pytest.mark.parametrize("name", ["C1", "C2", "C3", "C4", "N1", "N2", "N3", "N4"])
def test_plan_configs(pakr, orc, name):
    p, cfg = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    res = pl.plan(cfg.seed, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    assert res["replans_run"] == cfg.n_replans and res["termination"] == 0
    op = _check_plan(orc, p, res)
    # c_best strictly decreasing over successful replans, constant over failed ones
    rc = res["replan_cost"]
    assert np.all(np.diff(rc) <= 0)
    assert int((np.r_[np.inf, rc[:-1]] > rc).sum()) == res["replans_solved"]
    assert res["cost"] == pytest.approx(float(rc[-1]))
    assert res["children"] == res["iterations"] * cfg.B * cfg.K
    assert res["iterations"] == int(res["replan_iters"].sum())
    tree = pl.read_tree(cfg.B, cfg.K, cfg.tree_capacity, res["final_tree_nodes"])
    assert res["final_tree_nodes"] == res["replan_nodes"][-1]
    _check_tree(orc, op, p, tree, cfg.tree_capacity)
    # deterministic (time_budget <= 0): same seed, same everything
    res2 = pl.plan(cfg.seed, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    np.testing.assert_array_equal(res["path_states"], res2["path_states"])
    np.testing.assert_array_equal(res["replan_nodes"], res2["replan_nodes"])
    res3 = pl.plan(cfg.seed + 1, cfg.B, cfg.K, cfg.tree_capacity, 1)
    assert res3["replan_nodes"][0] != res["replan_nodes"][0]
    pl.close()


def test_plan_c1_lockstep_with_oracle(pakr, orc):
    """C1, replan 0: the GPU loop and the oracle loop walk the same iterations (same randoms, fp32 vs
    fp64).  A near-tie flip may legitimately break exact lock-step (H5), so the hard assertions are
    the statistics; exact equality is asserted only if the trees have the same size."""
    p, cfg = wl.config1()
    pl = pakr.Planner(p)
    res = pl.plan(0, cfg.B, cfg.K, cfg.tree_capacity, 1)
    op = orc.OracleProblem(p)
    ref = orc.plan(op, 0, cfg.B, cfg.K, cfg.tree_capacity, 1)
    assert res["outcome"] == ref["outcome"] == 1
    assert abs(res["replan_iters"][0] - ref["replan_iters"][0]) <= 2
    assert abs(res["replan_nodes"][0] - ref["replan_nodes"][0]) <= 0.02 * ref["replan_nodes"][0]
    if res["replan_nodes"][0] == ref["replan_nodes"][0]:
        assert res["cost"] == pytest.approx(ref["cost"], rel=1e-6)
        np.testing.assert_array_equal(res["path_nodes"], ref["path_nodes"])
        np.testing.assert_allclose(res["path_states"], ref["path_states"], atol=1e-4)
    pl.close()


def test_plan_seeds_c5_point_and_first_solution_time(pakr, orc):
    p, cfg = wl.config5(B=1024, K=16, tree_capacity=1 << 21)
    pl = pakr.Planner(p)
    for seed in range(3):
        res = pl.plan(seed, cfg.B, cfg.K, cfg.tree_capacity, 1)
        _check_plan(orc, p, res)
        assert 0 < res["first_solution_ms"] <= res["device_ms"]
    pl.close()


@pytest.mark.parametrize("B,K", [(16384, 16), (4096, 64)])
def test_plan_c5_large_batches(pakr, orc, B, K):
    """Config 5's corner points: B*K = 262,144 children per iteration (insert's large-batch path, K = 64,
    multi-hundred-thousand-node trees); the plan is re-propagated by the oracle and the tree checked."""
    p, cfg = wl.config5(B=B, K=K)
    pl = pakr.Planner(p)
    res = pl.plan(1, B, K, cfg.tree_capacity, 1)
    op = _check_plan(orc, p, res)
    assert res["children"] == res["iterations"] * B * K and res["final_tree_nodes"] > 100000
    tree = pl.read_tree(B, K, cfg.tree_capacity, res["final_tree_nodes"])
    _check_tree(orc, op, p, tree, cfg.tree_capacity, n_samples=200)
    res2 = pl.plan(1, B, K, cfg.tree_capacity, 1)
    np.testing.assert_array_equal(res["path_states"], res2["path_states"])
    pl.close()


def test_plan_time_budget_and_no_solution(pakr, orc):
    p, cfg = wl.config2()
    pl = pakr.Planner(p)
    res = pl.plan(0, cfg.B, cfg.K, cfg.tree_capacity, 4096, time_budget_ms=30.0)
    assert res["termination"] == 1 and res["replans_run"] < 4096
    assert 30.0 <= res["device_ms"] < 60.0
    _check_plan(orc, p, res)
    # two iterations cannot reach the goal: "no solution" is an outcome, not an error
    res = pl.plan(0, 64, 2, 4096, 2, max_iters_per_replan=2)
    assert res["outcome"] == 0 and res["path_len"] == 0 and np.isinf(res["cost"])
    assert res["iterations"] == 4 and res["replans_solved"] == 0
    # tiny capacity: the tree fills and the replan ends as "full"
    res = pl.plan(0, 256, 8, 1000, 1)
    assert res["outcome"] == 0 and res["final_tree_nodes"] == 1000
    pl.close()


def test_abi_errors(pakr):
    import torch
    p, cfg = wl.config1()
    pl = pakr.Planner(p)
    L = pakr.lib()
    assert pl.workspace_bytes(0, 4, 1000) == 0 and pl.workspace_bytes(16, 0, 1000) == 0
    assert pl.workspace_bytes(16, 4, 1) == 0
    ws = pl.workspace(64, 4, 4096)
    small = torch.empty(1024, dtype=torch.uint8, device="cuda")
    with pytest.raises(pakr.PakrError) as e:
        pl.plan(0, 64, 4, 4096, 1, workspace=small)
    assert e.value.status == 3
    with pytest.raises(pakr.PakrError) as e:
        pl.plan(0, 64, 4, 4096, 0)
    assert e.value.status == 1
    with pytest.raises(pakr.PakrError) as e:  # path buffer too small -> BUFFER_TOO_SMALL, length reported
        pl.plan(0, cfg.B, cfg.K, cfg.tree_capacity, 1, path_capacity=3)
    assert e.value.status == 4
    # invalid problems never reach the device
    import dataclasses
    for bad in (dataclasses.replace(p, state_dim=5), dataclasses.replace(p, dt=0.0),
                dataclasses.replace(p, state_lo=p.state_hi + 1), dataclasses.replace(p, dynamics_id=9),
                dataclasses.replace(p, goal_dims=np.array([0, 4], np.int32)),      # goal dim out of range
                dataclasses.replace(p, goal_dims=np.array([1, 1], np.int32))):     # repeated goal dim
        with pytest.raises(pakr.PakrError) as e:
            pakr.Planner(bad)
        assert e.value.status in (1, 2)
    pl.close()
    # the Acrobot takes no obstacles (its position dims are angles) and needs its eight parameters
    a, _ = wl.CONFIGS["N4"]()
    with pytest.raises(pakr.PakrError) as e:
        pakr.Planner(dataclasses.replace(a, obstacles=np.array([[0.0, 0.0, 0.5]], np.float32)))
    assert e.value.status == 2
    with pytest.raises(pakr.PakrError) as e:
        pakr.Planner(dataclasses.replace(a, dyn_params=a.dyn_params[:5]))
    assert e.value.status == 1
    with pytest.raises(pakr.PakrError) as e:
        pakr.Planner(dataclasses.replace(a, dim_kind=np.array([1, 0, 0, 0], np.uint8)))
    assert e.value.status == 2


@pytest.mark.parametrize("name,iters", [("C1", 12), ("C2", 9), ("C3", 6), ("N1", 7), ("N2", 8), ("N4", 8)])
def test_plan_loop_equals_chain_of_single_steps(pakr, name, iters):
    """The device-resident loop (NN look-ahead scan, fused tail scan, two key buffers) must build exactly
    the tree that `iters` separate pakr_expand_step calls build (no look-ahead there): bit-exact."""
    p, cfg = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    cap = 1 + iters * cfg.B * cfg.K
    res = pl.plan(7, cfg.B, cfg.K, cap, 1, max_iters_per_replan=iters)
    n_loop = res["final_tree_nodes"]
    loop_tree = pl.read_tree(cfg.B, cfg.K, cap, n_loop)
    tree = pl.new_tree(cap)
    c_best = float("inf")
    done = 0
    for it in range(iters):
        out = pl.expand_step(tree, 7, 0, it, cfg.B, cfg.K, c_best=c_best)
        done += 1
        if out["goal_node"] >= 0:
            break
    assert done == res["iterations"]
    n_chain = int(tree["n_nodes"][0].item())
    assert n_chain == n_loop and n_loop > cfg.B
    D, m = p.state_dim, p.control_dim
    np.testing.assert_array_equal(tree["states"][:n_chain, :D].cpu().numpy(), loop_tree["states"])
    np.testing.assert_array_equal(tree["actions"][:n_chain, :m].cpu().numpy(), loop_tree["actions"])
    np.testing.assert_array_equal(tree["parents"][:n_chain].cpu().numpy(), loop_tree["parents"])
    np.testing.assert_array_equal(tree["costs"][:n_chain].cpu().numpy(), loop_tree["costs"])
    pl.close()


@pytest.mark.parametrize("name,seeds", [("C1", 12), ("C2", 8), ("N2", 6), ("N4", 6)])
def test_plan_many_seeds_validated(pakr, orc, name, seeds):
    """Every returned plan of a spread of planner seeds is re-propagated by the oracle (north_star end-to-end bar)."""
    p, cfg = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    costs = []
    for seed in range(100, 100 + seeds):
        res = pl.plan(seed, cfg.B, cfg.K, cfg.tree_capacity, 3)
        _check_plan(orc, p, res)
        costs.append(res["cost"])
    assert len(set(costs)) >= 1
    pl.close()


def test_plan_initial_cost_bound(pakr, orc):
    """pakr_plan under a bound handed in from outside (NEXT-4): prunes from the first replan; reports only
    what this call found; the oracle's loop with the same bound agrees on C1."""
    p, cfg = wl.config1()
    pl = pakr.Planner(p)
    free = pl.plan(3, cfg.B, cfg.K, cfg.tree_capacity, 1)
    assert free["outcome"] == 1
    c0 = free["cost"]
    res = pl.plan(4, cfg.B, cfg.K, cfg.tree_capacity, 4, initial_cost_bound=c0)
    if res["outcome"]:
        assert res["cost"] < c0
        _check_plan(orc, p, res)
    else:
        assert res["path_len"] == 0 and np.isinf(res["cost"])
    assert np.all(res["replan_cost"] <= np.float32(c0))
    # a bound nothing can beat: every child is pruned, no solution, and that is not an error
    res = pl.plan(4, cfg.B, cfg.K, cfg.tree_capacity, 2, initial_cost_bound=1e-3, max_iters_per_replan=5)
    assert res["outcome"] == 0 and res["inserted"] == 0
    op = orc.OracleProblem(p)
    ref = orc.plan(op, 4, cfg.B, cfg.K, cfg.tree_capacity, 1, initial_cost_bound=c0)
    one = pl.plan(4, cfg.B, cfg.K, cfg.tree_capacity, 1, initial_cost_bound=c0)
    assert one["outcome"] == ref["outcome"]
    assert abs(int(one["replan_iters"][0]) - int(ref["replan_iters"][0])) <= 2
    pl.close()


@pytest.mark.parametrize("name,iters", [("C2", 9), ("C3", 6), ("C1", 12), ("C4", 5), ("N1", 8), ("C5", 4)])
def test_plan_loop_with_nn_index_equals_scan(pakr, name, iters):
    """Inside the device loop the index is rebuilt as the tree grows and the rows added since are scanned:
    the tree must be bit-identical to the one the scan tiers build (C5: the B = 4096, K = 64 sweep point)."""
    p, cfg = wl.config5(B=4096, K=64) if name == "C5" else wl.CONFIGS[name]()
    cap = 1 + iters * cfg.B * cfg.K
    trees = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_INDEX):
        res = pl.plan(7, cfg.B, cfg.K, cap, 1, max_iters_per_replan=iters, nn_mode=mode)
        trees[mode] = (res["final_tree_nodes"], pl.read_tree(cfg.B, cfg.K, cap, res["final_tree_nodes"]))
    pl.close()
    assert trees[pakr.NN_SCAN][0] == trees[pakr.NN_INDEX][0] > cfg.B
    for k in ("states", "actions", "parents", "costs"):
        np.testing.assert_array_equal(trees[pakr.NN_SCAN][1][k], trees[pakr.NN_INDEX][1][k])


@pytest.mark.parametrize("name,iters", [("C4", 8), ("C5", 5)])
def test_plan_loop_auto_policy_equals_scan(pakr, name, iters):
    """PAKR_NN_AUTO is what bench.py times.  At B = 4096 it searches the index over the rows sorted at the last rebuild
    and scans the rows added since with the tiled tier, rebuilding only when that remainder has grown enough.  On C4
    (B = 4096, K = 16) the first batch takes the tree past the engagement size (48.8 k rows), and iterations 3-5 add
    only 0.5-3 k rows each: they run index + remainder without a rebuild.  C5 (4096, 64) rebuilds every iteration.
    A wrong (non-nearest) parent would still give a valid plan, so the whole tree must equal the scan's bit for bit --
    and the index must really have answered (fewer distance evaluations than pairs)."""
    p, cfg = wl.config5(B=4096, K=64) if name == "C5" else wl.CONFIGS[name]()
    cap = 1 + iters * cfg.B * cfg.K
    got = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_AUTO):
        res = pl.plan(7, cfg.B, cfg.K, cap, 1, max_iters_per_replan=iters, nn_mode=mode)
        got[mode] = (res, pl.read_tree(cfg.B, cfg.K, cap, res["final_tree_nodes"]))
    pl.close()
    scan, auto = got[pakr.NN_SCAN][0], got[pakr.NN_AUTO][0]
    assert scan["final_tree_nodes"] == auto["final_tree_nodes"] > 60000
    assert scan["iterations"] == auto["iterations"] == iters
    for k in ("states", "actions", "parents", "costs"):
        np.testing.assert_array_equal(got[pakr.NN_SCAN][1][k], got[pakr.NN_AUTO][1][k])
    assert scan["nn_pairs"] == auto["nn_pairs"] == scan["nn_pairs_evaluated"]
    assert auto["nn_pairs_evaluated"] < 0.5 * auto["nn_pairs"], "the index did not engage"
    assert auto["phase_ms"][3] > 0.0   # at least one rebuild ran inside the loop


@pytest.mark.parametrize("seed", [0, 1])
def test_plan_c1_lockstep_with_oracle_over_all_replans(pakr, orc, seed):
    """Alg. 1 l.1-4 at the loop level: all 10 replans of BASELINE config 1 against orc.plan --
    fresh tree and re-keyed draws per replan, c_best carried over.  fp32 vs fp64 may flip a near-tie, so node counts get
    2 % and iteration counts +-2; costs are multiples of the edge duration and must be equal."""
    p, cfg = wl.config1()
    pl = pakr.Planner(p)
    res = pl.plan(seed, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    op = orc.OracleProblem(p)
    ref = orc.plan(op, seed, cfg.B, cfg.K, cfg.tree_capacity, cfg.n_replans)
    pl.close()
    assert res["replans_run"] == ref["replans_run"] == 10
    assert res["replans_solved"] == ref["replans_solved"] >= 2
    for r in range(10):
        assert abs(int(res["replan_iters"][r]) - int(ref["replan_iters"][r])) <= 2, r
        assert abs(int(res["replan_nodes"][r]) - int(ref["replan_nodes"][r])) <= 0.02 * ref["replan_nodes"][r], r
        assert res["replan_cost"][r] == pytest.approx(ref["replan_cost"][r], rel=1e-6), r
        assert res["replan_nodes"][r] <= 1 + int(res["replan_iters"][r]) * cfg.B * cfg.K, r   # grown from the root alone
    assert res["cost"] == pytest.approx(ref["cost"], rel=1e-6)


def test_plan_small_b_stream_tier_and_no_obstacles(pakr, orc):
    """B <= 16 runs the streaming-tier kernel through the whole device loop (look-ahead, in-phase insert, tail
    rounds): same tree as the chain of single steps; and a problem without obstacles plans fine."""
    import dataclasses
    p, _ = wl.config2()
    pl = pakr.Planner(p)
    B, K, iters = 8, 16, 10
    cap = 1 + iters * B * K
    res = pl.plan(5, B, K, cap, 1, max_iters_per_replan=iters)
    loop_tree = pl.read_tree(B, K, cap, res["final_tree_nodes"])
    tree = pl.new_tree(cap)
    for it in range(res["iterations"]):
        pl.expand_step(tree, 5, 0, it, B, K)
    n = int(tree["n_nodes"][0].item())
    assert n == res["final_tree_nodes"] > 200
    np.testing.assert_array_equal(tree["states"][:n, :p.state_dim].cpu().numpy(), loop_tree["states"])
    np.testing.assert_array_equal(tree["parents"][:n].cpu().numpy(), loop_tree["parents"])
    pl.close()
    p0 = dataclasses.replace(p, obstacles=p.obstacles[:0])
    pl = pakr.Planner(p0)
    res = pl.plan(0, 512, 8, 1 << 18, 2)
    _check_plan(orc, p0, res)
    pl.close()


@pytest.mark.parametrize("name,B,K,iters", [("C4", 4096, 16, 6), ("C5", 4096, 64, 4), ("N3", 2048, 16, 8), ("C2", 16384, 8, 4)])
def test_plan_loop_with_nn_filter_equals_scan(pakr, name, B, K, iters):
    """Inside the device loop the filter rows are written at insert time and the filter answers the look-ahead NN and
    the scans of freshly appended rows: the tree must be bit-identical to the one the fp32 scan builds."""
    p, cfg = wl.config5(B=B, K=K) if name == "C5" else wl.CONFIGS[name]()
    cap = 1 + iters * B * K
    trees = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_FILTER):
        res = pl.plan(7, B, K, cap, 1, max_iters_per_replan=iters, nn_mode=mode)
        trees[mode] = (res["final_tree_nodes"], pl.read_tree(B, K, cap, res["final_tree_nodes"]), res["nn_pairs_filtered"])
    pl.close()
    assert trees[pakr.NN_SCAN][0] == trees[pakr.NN_FILTER][0] > B
    assert trees[pakr.NN_SCAN][2] == 0 and trees[pakr.NN_FILTER][2] > 0
    for k in ("states", "actions", "parents", "costs"):
        np.testing.assert_array_equal(trees[pakr.NN_SCAN][1][k], trees[pakr.NN_FILTER][1][k])


def test_workspace_sized_for_the_nn_mode(pakr):
    """pakr_workspace_bytes_for: a caller that knows its nn_mode does not pay for the other tiers' buffers (C4 under
    AUTO: no 96 B/node filter rows).  A workspace of exactly that size runs that mode with the same result as the
    all-tiers workspace; one byte less is refused before anything is launched."""
    import torch
    p, cfg = wl.config4()
    B, K, cap, iters = cfg.B, cfg.K, 1 + 6 * cfg.B * cfg.K, 6
    pl = pakr.Planner(p)
    full = pl.workspace_bytes(B, K, cap)
    need = {m: pl.workspace_bytes_for(B, K, cap, m) for m in (pakr.NN_AUTO, pakr.NN_SCAN, pakr.NN_INDEX, pakr.NN_FILTER)}
    assert all(0 < v <= full for v in need.values())
    assert need[pakr.NN_SCAN] < need[pakr.NN_AUTO] == need[pakr.NN_INDEX] < full
    assert need[pakr.NN_SCAN] < need[pakr.NN_FILTER] < full
    assert full - need[pakr.NN_AUTO] >= 96 * cap          # the filter rows are not charged to AUTO
    assert pl.workspace_bytes_for(B, K, cap, 9) == 0
    ref = pl.plan(2, B, K, cap, 1, max_iters_per_replan=iters, nn_mode=pakr.NN_SCAN)
    ref_tree = pl.read_tree(B, K, cap, ref["final_tree_nodes"])
    for mode, nbytes in need.items():
        ws = torch.empty(nbytes, dtype=torch.uint8, device="cuda")
        res = pl.plan(2, B, K, cap, 1, max_iters_per_replan=iters, nn_mode=mode, workspace=ws)
        assert res["final_tree_nodes"] == ref["final_tree_nodes"]
        tree = pl.read_tree(B, K, cap, res["final_tree_nodes"], workspace=ws)
        np.testing.assert_array_equal(tree["states"], ref_tree["states"])
        np.testing.assert_array_equal(tree["parents"], ref_tree["parents"])
        assert pl.read_stats(B, K, cap, workspace=ws)["iterations"] == iters
        with pytest.raises(pakr.PakrError) as e:
            pl.plan(2, B, K, cap, 1, max_iters_per_replan=iters, nn_mode=mode, workspace=ws[:nbytes - 1])
        assert e.value.status == 3
    # B <= 16 runs the streaming tier in every mode: packed rows, no index or filter buffers
    small = {m: pl.workspace_bytes_for(8, 4, 100000, m) for m in need}
    assert len(set(small.values())) == 1 and small[pakr.NN_AUTO] == pl.workspace_bytes(8, 4, 100000)
    pl.close()
