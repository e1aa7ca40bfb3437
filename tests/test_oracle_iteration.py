"""Pins of the oracle's NN, collision, bounds, prune/goal, insert order and AO-x loop
(SURVEY.md 8(c) pin table): hand cases, analytic geometry, brute force and invariants."""
import dataclasses
import math

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl


def _free(p, **kw):
    lo = np.where(np.isfinite(p.state_lo), -1e6, p.state_lo).astype(np.float32)
    hi = np.where(np.isfinite(p.state_hi), 1e6, p.state_hi).astype(np.float32)
    return dataclasses.replace(p, obstacles=p.obstacles[:0], state_lo=lo, state_hi=hi, **kw)


# ------------------------------------------------------------------ nearest neighbour (P5, P6)
def test_nn_hand_cases(orc):
    p, _ = wl.config3()  # has an angle dim
    op = orc.OracleProblem(p)
    q = np.array([5.0, 5.0, 0.1, 0.2, -0.3])
    assert op.nearest(q[None, :] + 3.0, q) == (0, pytest.approx(op.dist2(q + 3.0, q)))  # n = 1 -> 0
    nodes = np.array([[0, 0, 0, 0, 0], [5, 5, 0.1, 0.2, -0.3], [5, 5, 0.1, 0.2, -0.3], [9, 9, 0, 0, 0]], float)
    i, d2 = op.nearest(nodes, q)  # query equals a node; duplicates -> lowest index
    assert (i, d2) == (1, 0.0)
    # plain Euclidean value
    assert op.dist2([1, 2, 0, 0, 0], [4, 6, 0, 0, 0]) == pytest.approx(25.0)
    # angle wrap: pi - eps and -pi + eps are 2 eps apart
    eps = 1e-3
    assert op.dist2([0, 0, math.pi - eps, 0, 0], [0, 0, -math.pi + eps, 0, 0]) == pytest.approx(4 * eps * eps, rel=1e-9)
    # weights: zero-weight dims are ignored, others scale linearly
    pw = dataclasses.replace(p, nn_weight=np.array([2, 0, 0.5, 0, 3], np.float32))
    ow = orc.OracleProblem(pw)
    assert ow.dist2([1, 100, 0.2, -50, 1], [0, 0, 0, 0, 0]) == pytest.approx(2 * 1 + 0.5 * 0.04 + 3 * 1)


def test_nn_matches_numpy_bruteforce(orc):
    rng = np.random.default_rng(1)
    for cfg in (wl.config2, wl.config3, wl.config4):
        p, _ = cfg()
        op = orc.OracleProblem(p)
        tree = wl.random_tree(p, 777, seed=3)["states"].astype(np.float64)
        w = p.nn_weight.astype(np.float64)
        ang = p.dim_kind == wl.DIM_ANGLE
        for s in range(20):
            q = op.sample_state(9, 0, 0, s)
            d = q[None, :] - tree
            d[:, ang] = (d[:, ang] + math.pi) % (2 * math.pi) - math.pi
            d2 = (w * d * d).sum(1)
            i, v = op.nearest(tree, q)
            assert i == int(np.argmin(d2))
            assert v == pytest.approx(d2.min(), rel=1e-12)


# ------------------------------------------------------------------ collision / bounds (P10-P12)
def test_circle_collision_analytic(orc):
    p, _ = wl.config1()
    p = dataclasses.replace(p, obstacles=np.array([[5, 5, 1.0], [2, 8, 0.5]], np.float32))
    op = orc.OracleProblem(p)
    for ang in np.linspace(0, 2 * math.pi, 7):
        c, s = math.cos(ang), math.sin(ang)
        assert op.obstacle_margin([5 + 1.001 * c, 5 + 1.001 * s, 0, 0]) > 0
        assert op.obstacle_margin([5 + 0.999 * c, 5 + 0.999 * s, 0, 0]) < 0
    assert op.obstacle_margin([6.0, 5.0, 0, 0]) == 0.0  # closed set: the rim collides (margin <= 0)
    assert op.obstacle_margin([5, 7.5, 9, 9]) == pytest.approx(1.5)  # velocities do not matter
    assert op.obstacle_margin([2, 8, 0, 0]) == pytest.approx(-0.5)


def test_aabb_collision_analytic(orc):
    p, _ = wl.config2()
    p = dataclasses.replace(p, obstacles=np.array([[1, 2, 3, 2, 4, 6]], np.float32))
    op = orc.OracleProblem(p)
    inside = lambda x: op.obstacle_margin(list(x) + [0, 0, 0]) <= 0
    assert inside([1.5, 3, 4.5])  # interior
    assert inside([1, 3, 4.5]) and inside([2, 4, 6]) and inside([1, 2, 3])  # face, corner: closed
    assert not inside([0.999, 3, 4.5]) and not inside([1.5, 4.001, 4.5]) and not inside([1.5, 3, 6.001])
    assert not inside([2.001, 4.001, 6.001])  # beyond a corner
    assert op.obstacle_margin([1.5, 3, 7.0, 0, 0, 0]) == pytest.approx(1.0)
    assert op.obstacle_margin([1.5, 3, 4.5, 0, 0, 0]) == pytest.approx(-0.5)  # nearest face is x at 0.5


def test_trajectory_hits_obstacle_at_closed_form_step(orc):
    """DI moving at constant velocity toward a circle: first colliding step from the closed form."""
    p, _ = wl.config1()
    q = dataclasses.replace(_free(p), obstacles=np.array([[3.0, 0.0, 1.0]], np.float32),
                            steps_per_edge=60)
    op = orc.OracleProblem(q)
    dt = float(np.float32(p.dt))
    v = 0.9
    # Euler with a = 0: p_j = v j dt; collides when p_j >= 2.0 (rim, closed)
    j_hit = math.ceil(2.0 / (v * dt) - 1e-12)
    x, flags, fb, mm, _ = op.propagate([0, 0, v, 0], [0, 0])
    assert fb == j_hit and not (flags & orc.F_VALID) and not (flags & orc.F_COLLFREE)
    assert flags & orc.F_INBOUNDS
    # a shorter edge stops before the obstacle and stays valid
    q2 = dataclasses.replace(q, steps_per_edge=j_hit - 1)
    x, flags, fb, mm, _ = orc.OracleProblem(q2).propagate([0, 0, v, 0], [0, 0])
    assert fb == 0 and flags & orc.F_VALID
    assert mm == pytest.approx(2.0 - v * (j_hit - 1) * dt)


def test_bounds_violation_closed_form_step(orc):
    """P12: DI with v0 = 0.9, a = +1 leaves |v| <= 1 at the closed-form step; child is rejected."""
    p, _ = wl.config1()
    q = dataclasses.replace(p, obstacles=p.obstacles[:0])
    op = orc.OracleProblem(q)
    dt = float(np.float32(p.dt))
    j_bad = math.floor(0.1 / dt + 1e-9) + 1  # first j with 0.9 + j dt > 1
    x, flags, fb, _, _ = op.propagate([5, 5, 0.9, 0], [1.0, 0])
    assert fb == j_bad and not (flags & orc.F_INBOUNDS) and not (flags & orc.F_VALID)
    assert flags & orc.F_COLLFREE
    assert op.bounds_margin([5, 5, 1.0, 0]) == 0.0  # closed interval: on the bound is inside
    assert op.bounds_margin([5, 5, 1.0 + 1e-9, 0]) < 0
    # P13: angle dims are never bounds-tested
    p3, _ = wl.config3()
    assert orc.OracleProblem(p3).bounds_margin([5, 5, 17.0, 0, 0]) > 0


# ------------------------------------------------------------------ heuristic / goal / prune
def test_heuristic_and_goal(orc):
    p, _ = wl.config1()
    op = orc.OracleProblem(p)
    assert op.heuristic([9.5, 9.5, 1, 1]) == 0.0
    assert op.heuristic([9.5, 9.9, 0, 0]) == 0.0  # inside the ball
    assert op.heuristic([9.5, 6.5, 0, 0]) == pytest.approx((3.0 - 0.5) / float(np.float32(math.sqrt(2))))
    assert op.in_goal([9.5, 9.0, 0.3, -1])[0]  # rim, closed; velocities free
    assert not op.in_goal([9.5, 8.999, 0, 0])[0]
    q = dataclasses.replace(p, heuristic_speed=float("inf"))
    assert orc.OracleProblem(q).heuristic([0, 0, 0, 0]) == 0.0
    p3, _ = wl.config3()
    o3 = orc.OracleProblem(p3)
    assert o3.in_goal([19, 19, 0.49, 0, 0])[0] and not o3.in_goal([19, 19, 0.51, 0, 0])[0]
    assert o3.in_goal([19, 19, -0.49, 0, 0])[0] and not o3.in_goal([19, 19, math.pi, 0, 0])[0]


def _one_iteration(orc, p, B, K, c_best, n_tree=200, cap=None, seed=5):
    op = orc.OracleProblem(p)
    t = wl.random_tree(p, n_tree, seed=11)
    tree = orc.OracleTree(op, cap or (n_tree + B * K))
    tree.load(t["states"], t["actions"], t["parents"], t["costs"])
    out = orc.expand_iteration(op, tree, seed, 0, 0, B, K, c_best)
    return op, t, tree, out


def test_prune_extremes_and_flags(orc):
    p, _ = wl.config2()
    op, t, tree, out = _one_iteration(orc, p, 64, 4, float("inf"))
    f = out["child_flags"]
    assert np.all(f & orc.F_NOTPRUNED)  # c_best = inf: nothing pruned (P16)
    assert out["n_inserted"] == int(((f & orc.F_VALID) != 0).sum()) > 0
    op, t, tree, out0 = _one_iteration(orc, p, 64, 4, 0.0)
    assert not np.any(out0["child_flags"] & orc.F_NOTPRUNED) and out0["n_inserted"] == 0
    # an intermediate bound prunes exactly the children with c_new + h >= c_best
    cb = float(np.median(out["child_cost"]) + 8.0)
    op, t, tree, out1 = _one_iteration(orc, p, 64, 4, cb)
    h = np.array([op.heuristic(x) for x in out1["child_state"]])
    np.testing.assert_array_equal((out1["child_flags"] & orc.F_NOTPRUNED) != 0, out1["child_cost"] + h < cb)
    assert 0 < ((out1["child_flags"] & orc.F_NOTPRUNED) != 0).sum() < 256


def test_iteration_is_copy_if_and_frozen_snapshot(orc):
    """Insert order = std::copy_if over child index (P20); NN sees only the snapshot."""
    p, _ = wl.config3()
    B, K, n0 = 96, 5, 300
    op, t, tree, out = _one_iteration(orc, p, B, K, float("inf"), n_tree=n0)
    f = out["child_flags"]
    keep = np.nonzero((f & orc.F_VALID) != 0)[0]
    assert tree.n == n0 + len(keep) == n0 + out["n_inserted"]
    np.testing.assert_array_equal(tree.states[n0:tree.n], out["child_state"][keep])
    np.testing.assert_array_equal(tree.actions[n0:tree.n], out["child_ctrl"][keep])
    np.testing.assert_array_equal(tree.costs[n0:tree.n], out["child_cost"][keep])
    np.testing.assert_array_equal(tree.parents[n0:tree.n], out["nn_idx"][keep // K])
    assert out["nn_idx"].max() < n0  # frozen snapshot
    # every child's parent/cost/control bookkeeping
    edge = p.steps_per_edge * float(np.float32(p.dt))
    np.testing.assert_allclose(out["child_cost"], t["costs"][out["nn_idx"]][np.arange(B * K) // K] + edge, atol=1e-12)
    for c in (0, 7, B * K - 1):
        s, k = divmod(c, K)
        np.testing.assert_array_equal(out["child_ctrl"][c], op.sample_control(5, 0, 0, s, k))
        np.testing.assert_array_equal(out["x_rand"][s], op.sample_state(5, 0, 0, s))
        x, fl, *_ = op.propagate(t["states"][out["nn_idx"][s]].astype(np.float64), out["child_ctrl"][c])
        np.testing.assert_array_equal(out["child_state"][c], x)
    # capacity overflow: only the first cap - n survivors are inserted
    room = 17
    op, t, tree2, out2 = _one_iteration(orc, p, B, K, float("inf"), n_tree=n0, cap=n0 + room)
    assert tree2.n == n0 + room and out2["n_inserted"] == room
    np.testing.assert_array_equal(tree2.states[n0:], out["child_state"][keep[:room]])
    ins = np.nonzero((out2["child_flags"] & orc.F_INSERTED) != 0)[0]
    np.testing.assert_array_equal(ins, keep[:room])


def test_branching_only_adds_candidates(orc):
    """the K>1 planner evaluates every child of the K=1 planner... with this keying
    the (s, k=0) children of K=4 are exactly the K=1 children."""
    p, _ = wl.config2()
    _, _, _, o1 = _one_iteration(orc, p, 32, 1, float("inf"))
    _, _, _, o4 = _one_iteration(orc, p, 32, 4, float("inf"))
    np.testing.assert_array_equal(o1["nn_idx"], o4["nn_idx"])
    np.testing.assert_array_equal(o1["child_state"], o4["child_state"][::4])
    np.testing.assert_array_equal(o1["child_flags"] & 31, o4["child_flags"][::4] & 31)


def test_goal_winner(orc):
    """Goal children are inserted; winner = min c_new, ties -> lowest child index (P18, P19)."""
    p, _ = wl.config1()
    q = dataclasses.replace(p, obstacles=p.obstacles[:0], goal_radius=3.0)
    op = orc.OracleProblem(q)
    tree = orc.OracleTree(op, 4096)
    n0 = 50
    rng = np.random.default_rng(0)
    st = np.zeros((n0, 4))
    st[:, :2] = rng.uniform(7.5, 9.5, size=(n0, 2))  # every node already near the goal
    st[0] = q.start
    costs = rng.integers(1, 4, n0) * 0.5
    costs[0] = 0
    tree.load(st, np.zeros((n0, 2)), np.r_[-1, np.zeros(n0 - 1)].astype(np.int32), costs)
    out = orc.expand_iteration(op, tree, 3, 0, 0, 64, 4, float("inf"))
    g = np.nonzero((out["child_flags"] & orc.F_GOAL) != 0)[0]
    assert len(g) > 5 and out["goal"]
    best = g[np.argmin(out["child_cost"][g])]  # argmin returns the first minimum
    ins = np.nonzero((out["child_flags"] & orc.F_INSERTED) != 0)[0]
    assert out["goal_node"] == n0 + int(np.nonzero(ins == best)[0][0])
    assert out["new_c_best"] == out["child_cost"][best]
    assert np.all((out["child_flags"][g] & orc.F_INSERTED) != 0)


# ------------------------------------------------------------------ AO-x loop (Alg. 1 l.1-18)
@pytest.fixture(scope="module")
def c1_plan(orc):
    p, cfg = wl.config1()
    op = orc.OracleProblem(p)
    res = orc.plan(op, 0, cfg.B, cfg.K, cfg.tree_capacity, 4, max_iters_per_replan=40)
    return p, cfg, op, res


def test_plan_c1_solves_and_validates(orc, c1_plan):
    p, cfg, op, res = c1_plan
    assert res["outcome"] == 1 and res["replans_solved"] >= 1
    code, cost, err = op.validate_plan(res["path_states"], res["path_controls"])
    assert code == 0 and err < 1e-9
    assert cost == pytest.approx(res["cost"], rel=1e-12)
    code, cost, err = op.validate_plan(res["path_states"], res["path_controls"], per_edge=True)
    assert code == 0 and err < 1e-12
    edge = p.steps_per_edge * float(np.float32(p.dt))
    assert res["cost"] == pytest.approx((res["path_len"] - 1) * edge, rel=1e-12)
    # c_best strictly decreasing over successful replans
    rc = res["replan_cost"][:res["replans_run"]]
    solved = np.r_[True, rc[1:] < rc[:-1]] & np.isfinite(rc)
    assert np.all(np.diff(rc) <= 0) and solved.sum() == res["replans_solved"]
    # admissibility along the returned path: g + h <= g(goal)
    g = np.arange(res["path_len"]) * edge
    h = np.array([op.heuristic(x) for x in res["path_states"]])
    assert np.all(g + h <= res["cost"] + 1e-9)
    # a corrupted plan is rejected
    bad = res["path_controls"].copy()
    bad[len(bad) // 2] = -bad[len(bad) // 2] + 0.5
    assert op.validate_plan(res["path_states"], np.clip(bad, -1, 1))[0] != 0


def test_tree_invariants(orc, c1_plan):
    p, cfg, op, res = c1_plan
    T = res["tree"]
    n = T.n
    assert 1 < n <= cfg.tree_capacity
    par, cost = T.parents[:n], T.costs[:n]
    assert par[0] == -1 and np.all(par[1:] < np.arange(1, n)) and np.all(par[1:] >= 0)
    edge = p.steps_per_edge * float(np.float32(p.dt))
    np.testing.assert_allclose(cost[1:], cost[par[1:]] + edge, atol=1e-12)
    for i in np.random.default_rng(0).integers(1, n, 200):
        assert op.bounds_margin(T.states[i]) >= 0 and op.obstacle_margin(T.states[i]) > 0
        x, fl, *_ = op.propagate(T.states[par[i]], T.actions[i])
        assert fl & orc.F_VALID
        np.testing.assert_array_equal(x, T.states[i])


def test_plan_is_deterministic_and_seed_sensitive(orc):
    p, cfg = wl.config1()
    op = orc.OracleProblem(p)
    a = orc.plan(op, 3, 128, 4, 8192, 1, max_iters_per_replan=40)
    b = orc.plan(op, 3, 128, 4, 8192, 1, max_iters_per_replan=40)
    c = orc.plan(op, 4, 128, 4, 8192, 1, max_iters_per_replan=40)
    assert a["iterations"] == b["iterations"] and a["inserted"] == b["inserted"]
    np.testing.assert_array_equal(a["path_states"], b["path_states"])
    assert (a["inserted"], a["iterations"]) != (c["inserted"], c["iterations"])
