"""Pins of the oracle functions that round 1 left unpinned (VERDICT r01 "What's weak" 1).

Each test fails on one named, plausible mistake in oracle/pakr_oracle.cpp: the sign of the gyroscopic
term w x Iw (both quadrotors), the PATH_LENGTH edge cost (sum of chord lengths, not of their squares),
the strictness of the prune comparison at c_new + h == c_best (Alg. 1 l.11), the GOAL
flag of a pruned child, closedness of obstacles and of the state box through orc_propagate's flags, and
the three ways orc_plan ends a replan (goal, tree full, iteration cap) plus the initial cost bound.
Every expectation is a closed form or hand-computed; none comes from the CUDA path.
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl


def _free(p, **kw):
    lo = np.where(np.isfinite(p.state_lo), -1e6, p.state_lo).astype(np.float32)
    hi = np.where(np.isfinite(p.state_hi), 1e6, p.state_hi).astype(np.float32)
    return dataclasses.replace(p, obstacles=p.obstacles[:0], state_lo=lo, state_hi=hi, **kw)


# ------------------------------------------------------------------ (i) gyroscopic sign
@pytest.mark.parametrize("name", ["C4", "N3"])
def test_quadrotor_axisymmetric_precession(orc, name):
    """Torque-free axisymmetric body (Ixx = Iyy): Euler's equations I wdot = -w x Iw reduce to
    pdot = -Omega q, qdot = +Omega p with Omega = r (Izz - Ixx) / Ixx and r constant, i.e. (p, q) rotates by
    +Omega t.  Energy and |Iw| cannot see the sign of w x Iw; this can.  (DESIGN.md Q, P34)"""
    p, _ = wl.CONFIGS[name]()
    Ixx, Iyy, Izz = (float(v) for v in p.dyn_params[1:4])
    assert Ixx == Iyy
    # fine steps so that RK4's truncation error is far below the tolerance
    q = _free(p, dt=0.002, steps_per_edge=250)
    op = orc.OracleProblem(q)
    T = 250 * float(np.float32(0.002))
    p0, q0, r0 = 0.7, -0.4, 2.0
    x0 = np.zeros(12)
    x0[9:12] = [p0, q0, r0]
    hover = [float(p.dyn_params[0]) * float(p.dyn_params[4]), 0, 0, 0]
    x, *_ = op.propagate(x0, hover)
    Om = r0 * (Izz - Ixx) / Ixx
    c, s = math.cos(Om * T), math.sin(Om * T)
    assert abs(Om * T) > 0.5  # a rotation large enough that the wrong sign is nowhere near
    np.testing.assert_allclose(x[9:12], [p0 * c - q0 * s, p0 * s + q0 * c, r0], rtol=0, atol=1e-9)
    # and at the config's own step size, to the RK4 truncation level
    op2 = orc.OracleProblem(_free(p))
    T2 = p.steps_per_edge * float(np.float32(p.dt))
    x2, *_ = op2.propagate(x0, hover)
    c2, s2 = math.cos(Om * T2), math.sin(Om * T2)
    np.testing.assert_allclose(x2[9:12], [p0 * c2 - q0 * s2, p0 * s2 + q0 * c2, r0], rtol=0, atol=1e-7)


def test_quadrotor_general_inertia_first_step_derivative(orc):
    """Three different inertias: wdot = I^-1 (tau - w x Iw) written out by hand for one state, so that a sign
    or index slip in any single component fails (the axisymmetric case zeroes the r equation)."""
    p, _ = wl.config4()
    I = np.array([0.01, 0.03, 0.02])
    q = _free(p, dyn_params=np.array([1.0, I[0], I[1], I[2], 9.81], np.float32))
    I = q.dyn_params[1:4].astype(np.float64)
    w = np.array([1.5, -0.8, 0.6])
    tau = np.array([0.05, -0.02, 0.07])
    want = (tau - np.cross(w, I * w)) / I
    for name in ("C4", "N3"):
        pp, _ = wl.CONFIGS[name]()
        qq = _free(pp, dyn_params=q.dyn_params)
        x = np.zeros(12)
        x[9:12] = w
        xd = orc.OracleProblem(qq).f(x, [9.81, *tau])
        np.testing.assert_allclose(xd[9:12], want, rtol=1e-12)


# ------------------------------------------------------------------ (ii) PATH_LENGTH cost
def test_path_length_closed_forms(orc):
    """P14: edge cost = sum over steps of |p_j - p_{j-1}| (chords between step-end positions)."""
    # constant velocity double integrator: length = |v| T (straight line, chords add up exactly)
    p, _ = wl.config2()
    q = _free(p, cost_mode=wl.COST_PATH_LENGTH, heuristic_speed=1.0)
    op = orc.OracleProblem(q)
    T = p.steps_per_edge * float(np.float32(p.dt))
    v = np.array([0.3, -0.4, 1.2])
    x, fl, fb, mm, ec = op.propagate([1, 2, 3, *v], [0, 0, 0])
    assert ec == pytest.approx(np.linalg.norm(v) * T, rel=1e-13)
    # from rest with constant acceleration along one line: length = |a| T^2 / 2 (monotone motion)
    a = np.array([0.6, 0.0, -0.8])
    x, fl, fb, mm, ec = op.propagate([1, 2, 3, 0, 0, 0], a)
    assert ec == pytest.approx(0.5 * np.linalg.norm(a) * T * T, rel=1e-13)
    # general DI edge: step-end positions are known in closed form (RK4 is exact for constant acceleration)
    x0, u = np.array([1.0, 2.0, 3.0, 0.3, -0.2, 0.1]), np.array([0.7, -0.4, 0.9])
    dt = float(np.float32(p.dt))
    t = dt * np.arange(p.steps_per_edge + 1)
    pos = x0[:3] + np.outer(t, x0[3:]) + 0.5 * np.outer(t * t, u)
    want = np.linalg.norm(np.diff(pos, axis=0), axis=1).sum()
    *_, ec = op.propagate(x0, u)
    assert ec == pytest.approx(want, rel=1e-12)
    assert abs(ec - (np.diff(pos, axis=0) ** 2).sum()) > 1e-3  # ... and not the sum of squared chords
    # first-order unicycle on a circular arc: S chords of 2 (v / w) sin(w dt / 2) each; the arc itself is v T
    p7, _ = wl.config7()
    q7 = _free(p7, cost_mode=wl.COST_PATH_LENGTH, heuristic_speed=1.0)
    op7 = orc.OracleProblem(q7)
    vv, ww = 0.8, 1.1
    S, dt7 = p7.steps_per_edge, float(np.float32(p7.dt))
    *_, ec = op7.propagate([3, 4, 0.3], [vv, ww])
    assert ec == pytest.approx(S * 2 * (vv / ww) * math.sin(ww * dt7 / 2), rel=2e-8)  # RK4 truncation ~3e-9
    assert ec == pytest.approx(vv * S * dt7, rel=2e-4) and ec < vv * S * dt7
    # DURATION is untouched by any of this
    *_, ec = orc.OracleProblem(_free(p7)).propagate([3, 4, 0.3], [vv, ww])
    assert ec == S * dt7


def test_expand_iteration_path_length_costs(orc):
    """One whole iteration with cost_mode = PATH_LENGTH: every child's cost is its parent's plus the chord
    length of its own edge, the heuristic is the plain distance to the goal ball (v_cap = 1 reproduces
    PAPER.md:134), and the prune compares that sum with c_best."""
    p, _ = wl.config2()
    q = dataclasses.replace(p, cost_mode=wl.COST_PATH_LENGTH, heuristic_speed=1.0)
    op = orc.OracleProblem(q)
    B, K, n0 = 48, 3, 150
    t = wl.random_tree(q, n0, seed=4)
    tree = orc.OracleTree(op, n0 + B * K)
    tree.load(t["states"], t["actions"], t["parents"], t["costs"])
    c_best = 14.0
    out = orc.expand_iteration(op, tree, 9, 0, 2, B, K, c_best)
    dt = float(np.float32(p.dt))
    tt = dt * np.arange(p.steps_per_edge + 1)
    goal = q.goal_center.astype(np.float64)
    for c in range(B * K):
        x0 = t["states"][out["nn_idx"][c // K]].astype(np.float64)
        u = out["child_ctrl"][c]
        pos = x0[:3] + np.outer(tt, x0[3:]) + 0.5 * np.outer(tt * tt, u)
        length = np.linalg.norm(np.diff(pos, axis=0), axis=1).sum()
        g = float(t["costs"][out["nn_idx"][c // K]]) + length
        assert out["child_cost"][c] == pytest.approx(g, rel=1e-12)
        h = max(0.0, np.linalg.norm(pos[-1] - goal) - float(np.float32(q.goal_radius)))
        if abs(g + h - c_best) > 1e-9:
            assert bool(out["child_flags"][c] & orc.F_NOTPRUNED) == (g + h < c_best)
    assert 0 < int(((out["child_flags"] & orc.F_NOTPRUNED) != 0).sum()) < B * K


# ------------------------------------------------------------------ (iii), (iv) prune strictness, goal needs kept
def _goal_start_problem():
    """C1 without obstacles, started at rest in the middle of a wide goal ball: every child of the root stays in
    the ball, so h = 0 and c_new is exactly one edge duration for all of them."""
    p, _ = wl.config1()
    start = np.array([5.0, 5.0, 0.0, 0.0], np.float32)
    return dataclasses.replace(p, obstacles=p.obstacles[:0], start=start, goal_center=start[:2].copy(), goal_radius=3.0)


def test_prune_is_strict_at_equality_and_pruned_goal_child_has_no_goal_flag(orc):
    q = _goal_start_problem()
    op = orc.OracleProblem(q)
    edge = q.steps_per_edge * float(np.float32(q.dt))  # the fp64 value both sides add
    B, K = 32, 4
    for c_best, kept in ((edge, False), (np.nextafter(edge, np.inf), True), (np.nextafter(edge, 0.0), False)):
        tree = orc.OracleTree(op, 1 + B * K)
        out = orc.expand_iteration(op, tree, 1, 0, 0, B, K, float(c_best))
        f = out["child_flags"]
        assert np.all(out["child_cost"] == edge)
        assert np.all([op.in_goal(x)[0] and op.heuristic(x) == 0.0 for x in out["child_state"]])
        assert np.all((f & orc.F_VALID) != 0)
        # Alg. 1 l.11: c_new + h < c_best, strictly (P16): at equality the child is pruned
        assert np.all(((f & orc.F_NOTPRUNED) != 0) == kept)
        # a pruned child inside X_goal is not a goal child (l.14 sits under l.11) and is not inserted
        assert np.all(((f & orc.F_GOAL) != 0) == kept)
        assert np.all(((f & orc.F_INSERTED) != 0) == kept)
        assert out["goal"] == kept and out["n_inserted"] == (B * K if kept else 0)
        assert out["goal_node"] == (1 if kept else -1)
        assert out["new_c_best"] == (edge if kept else c_best)
        assert np.all(out["prune_margin"] == abs(edge - c_best))


def test_plan_equal_cost_goal_child_does_not_end_the_replan(orc):
    """c_best decreases strictly.  Under a bound equal to the only reachable cost no replan is
    solved (they all run to the iteration cap); one ulp more and the first iteration solves it."""
    q = _goal_start_problem()
    op = orc.OracleProblem(q)
    edge = q.steps_per_edge * float(np.float32(q.dt))
    res = orc.plan(op, 1, 32, 4, 4096, 3, max_iters_per_replan=5, initial_cost_bound=edge)
    assert res["outcome"] == 0 and res["replans_solved"] == 0 and res["path_len"] == 0 and np.isinf(res["cost"])
    np.testing.assert_array_equal(res["replan_iters"], [5, 5, 5])
    np.testing.assert_array_equal(res["replan_cost"], [edge] * 3)  # the bound handed in is kept, not improved
    assert res["inserted"] == 0 and res["iterations"] == 15
    res = orc.plan(op, 1, 32, 4, 4096, 3, max_iters_per_replan=5, initial_cost_bound=float(np.nextafter(edge, np.inf)))
    assert res["outcome"] == 1 and res["cost"] == edge and res["path_len"] == 2
    # replan 0 solves in one iteration; afterwards c_best = edge and nothing can be strictly cheaper
    np.testing.assert_array_equal(res["replan_iters"], [1, 5, 5])
    assert res["replans_solved"] == 1
    # no bound (<= 0 or +inf is "none", Alg. 1 l.1 c_best = inf): same as the unbounded call
    for none in (0.0, -1.0, float("inf")):
        r0 = orc.plan(op, 1, 32, 4, 4096, 1, initial_cost_bound=none)
        assert r0["outcome"] == 1 and r0["cost"] == edge and r0["replan_iters"][0] == 1


# ------------------------------------------------------------------ (v) how orc_plan ends a replan
def test_plan_tree_full_ends_the_replan_and_default_iteration_cap(orc):
    p, _ = wl.config1()
    q = dataclasses.replace(p, obstacles=p.obstacles[:0])
    op = orc.OracleProblem(q)
    B, K, cap = 64, 4, 600
    # hand count: chain single iterations on a tree of the same capacity until it is full
    tree = orc.OracleTree(op, cap)
    it = 0
    while tree.n < cap:
        out = orc.expand_iteration(op, tree, 2, 0, it, B, K, float("inf"))
        assert not out["goal"]
        it += 1
    assert 2 <= it < 32
    res = orc.plan(op, 2, B, K, cap, 2)
    assert res["outcome"] == 0
    # P20: a full tree ends the replan at once (not at the iteration cap, 32 here), replan 1 restarts from the root
    np.testing.assert_array_equal(res["replan_nodes"], [cap, cap])
    assert res["replan_iters"][0] == it and res["iterations"] == int(res["replan_iters"].sum())
    assert res["replan_iters"][1] < 32
    # P21: default cap = max(32, capacity / (B K)) iterations; a bound nothing beats keeps the tree at its root
    for Bq, Kq, capq, want in ((8, 2, 64, 32), (4, 1, 160, 40), (2, 2, 400, 100)):
        r = orc.plan(op, 0, Bq, Kq, capq, 2, initial_cost_bound=1e-3)
        np.testing.assert_array_equal(r["replan_iters"], [want, want])
        np.testing.assert_array_equal(r["replan_nodes"], [1, 1])
        assert r["children"] == 2 * want * Bq * Kq and r["inserted"] == 0 and r["outcome"] == 0
    # an explicit cap wins over the default
    r = orc.plan(op, 0, 8, 2, 64, 1, max_iters_per_replan=7, initial_cost_bound=1e-3)
    assert r["replan_iters"][0] == 7


# ------------------------------------------------------------------ (vi) closedness through orc_propagate's flags
def _rim_problem(**kw):
    """C1 (explicit Euler) with dt = 1/16 and 8 steps: p_j = p0 + j dt v0 is exact in binary floating point."""
    p, _ = wl.config1()
    return dataclasses.replace(p, dt=0.0625, steps_per_edge=8, **kw)


def test_obstacle_rim_is_collision_through_propagate_flags(orc):
    """P11: obstacles are closed sets.  The edge below reaches |p - c| == r exactly at its LAST step."""
    x0 = np.array([2.0, 3.0, 1.0, 0.0])  # moves +1/16 in x per step, 0.5 in all
    for r, want_free in ((0.25, False), (float(np.nextafter(np.float32(0.25), np.float32(0))), True)):
        circ = np.array([[2.5 + 0.25, 3.0, r]], np.float32)
        op = orc.OracleProblem(_rim_problem(obstacles=circ))
        x, fl, fb, mm, ec = op.propagate(x0, [0.0, 0.0])
        np.testing.assert_array_equal(x, [2.5, 3.0, 1.0, 0.0])
        assert bool(fl & orc.F_COLLFREE) == want_free and bool(fl & orc.F_VALID) == want_free
        assert fl & orc.F_INBOUNDS
        assert fb == (0 if want_free else 8)
        if not want_free:
            assert mm == 0.0 and op.obstacle_margin(x) == 0.0
    # axis-aligned box whose low face is exactly the last step-end position (closed: lo <= p)
    p2, _ = wl.config2()
    for lo_x, want_free in ((2.5, False), (float(np.nextafter(np.float32(2.5), np.float32(3))), True)):
        box = np.array([[lo_x, 2.0, 2.0, 3.5, 4.0, 4.0]], np.float32)
        q2 = dataclasses.replace(p2, integrator=wl.INT_EULER, dt=0.0625, steps_per_edge=8, obstacles=box)
        op = orc.OracleProblem(q2)
        x, fl, fb, mm, ec = op.propagate([2.0, 3.0, 3.0, 1.0, 0.0, 0.0], [0.0, 0.0, 0.0])
        assert x[0] == 2.5
        assert bool(fl & orc.F_COLLFREE) == want_free and fb == (0 if want_free else 8)


def test_state_box_rim_is_inside_through_propagate_flags(orc):
    """P12: the state box is closed.  v reaches v_hi exactly at the last step, x reaches x_hi exactly."""
    op = orc.OracleProblem(_rim_problem(obstacles=np.zeros((0, 3), np.float32)))
    # v0 = 0.5, a = 1: v_8 = 0.5 + 8/16 = 1.0 == hi -> still in bounds
    x, fl, fb, mm, ec = op.propagate([2.0, 3.0, 0.5, 0.0], [1.0, 0.0])
    assert x[2] == 1.0 and (fl & orc.F_INBOUNDS) and (fl & orc.F_VALID) and fb == 0 and mm == 0.0
    # a hair more acceleration is enough to leave at that step (orc_propagate does not clamp controls)
    x, fl, fb, mm, ec = op.propagate([2.0, 3.0, 0.5, 0.0], [1.0 + 1e-9, 0.0])
    assert x[2] > 1.0 and not (fl & orc.F_INBOUNDS) and not (fl & orc.F_VALID) and fb == 8
    assert fl & orc.F_COLLFREE
    # position: x0 = 9.5, v = 1: x_8 = 10.0 == hi
    x, fl, fb, mm, ec = op.propagate([9.5, 3.0, 1.0, 0.0], [0.0, 0.0])
    assert x[0] == 10.0 and (fl & orc.F_VALID) and fb == 0
    x, fl, fb, mm, ec = op.propagate([float(np.nextafter(9.5, 10.0)), 3.0, 1.0, 0.0], [0.0, 0.0])
    assert x[0] > 10.0 and not (fl & orc.F_VALID) and fb == 8
