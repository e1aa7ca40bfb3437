"""Pins for the parts of the oracle that the round-2 mutation run found unpinned:
orc_validate_plan's three rejection codes and its per_edge switch, orc_plan's per-replan tree reset and re-keying of
the draws with the replan index (Alg. 1 l.1-4), the stream selector of SampleControls (Alg. 1 l.8,
PAPER.md:102), dropped goal children (reading P20) and the half-open wrap interval (reading P13).

Every expected value below is fixed by the problem statement itself (hand-built roll-outs of the linear double
integrator, counts, closed forms), not by re-running the function under test.
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl


def _di2(**kw):
    """C1's 2-D double integrator (Euler, dt = 0.05, 10 steps per edge) with hand-placed obstacles / goal."""
    p, _ = wl.config1()
    base = dict(obstacles=np.zeros((0, 3), np.float32), start=np.array([1.0, 1.0, 0.0, 0.0], np.float32),
                goal_center=np.array([1.0, 1.0], np.float32), goal_radius=0.05)
    base.update(kw)
    return dataclasses.replace(p, **base)


def _rollout(op, x0, controls):
    xs = [np.asarray(x0, np.float64)]
    for u in controls:
        x, fl, *_ = op.propagate(xs[-1], u)
        xs.append(x)
    return np.array(xs)


# Six edges of 0.5 s each: accelerate +x at 0.5 for three edges, brake for three (|v| stays below the box's 1).
# Euler with the OLD velocity (x += v dt, then v += u dt) over 10 steps of dt = fp32(0.05): written out below,
# no oracle call involved.
_U = np.array([[0.5, 0.0]] * 3 + [[-0.5, 0.0]] * 3)
_DT = float(np.float32(0.05))


def _closed_form_x(n_edges):
    x, v = 1.0, 0.0
    for e in range(n_edges):
        for _ in range(10):
            x += v * _DT
            v += _U[e, 0] * _DT
    return x, v


def test_validate_plan_accepts_the_hand_built_plan(orc):
    xe, ve = _closed_form_x(6)
    assert abs(ve) < 1e-12 and 2.05 < xe < 2.15        # comes to rest ~1.1 m further on (2 x 0.5 x 0.5 x 1.5^2 less Euler's lag)
    p = _di2(goal_center=np.array([xe, 1.0], np.float32))
    op = orc.OracleProblem(p)
    xs = _rollout(op, p.start, _U)
    assert xs[-1][0] == pytest.approx(xe, abs=1e-12)    # the roll-out is the closed form
    code, cost, err = op.validate_plan(xs, _U)
    assert code == 0 and err == 0.0
    assert cost == pytest.approx(6 * 10 * _DT, rel=1e-12)


def test_validate_plan_code_1_is_the_collision_check(orc):
    """The middle edge runs through a circle; every control is inside the box and the roll-out still ends in X_goal:
    only the validity check of the steps can object, and the code says so."""
    xe, _ = _closed_form_x(6)
    xm, _ = _closed_form_x(3)
    p = _di2(goal_center=np.array([xe, 1.0], np.float32),
             obstacles=np.array([[xm, 1.0, 0.05]], np.float32))   # on the path, clear of start and goal
    op = orc.OracleProblem(p)
    free = orc.OracleProblem(_di2(goal_center=np.array([xe, 1.0], np.float32)))
    xs = _rollout(free, p.start, _U)
    assert op.obstacle_margin(xs[3]) <= 0 < op.obstacle_margin(xs[0]) and op.obstacle_margin(xs[-1]) > 0
    assert op.in_goal(xs[-1])[0]
    assert op.validate_plan(xs, _U)[0] == 1
    assert op.validate_plan(xs, _U, per_edge=True)[0] == 1


def test_validate_plan_code_2_is_the_goal_check(orc):
    """A valid roll-out that stops one edge short of X_goal: collision free, controls in the box, exactly code 2."""
    xe, _ = _closed_form_x(6)
    p = _di2(goal_center=np.array([xe, 1.0], np.float32))
    op = orc.OracleProblem(p)
    xs = _rollout(op, p.start, _U)
    assert not op.in_goal(xs[5])[0] and op.in_goal(xs[6])[0]
    assert op.validate_plan(xs[:6], _U[:5])[0] == 2
    assert op.validate_plan(xs[:6], _U[:5], per_edge=True)[0] == 2
    assert op.validate_plan(xs, _U)[0] == 0


def test_validate_plan_code_3_is_the_control_box_check(orc):
    """One control component 1 % outside U (a push in y, braked again two edges later).  The goal ball is wide enough
    that the roll-out still ends inside it and nothing is in the way: only the control-box check can object."""
    xe, _ = _closed_form_x(6)
    p = _di2(goal_center=np.array([xe, 1.0], np.float32), goal_radius=1.0)
    op = orc.OracleProblem(p)
    u = _U.copy()
    u[1, 1], u[3, 1] = 1.01, -1.0
    xs = _rollout(op, p.start, u)
    assert op.in_goal(xs[-1])[0] and all(op.bounds_margin(x) > 0 for x in xs)
    assert op.validate_plan(xs, u)[0] == 3
    u[1, 1] = 1.0  # the rim of the box belongs to U
    xs = _rollout(op, p.start, u)
    assert op.in_goal(xs[-1])[0] and op.validate_plan(xs, u)[0] == 0


def test_validate_plan_per_edge_restarts_from_the_stored_node(orc):
    """Stored states that are each 1 mm further along x than the propagation of the previous STORED state: edge by edge
    (per_edge = 1, the tree-invariant form) every edge is off by exactly that 1 mm; as one roll-out from x_init
    (per_edge = 0) the offsets add up to 6 mm at the end (the model is linear, the offset is in position only)."""
    xe, _ = _closed_form_x(6)
    p = _di2(goal_center=np.array([xe, 1.0], np.float32), goal_radius=0.3)
    op = orc.OracleProblem(p)
    xs = [np.asarray(p.start, np.float64)]
    for u in _U:
        x, *_ = op.propagate(xs[-1], u)
        x[0] += 1e-3
        xs.append(x)
    xs = np.array(xs)
    code1, _, err1 = op.validate_plan(xs, _U, per_edge=True)
    code0, _, err0 = op.validate_plan(xs, _U, per_edge=False)
    assert code1 == 0 and code0 == 0
    assert err1 == pytest.approx(1e-3, abs=1e-12)
    assert err0 == pytest.approx(6e-3, abs=1e-12)


# ------------------------------------------------------------------ orc_plan: reset and re-keying per replan
def _unsolvable():
    """The goal sits behind a ring of circles: no replan can solve, every replan runs its full iteration cap."""
    ring = [[9.0 + 0.9 * math.cos(a), 9.0 + 0.9 * math.sin(a), 0.5] for a in np.linspace(0, 2 * math.pi, 12, endpoint=False)]
    return _di2(start=np.array([1.0, 1.0, 0.0, 0.0], np.float32), goal_center=np.array([9.0, 9.0], np.float32),
                goal_radius=0.2, obstacles=np.array(ring, np.float32))


def test_plan_starts_every_replan_from_a_fresh_tree(orc):
    """Alg. 1 l.4: T <- {x_init} at the head of EVERY replan.  With 2 iterations of B*K = 64 children a replan can hold
    at most 1 + 128 nodes; a tree carried over from the previous replan would exceed that in replan 1 or 2."""
    p = _unsolvable()
    op = orc.OracleProblem(p)
    B, K = 16, 4
    res = orc.plan(op, 3, B, K, 4096, 3, max_iters_per_replan=2)
    assert res["replans_run"] == 3 and res["replans_solved"] == 0 and res["outcome"] == 0
    assert list(res["replan_iters"]) == [2, 2, 2]
    assert all(1 < n <= 1 + 2 * B * K for n in res["replan_nodes"]), res["replan_nodes"]
    assert res["inserted"] == sum(int(n) - 1 for n in res["replan_nodes"])
    assert res["tree"].n == res["replan_nodes"][2]


def test_plan_keys_the_draws_with_the_replan_index(orc):
    """north_star (1): draws are keyed by (seed, REPLAN, iteration, sample, branch).  The tree orc_plan leaves behind
    after its last replan r = 2 must be the tree two hand-driven iterations with r = 2 grow from the root -- and not the
    one r = 0 grows (which a planner that forgot to pass r on would leave)."""
    p = _unsolvable()
    op = orc.OracleProblem(p)
    B, K, cap = 16, 4, 4096
    res = orc.plan(op, 3, B, K, cap, 3, max_iters_per_replan=2)
    trees = {}
    for r in (0, 2):
        T = orc.OracleTree(op, cap)
        T.reset()
        for it in range(2):
            orc.expand_iteration(op, T, 3, r, it, B, K)
        trees[r] = (T.n, T.states[:T.n].copy(), T.parents[:T.n].copy())
    n, states, parents = trees[2]
    assert res["tree"].n == n == res["replan_nodes"][2]
    np.testing.assert_array_equal(res["tree"].states[:n], states)
    np.testing.assert_array_equal(res["tree"].parents[:n], parents)
    n0, states0, _ = trees[0]
    assert n0 == res["replan_nodes"][0]
    assert n0 != n or not np.array_equal(states0, states)      # r really changes the draws
    # and the first sampled state of replan 1 is the (seed, r = 1, it = 0, s = 0) draw, word for word
    x = op.sample_state(3, 1, 0, 0)
    for d in range(4):
        w = orc.draw_word(3, 0, 1, 0, 0, 0, d)
        assert x[d] == orc.uniform_f32(w, float(p.state_lo[d]), float(p.state_hi[d]))
    assert not np.array_equal(x, op.sample_state(3, 0, 0, 0))


# ------------------------------------------------------------------ SampleControls draws from its own stream
def test_sample_control_uses_the_control_stream(orc):
    """Alg. 1 l.8 / reading P7: the control of (s, k) comes from the words of stream kind = 1 -- for k = 0 too, where a
    sampler reading the state stream (kind = 0) would hand back the first words of the sampled state x_rand(s)."""
    p, _ = wl.config1()
    op = orc.OracleProblem(p)
    for (seed, r, it, s, k) in [(0, 0, 0, 0, 0), (7, 2, 5, 31, 0), (7, 2, 5, 31, 3)]:
        u = op.sample_control(seed, r, it, s, k)
        for j in range(2):
            w1 = orc.draw_word(seed, it, r, s, 1, k, j)
            w0 = orc.draw_word(seed, it, r, s, 0, k, j)
            assert w1 != w0
            assert u[j] == orc.uniform_f32(w1, float(p.control_lo[j]), float(p.control_hi[j]))
            assert u[j] != orc.uniform_f32(w0, float(p.control_lo[j]), float(p.control_hi[j]))
    # a control box equal to the state box of dims 0, 1 would make state and control of (s, k = 0) collide if they shared
    # a stream: they must differ
    q = dataclasses.replace(p, control_lo=p.state_lo[:2].copy(), control_hi=p.state_hi[:2].copy())
    oq = orc.OracleProblem(q)
    assert not np.array_equal(oq.sample_control(1, 0, 0, 5, 0), oq.sample_state(1, 0, 0, 5)[:2])


# ------------------------------------------------------------------ P20: goal flags of dropped children are ignored
def test_goal_child_beyond_capacity_cannot_win(orc):
    """Reading P20: children are appended in ascending child index while the tree has room; a goal child that found no
    room is not in the tree, so it cannot end the replan.  The goal ball is the whole workspace (every kept child is a
    goal child); with room for exactly one more node the winner must be that node whatever the later children cost."""
    p, _ = wl.config1()
    p = dataclasses.replace(p, obstacles=p.obstacles[:0], goal_center=np.array([5.0, 5.0], np.float32), goal_radius=20.0,
                            start=np.array([5.0, 5.0, 0.0, 0.0], np.float32))
    op = orc.OracleProblem(p)
    B, K = 8, 2
    host = wl.random_tree(p, 40, seed=5)          # costs differ from node to node: children's costs differ too
    full = orc.OracleTree(op, 40 + B * K)
    full.load(host["states"], host["actions"], host["parents"], host["costs"])
    ref = orc.expand_iteration(op, full, 2, 0, 0, B, K)
    keep = np.nonzero((ref["child_flags"] & 1) != 0)[0]
    assert len(keep) >= 4 and np.all((ref["child_flags"][keep] & 16) != 0)
    first = keep[0]
    cheaper_later = keep[ref["child_cost"][keep] < ref["child_cost"][first]]
    assert len(cheaper_later) > 0, "pick another seed: the pin needs a cheaper goal child after the first kept one"
    assert ref["goal_node"] == 40 + int(np.nonzero(keep == keep[np.argmin(ref["child_cost"][keep])])[0][0])
    # now with room for one node only
    tight = orc.OracleTree(op, 41)
    tight.load(host["states"], host["actions"], host["parents"], host["costs"])
    out = orc.expand_iteration(op, tight, 2, 0, 0, B, K)
    assert out["n_inserted"] == 1 and tight.n == 41
    assert out["goal_node"] == 40 and out["new_c_best"] == ref["child_cost"][first]
    # and with no room at all nobody wins
    none = orc.OracleTree(op, 40)
    none.load(host["states"], host["actions"], host["parents"], host["costs"])
    out = orc.expand_iteration(op, none, 2, 0, 0, B, K)
    assert out["n_inserted"] == 0 and out["goal_node"] == -1 and not out["goal"]


# ------------------------------------------------------------------ P13: angles live in [-pi, pi)
def test_wrap_pi_interval_is_half_open(orc):
    assert orc.wrap_pi(math.pi) == -math.pi
    assert orc.wrap_pi(-math.pi) == -math.pi
    assert orc.wrap_pi(3 * math.pi) == pytest.approx(-math.pi, abs=1e-15) and orc.wrap_pi(3 * math.pi) < 0
    assert orc.wrap_pi(math.nextafter(math.pi, 0.0)) == math.nextafter(math.pi, 0.0)
