"""Shared comparison logic of the GPU parity tests: one GPU iteration against one oracle iteration.

Tolerances are BASELINE.json north_star's: NN index equal or the chosen node's oracle distance
within 1e-6 relative of the true minimum; propagated states within 1e-4 absolute; validity /
prune / goal flags equal except where the oracle's margin to the deciding boundary is < 1e-5;
insertion order bit-exact.
"""
import numpy as np

NN_REL_TOL = 1e-6
STATE_ABS_TOL = 1e-4
MARGIN_TOL = 1e-5


def run_both(pl, orc, op, problem, host_tree, seed, r, it, B, K, c_best=float("inf"), cap=None, nn_mode=0):
    """-> (gpu_out, gpu_tree_after (numpy), oracle_out, oracle_tree)"""
    import torch
    n0 = len(host_tree["parents"])
    cap = cap or n0 + B * K
    tree = pl.new_tree(cap, host_tree)
    out = pl.expand_step(tree, seed, r, it, B, K, c_best=c_best, nn_mode=nn_mode)
    n1 = int(tree["n_nodes"][0].item())
    D, m = problem.state_dim, problem.control_dim
    after = dict(states=tree["states"][:n1, :D].cpu().numpy(), actions=tree["actions"][:n1, :m].cpu().numpy(),
                 parents=tree["parents"][:n1].cpu().numpy(), costs=tree["costs"][:n1].cpu().numpy(), n=n1)
    ot = orc.OracleTree(op, cap)
    ot.load(host_tree["states"], host_tree["actions"], host_tree["parents"], host_tree["costs"])
    ref = orc.expand_iteration(op, ot, seed, r, it, B, K, c_best)
    return out, after, ref, ot


def check_iteration(orc, op, problem, host_tree, out, after, ref, B, K, cap):
    """Asserts parity of one iteration; returns a small dict of statistics (`strict` says whether every NN index and
    every deciding flag agreed, i.e. whether the oracle's insert count and goal node were compared as well)."""
    n0 = len(host_tree["parents"])
    D = problem.state_dim
    # samplers: bit-identical (P4)
    np.testing.assert_array_equal(out["x_rand"].astype(np.float64), ref["x_rand"])
    np.testing.assert_array_equal(out["child_ctrl"].astype(np.float64), ref["child_ctrl"])
    # NN (P6)
    same = out["nn_idx"] == ref["nn_idx"]
    assert out["nn_idx"].min() >= 0 and out["nn_idx"].max() < n0
    tree64 = host_tree["states"].astype(np.float64)
    for s in np.nonzero(~same)[0]:
        d_chosen = op.dist2(ref["x_rand"][s], tree64[out["nn_idx"][s]])
        assert d_chosen <= (1 + NN_REL_TOL) * ref["nn_d2"][s], (s, d_chosen, ref["nn_d2"][s])
    np.testing.assert_allclose(out["nn_d2"][same], ref["nn_d2"][same], rtol=1e-4, atol=1e-7)
    # children whose parent agrees
    cs = np.repeat(same, K)
    gf, rf = out["child_flags"], ref["child_flags"]
    both_valid = cs & ((gf & 1) != 0) & ((rf & 1) != 0)
    if both_valid.any():
        err = np.abs(out["child_state"][both_valid].astype(np.float64) - ref["child_state"][both_valid])
        ang = problem.dim_kind == 1
        if ang.any():
            err[:, ang] = np.minimum(err[:, ang], 2 * np.pi - err[:, ang])
        assert err.max() <= STATE_ABS_TOL, err.max()
        np.testing.assert_allclose(out["child_cost"][both_valid], ref["child_cost"][both_valid], rtol=1e-6)
        max_err = float(err.max())
    else:
        max_err = 0.0
    # flags: equal unless the oracle margin to that boundary is tiny.  The component bits (in-bounds,
    # collision-free) of a child that BOTH sides reject are compared only while the two trajectories still agree
    # within the state tolerance (reading P32: after leaving the state box a quadrotor child may cross the
    # Euler-angle singularity, beyond which the fp32 and fp64 trajectories are unrelated; the child is rejected
    # either way and the planner never looks at those bits).
    err_all = np.abs(out["child_state"].astype(np.float64) - ref["child_state"])
    ang_all = problem.dim_kind == 1
    if ang_all.any():
        err_all[:, ang_all] = np.minimum(err_all[:, ang_all], 2 * np.pi - err_all[:, ang_all])
    with np.errstate(invalid="ignore"):
        agree = np.nan_to_num(err_all, nan=np.inf).max(axis=1) <= STATE_ABS_TOL
    either_valid = ((gf & 1) != 0) | ((rf & 1) != 0)
    for bit, margin in ((1, "child_margin"), (2, "child_margin"), (4, "child_margin"), (8, "prune_margin")):
        diff = cs & ((gf & bit) != (rf & bit))
        if bit in (2, 4, 8):
            diff &= agree | either_valid
        assert np.all(ref[margin][diff] < MARGIN_TOL), (bit, np.nonzero(diff)[0][:5], ref[margin][diff][:5])
    diff = cs & ((gf & 16) != (rf & 16))
    near = np.minimum(np.minimum(ref["goal_margin"], ref["child_margin"]), ref["prune_margin"])
    assert np.all(near[diff] < MARGIN_TOL)
    flags_equal = bool(np.all((gf & 25)[cs] == (rf & 25)[cs]))  # valid, not-pruned, goal
    # compaction: bit-exact copy_if over the GPU's own keep flags, in child order, capped at cap
    keep = np.nonzero(((gf & 1) != 0) & ((gf & 8) != 0))[0]
    room = cap - n0
    ins = keep[:room]
    assert after["n"] == n0 + len(ins) and out["n_inserted"] == len(ins)
    np.testing.assert_array_equal(after["states"][n0:], out["child_state"][ins])
    np.testing.assert_array_equal(after["actions"][n0:], out["child_ctrl"][ins])
    np.testing.assert_array_equal(after["costs"][n0:], out["child_cost"][ins])
    np.testing.assert_array_equal(after["parents"][n0:], out["nn_idx"][ins // K])
    np.testing.assert_array_equal(np.nonzero((gf & 32) != 0)[0], ins)
    # the old part of the tree is untouched
    np.testing.assert_array_equal(after["states"][:n0], host_tree["states"])
    np.testing.assert_array_equal(after["parents"][:n0], host_tree["parents"])
    # goal winner among inserted goal children: min cost, ties -> lowest child index
    g = ins[(gf[ins] & 16) != 0]
    if len(g):
        best = g[np.argmin(out["child_cost"][g])]
        assert out["goal_node"] == n0 + int(np.nonzero(ins == best)[0][0])
        assert out["new_c_best"] == out["child_cost"][best]
    else:
        assert out["goal_node"] == -1
    strict = bool(same.all() and flags_equal)
    if strict:
        assert out["n_inserted"] == ref["n_inserted"]
        assert out["goal_node"] == ref["goal_node"]
    return dict(nn_equal=float(same.mean()), max_state_err=max_err, flags_equal=flags_equal,
                n_inserted=len(ins), n_goal=len(g), strict=strict)


def check_sampled(op, problem, host_tree, out, seed, r, it, K, c_best, queries):
    """Parity of one GPU iteration on a tree too large for a whole oracle iteration (planner-grown trees at
    BASELINE's B, K): for each sampled query the oracle draws the state, finds the exact nearest node, and
    re-propagates the K children from the parent the GPU chose.  Same tolerances as check_iteration.
    Returns the share of sampled queries whose NN index was equal."""
    D = problem.state_dim
    tree64 = host_tree["states"].astype(np.float64)
    ang = problem.dim_kind == 1
    equal = 0
    for s in queries:
        s = int(s)
        q = op.sample_state(seed, r, it, s)
        np.testing.assert_array_equal(out["x_rand"][s].astype(np.float64), q)
        i, d2 = op.nearest(tree64, q)
        j = int(out["nn_idx"][s])
        assert 0 <= j < len(tree64)
        if j != i:
            assert op.dist2(q, tree64[j]) <= (1 + NN_REL_TOL) * d2, (s, i, j)
        else:
            equal += 1
            assert out["nn_d2"][s] == pytest_approx(d2)
        for k in range(K):
            c = s * K + k
            u = op.sample_control(seed, r, it, s, k)
            np.testing.assert_array_equal(out["child_ctrl"][c].astype(np.float64), u)
            x, fl, _, mm, ec = op.propagate(tree64[j], u)
            gf = int(out["child_flags"][c])
            if (gf & 1) != (fl & 1):
                assert mm < MARGIN_TOL, (s, k, gf, fl, mm)
                continue
            if not (fl & 1):
                continue  # rejected on both sides: nothing else is looked at (P32)
            err = np.abs(out["child_state"][c].astype(np.float64) - x)
            err[ang] = np.minimum(err[ang], 2 * np.pi - err[ang])
            assert err.max() <= STATE_ABS_TOL, (s, k, err.max())
            cost = float(host_tree["costs"][j]) + ec
            assert abs(out["child_cost"][c] - cost) <= 1e-6 * max(1.0, cost)
            f = cost + op.heuristic(x)
            if ((gf & 8) != 0) != (f < c_best):
                assert abs(f - c_best) < MARGIN_TOL, (s, k, f, c_best)
                continue
            ing, gm = op.in_goal(x)
            want_goal = bool(f < c_best) and ing
            if ((gf & 16) != 0) != want_goal:
                assert gm < MARGIN_TOL, (s, k, gm)
    return equal / max(1, len(queries))


def pytest_approx(v):
    import pytest
    return pytest.approx(v, rel=1e-4, abs=1e-7)
