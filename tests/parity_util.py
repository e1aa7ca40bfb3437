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


def check_iteration(orc, op, problem, host_tree, out, after, ref, B, K, cap, strict_component_bits=False):
    """Asserts parity of one iteration; returns a small dict of statistics.  strict_component_bits=True drops
    reading P32's carve-out (used only to record, that the carve-out is needed whichever sine the
    kernel uses)."""
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
        if bit in (2, 4, 8) and not strict_component_bits:
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
    if same.all() and flags_equal:
        assert out["n_inserted"] == ref["n_inserted"]
        assert out["goal_node"] == ref["goal_node"]
    return dict(nn_equal=float(same.mean()), max_state_err=max_err, flags_equal=flags_equal,
                n_inserted=len(ins), n_goal=len(g))
