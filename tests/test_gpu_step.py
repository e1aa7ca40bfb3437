"""GPU parity of one expansion iteration (pakr_expand_step through the C ABI) against the oracle.

Teacher forcing (SURVEY.md 8(c) "T"): both sides start from the same tree snapshot and the same
(seed, replan, iteration) and must agree element by element under north_star's tolerances
(tests/parity_util.py).
"""
import dataclasses

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
    mod.lib()  # fails loudly if the extension is missing
    return mod


_CASES = [
    # config, n_tree, B, K
    ("C1", 1, 256, 4),
    ("C1", 31, 100, 3),
    ("C1", 33, 129, 1),
    ("C1", 4097, 256, 4),
    ("C2", 32, 64, 8),
    ("C2", 4095, 300, 5),
    ("C2", 20000, 1024, 8),
    ("C3", 4096, 257, 7),
    ("C3", 9000, 512, 8),
    ("C4", 2500, 384, 16),
    ("C4", 12345, 200, 9),
    ("C4", 30000, 1024, 16),
    ("C5", 7777, 256, 16),
    ("N1", 6000, 512, 8),   # Dubins airplane (NEXT-2)
    ("N1", 31, 100, 3),
    ("N2", 4097, 300, 5),   # first-order unicycle (NEXT-2)
    ("N2", 20000, 1024, 8),
    ("N3", 2500, 384, 16),  # quadcopter with body-frame velocities, PAPER.md:174 (NEXT-2)
    ("N3", 15000, 1024, 8),
    ("N4", 1, 64, 4),       # Acrobot, PAPER.md:209 (NEXT-2): two angle dims, goal ball in angle space
    ("N4", 4097, 300, 5),
    ("N4", 20000, 1024, 8),
    # B*K > 65,536 (more than 2048 warp units: the insert's per-thread-chunk prefix) and K = 64, as config 5 runs them
    ("C2", 5000, 2048, 64),   # B*K = 131,072
    ("C5", 5000, 4096, 64),   # B*K = 262,144, 128 boxes
    ("C2", 3000, 16384, 64),  # B*K = 2^20
    ("C4", 4000, 8192, 16),   # B*K = 131,072 on the 12-D model
]


@pytest.mark.parametrize("name,n0,B,K", _CASES)
def test_step_matches_oracle(pakr, orc, name, n0, B, K):
    from parity_util import check_iteration, run_both
    p, _ = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, n0, seed=n0 + B)
    cap = n0 + B * K
    out, after, ref, _ = run_both(pl, orc, op, p, host, seed=11, r=2, it=5, B=B, K=K, cap=cap)
    st = check_iteration(orc, op, p, host, out, after, ref, B, K, cap)
    assert st["nn_equal"] > 0.99
    _STRICT[(name, n0, B, K)] = st["strict"]
    pl.close()


_STRICT = {}


def test_step_matches_oracle_compared_the_insert_counts():
    """check_iteration compares the oracle's insert count and goal node only when every NN index and deciding flag
    agreed.  That must have been the case on most of the cases above, the smallest ones included: otherwise the
    oracle's own insert is never looked at."""
    if not _STRICT:
        pytest.skip("test_step_matches_oracle did not run in this session")
    ran = [k for k, v in _STRICT.items() if v]
    assert len(ran) >= len(_STRICT) // 2, (len(ran), len(_STRICT))
    small = [k for k in _STRICT if k[2] * k[3] <= 2048]
    assert small and all(_STRICT[k] for k in small), {k: _STRICT[k] for k in small}


def test_step_duplicates_and_ties(pakr, orc):
    """Duplicate nodes: the lowest index must win in every NN variant / tile split (P6, P26)."""
    from parity_util import check_iteration, run_both
    p, _ = wl.config2()
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, 6000, seed=3)
    host["states"][3000:] = host["states"][:3000]  # every node appears twice
    out, after, ref, _ = run_both(pl, orc, op, p, host, seed=1, r=0, it=0, B=512, K=2)
    np.testing.assert_array_equal(out["nn_idx"], ref["nn_idx"])
    assert out["nn_idx"].max() < 3000
    check_iteration(orc, op, p, host, out, after, ref, 512, 2, 6000 + 1024)
    pl.close()


def test_step_query_equals_node_and_zero_weight(pakr, orc):
    from parity_util import check_iteration, run_both
    p, _ = wl.config4()
    w = p.nn_weight.copy()
    w[3:] = 0.0  # NN over position only (PAPER.md:286 subset of dims)
    p = dataclasses.replace(p, nn_weight=w)
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, 5000, seed=4)
    # plant the exact sampled states of the first queries as nodes: their NN is that node, d2 == 0
    for s in range(8):
        host["states"][1000 + s] = op.sample_state(21, 0, 3, s).astype(np.float32)
    out, after, ref, _ = run_both(pl, orc, op, p, host, seed=21, r=0, it=3, B=128, K=4)
    np.testing.assert_array_equal(out["nn_idx"][:8], 1000 + np.arange(8))
    assert np.all(out["nn_d2"][:8] == 0.0)
    check_iteration(orc, op, p, host, out, after, ref, 128, 4, 5000 + 512)
    pl.close()


def test_step_prune_goal_and_overflow(pakr, orc):
    """Finite c_best prunes; goal children are inserted and the winner is the cheapest, lowest index;
    a full tree takes only the first cap - n survivors (P16, P19, P20)."""
    from parity_util import check_iteration, run_both
    p, _ = wl.config1()
    p = dataclasses.replace(p, obstacles=p.obstacles[:2], goal_radius=2.5)
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    n0 = 400
    rng = np.random.default_rng(0)
    host = wl.random_tree(p, n0, seed=9)
    host["states"][1:, :2] = rng.uniform(7.0, 9.8, size=(n0 - 1, 2)).astype(np.float32)
    host["states"][1:, 2:] = rng.uniform(-0.5, 0.5, size=(n0 - 1, 2)).astype(np.float32)
    B, K = 256, 4
    for c_best, cap in ((float("inf"), n0 + B * K), (4.0, n0 + B * K), (float("inf"), n0 + 37), (0.0, n0 + B * K)):
        out, after, ref, _ = run_both(pl, orc, op, p, host, seed=5, r=1, it=0, B=B, K=K, c_best=c_best, cap=cap)
        st = check_iteration(orc, op, p, host, out, after, ref, B, K, cap)
        if c_best == float("inf") and cap > n0 + 37:
            assert st["n_goal"] > 3 and out["goal_node"] >= n0
        if c_best == 0.0:
            assert st["n_inserted"] == 0 and after["n"] == n0
        if cap == n0 + 37:
            assert after["n"] == cap
    pl.close()


def test_step_goal_ball_over_listed_dims(pakr, orc):
    """pakr_problem.goal_dims: (i) the Acrobot's ball in (theta1, theta2) around (pi, 0) with nodes parked on both
    sides of the +-pi seam, so the wrapped difference decides; (ii) a double integrator whose goal ball spans a
    position AND a velocity dim (h = 0).  Goal flags, winner and c_best must match the oracle."""
    from parity_util import check_iteration, run_both
    p, _ = wl.CONFIGS["N4"]()
    rng = np.random.default_rng(3)
    n0, B, K = 600, 256, 4
    host = wl.random_tree(p, n0, seed=4)
    side = np.where(rng.random(n0 - 1) < 0.5, 1.0, -1.0)
    host["states"][1:, 0] = (side * (np.pi - rng.uniform(0.02, 0.5, n0 - 1))).astype(np.float32)
    host["states"][1:, 1] = rng.uniform(-0.5, 0.5, n0 - 1).astype(np.float32)
    host["states"][1:, 2:] = rng.uniform(-1.0, 1.0, (n0 - 1, 2)).astype(np.float32)
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    for c_best in (float("inf"), 3.0):
        out, after, ref, _ = run_both(pl, orc, op, p, host, seed=2, r=0, it=3, B=B, K=K, c_best=c_best)
        st = check_iteration(orc, op, p, host, out, after, ref, B, K, n0 + B * K)
        if c_best == float("inf"):
            assert st["n_goal"] > 5
            goal_rows = after["states"][n0:][(out["child_flags"][(out["child_flags"] & 32) != 0] & 16) != 0]
            assert (goal_rows[:, 0] > 2.5).any() and (goal_rows[:, 0] < -2.5).any()  # both sides of the seam
    pl.close()
    p1, _ = wl.config1()
    p1 = dataclasses.replace(p1, obstacles=p1.obstacles[:2], goal_dims=np.array([1, 2], np.int32),
                             goal_center=np.array([9.0, 0.25], np.float32), goal_radius=0.6, heuristic_speed=float("inf"))
    host = wl.random_tree(p1, 400, seed=9)
    host["states"][1:, 1] = rng.uniform(8.0, 9.8, 399).astype(np.float32)
    pl = pakr.Planner(p1)
    op = orc.OracleProblem(p1)
    out, after, ref, _ = run_both(pl, orc, op, p1, host, seed=5, r=1, it=0, B=B, K=K)
    st = check_iteration(orc, op, p1, host, out, after, ref, B, K, 400 + B * K)
    assert 3 < st["n_goal"] < st["n_inserted"]
    pl.close()


def test_step_path_length_cost_mode(pakr, orc):
    from parity_util import check_iteration, run_both
    p, _ = wl.config2()
    p = dataclasses.replace(p, cost_mode=wl.COST_PATH_LENGTH, heuristic_speed=1.0)
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, 3000, seed=2)
    out, after, ref, _ = run_both(pl, orc, op, p, host, seed=8, r=0, it=1, B=256, K=4, c_best=30.0)
    check_iteration(orc, op, p, host, out, after, ref, 256, 4, 3000 + 1024)
    pl.close()


def test_teacher_forced_run_c2(pakr, orc):
    """Grow a tree with the GPU from the root; at sampled iterations hand the GPU's snapshot to the
    oracle and compare that one iteration."""
    from parity_util import check_iteration
    import torch
    p, _ = wl.config2()
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    B, K, cap = 256, 8, 60000
    tree = pl.new_tree(cap)
    D, m = p.state_dim, p.control_dim
    for it in range(14):
        n0 = int(tree["n_nodes"][0].item())
        snap = dict(states=tree["states"][:n0, :D].cpu().numpy(), actions=tree["actions"][:n0, :m].cpu().numpy(),
                    parents=tree["parents"][:n0].cpu().numpy(), costs=tree["costs"][:n0].cpu().numpy())
        out = pl.expand_step(tree, 3, 0, it, B, K)
        if it in (0, 1, 5, 13):
            n1 = int(tree["n_nodes"][0].item())
            after = dict(states=tree["states"][:n1, :D].cpu().numpy(), actions=tree["actions"][:n1, :m].cpu().numpy(),
                         parents=tree["parents"][:n1].cpu().numpy(), costs=tree["costs"][:n1].cpu().numpy(), n=n1)
            ot = orc.OracleTree(op, cap)
            ot.load(snap["states"], snap["actions"], snap["parents"], snap["costs"])
            ref = orc.expand_iteration(op, ot, 3, 0, it, B, K)
            check_iteration(orc, op, p, snap, out, after, ref, B, K, cap)
    assert int(tree["n_nodes"][0].item()) > 2000
    pl.close()


@pytest.mark.parametrize("name,n0,B,finite", [
    ("C2", 300000, None, False), ("C3", 200000, None, True), ("C4", 150000, None, True), ("C5", 120000, None, False),
    # tree sizes of the NN microbenchmarks (SURVEY.md 7 stage 4: 2^20; bench.py --what phases: 2^20 .. 2^23)
    ("C2", 1 << 20, None, True), ("C4", 1 << 22, None, False), ("C5", 1 << 20, 16384, False),
    ("C2", 1 << 23, 8, False), ("C4", 1 << 23, 4, False),   # streaming tier at the size its roofline is quoted on
])
def test_full_size_sampled(pakr, orc, name, n0, B, finite):
    """BASELINE configs at full B, K (C4 is the bench launch configuration) on large trees: NN checked on
    sampled queries (oracle one by one), children of those queries checked exactly -- validity, and under a
    finite c_best the prune and goal bits too; the insert is checked over ALL children (bit-exact copy_if)."""
    p, cfg = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, n0, seed=77, flat=True)
    B, K = B or cfg.B, cfg.K
    edge = float(np.float32(p.steps_per_edge) * np.float32(p.dt))
    # every node of the flat tree costs one edge: children cost two; a bound at 2 edges + the median heuristic of
    # the box prunes roughly half of them
    c_best = float("inf")
    if finite:
        rs = np.random.default_rng(5)
        lo, hi = p.state_lo[:p.pos_dim].astype(np.float64), p.state_hi[:p.pos_dim].astype(np.float64)
        hs = [op.heuristic(np.r_[rs.uniform(lo, hi), np.zeros(p.state_dim - p.pos_dim)]) for _ in range(400)]
        c_best = 2 * edge + float(np.median(hs))
    tree = pl.new_tree(n0 + B * K, host)
    out = pl.expand_step(tree, 0, 0, 40, B, K, c_best=c_best)
    tree64 = host["states"].astype(np.float64)
    rng = np.random.default_rng(1)
    n_pruned = 0
    for s in rng.choice(B, min(24, B), replace=False):
        q = op.sample_state(0, 0, 40, int(s))
        np.testing.assert_array_equal(out["x_rand"][s].astype(np.float64), q)
        i, d2 = op.nearest(tree64, q)
        if out["nn_idx"][s] != i:
            assert op.dist2(q, tree64[out["nn_idx"][s]]) <= (1 + 1e-6) * d2
        for k in (0, K - 1):
            c = s * K + k
            u = op.sample_control(0, 0, 40, int(s), k)
            np.testing.assert_array_equal(out["child_ctrl"][c].astype(np.float64), u)
            x, fl, fb, mm, ec = op.propagate(tree64[out["nn_idx"][s]], u)
            gf = int(out["child_flags"][c])
            if mm > 1e-5:
                assert (gf & 1) == (fl & 1)
            if fl & 1 and gf & 1:
                err = np.abs(out["child_state"][c] - x)
                ang = p.dim_kind == 1
                err[ang] = np.minimum(err[ang], 2 * np.pi - err[ang])
                assert err.max() < 1e-4
                # Alg. 1 l.11 and l.14 on this child (the flat tree's nodes all cost one edge)
                g = float(host["costs"][out["nn_idx"][s]]) + ec
                assert out["child_cost"][c] == pytest.approx(g, rel=1e-6)
                f = g + op.heuristic(x)
                notpruned = f < c_best
                if abs(f - c_best) > 1e-5:
                    assert bool(gf & 8) == notpruned
                    n_pruned += not notpruned
                    ing, gm = op.in_goal(x)
                    if gm > 1e-5:
                        assert bool(gf & 16) == (notpruned and ing)
    if finite:
        assert n_pruned > 0 and 0.05 < float(((out["child_flags"] & 8) != 0).mean()) < 0.95
    # properties that hold at any size
    assert out["nn_idx"].min() >= 0 and out["nn_idx"].max() < n0
    keep = np.nonzero((out["child_flags"] & 9) == 9)[0]
    n1 = int(tree["n_nodes"][0].item())
    assert out["n_inserted"] == len(keep) == n1 - n0
    # insert order over ALL children: bit-exact copy_if of the kept children, in child order (P20)
    D, m = p.state_dim, p.control_dim
    np.testing.assert_array_equal(tree["states"][n0:n1, :D].cpu().numpy(), out["child_state"][keep])
    np.testing.assert_array_equal(tree["actions"][n0:n1, :m].cpu().numpy(), out["child_ctrl"][keep])
    np.testing.assert_array_equal(tree["costs"][n0:n1].cpu().numpy(), out["child_cost"][keep])
    np.testing.assert_array_equal(tree["parents"][n0:n1].cpu().numpy(), out["nn_idx"][keep // K])
    np.testing.assert_array_equal(np.nonzero((out["child_flags"] & 32) != 0)[0], keep)
    g = keep[(out["child_flags"][keep] & 16) != 0]
    if len(g):
        best = g[np.argmin(out["child_cost"][g])]
        assert out["goal_node"] == n0 + int(np.nonzero(keep == best)[0][0])
    else:
        assert out["goal_node"] == -1
    pl.close()


@pytest.mark.parametrize("name,n0,B,K", [("C2", 5000, 8, 4), ("C2", 70001, 16, 2), ("C3", 33, 5, 3),
                                         ("C4", 9000, 8, 16), ("C1", 1, 3, 2), ("C4", 40000, 13, 1)])
def test_step_streaming_tier_matches_oracle(pakr, orc, name, n0, B, K):
    """B <= 16 takes the HBM-bound streaming NN tier (one row per lane): same parity bar."""
    from parity_util import check_iteration, run_both
    p, _ = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    host = wl.random_tree(p, n0, seed=n0 + B, flat=n0 > 20000)
    cap = n0 + B * K
    out, after, ref, _ = run_both(pl, orc, op, p, host, seed=4, r=1, it=2, B=B, K=K, cap=cap)
    check_iteration(orc, op, p, host, out, after, ref, B, K, cap)
    pl.close()


@pytest.mark.parametrize("name", ["C2", "C3", "C4"])
def test_nn_tiers_agree_bit_for_bit(pakr, name):
    """The tiers have no observable semantics (P26): query s is the same Philox draw whatever B is,
    so the streaming tier (B = 16) and the tiled tier (B = 48) must return identical NN indices and d2."""
    p, _ = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    n0 = 50000
    host = wl.random_tree(p, n0, seed=12, flat=True)
    host["states"][25000:] = host["states"][:25000]  # every node twice: lowest index must win in both tiers
    outs = []
    for B in (16, 48):
        tree = pl.new_tree(n0 + B, host)
        outs.append(pl.expand_step(tree, 9, 0, 3, B, 1))
    np.testing.assert_array_equal(outs[0]["x_rand"], outs[1]["x_rand"][:16])
    np.testing.assert_array_equal(outs[0]["nn_idx"], outs[1]["nn_idx"][:16])
    np.testing.assert_array_equal(outs[0]["nn_d2"], outs[1]["nn_d2"][:16])
    assert outs[0]["nn_idx"].max() < 25000
    pl.close()


@pytest.mark.parametrize("name,n0,B,K", [("C2", 20000, 512, 2), ("C3", 9000, 300, 3), ("C3", 40000, 257, 2),
                                         ("C1", 700, 64, 4), ("C5", 60000, 1024, 1), ("C4", 30000, 512, 2),
                                         ("C4", 1025, 300, 1), ("N1", 5000, 256, 2), ("N2", 33000, 400, 2),
                                         ("N3", 70000, 256, 1), ("C2", 300000, 2048, 1), ("N4", 9000, 300, 2)])
def test_nn_index_tier_equals_scan_tier(pakr, orc, name, n0, B, K):
    """The NN index (exact spatial pruning) must return bit-identical NN indices
    and distances to the brute-force scan, on clustered trees too (queries far from every node search wide),
    and meets the oracle bar.  nn_mode: PAKR_NN_SCAN = scan tiers only, PAKR_NN_INDEX = index on any tree."""
    from parity_util import check_iteration, run_both
    p, _ = wl.CONFIGS[name]()
    host = wl.random_tree(p, n0, seed=n0, flat=n0 > 30000)
    # squeeze most positions into a corner blob, as a pruned AO-x tree is, and duplicate a few rows (ties)
    pd = p.pos_dim
    host["states"][n0 // 3:, :pd] = (p.state_lo[:pd] + 0.15 * (host["states"][n0 // 3:, :pd] - p.state_lo[:pd]))
    host["states"][n0 - 50:] = host["states"][100:150]
    outs = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_INDEX):
        tree = pl.new_tree(n0 + B * K, host)
        outs[mode] = pl.expand_step(tree, 5, 1, 4, B, K, nn_mode=mode)
        if mode == pakr.NN_INDEX:
            op = orc.OracleProblem(p)
            out, after, ref, _ = run_both(pl, orc, op, p, host, seed=5, r=1, it=4, B=B, K=K, cap=n0 + B * K,
                                          nn_mode=mode)
            check_iteration(orc, op, p, host, out, after, ref, B, K, n0 + B * K)
    pl.close()
    for k in ("x_rand", "nn_idx", "nn_d2", "child_state"):
        np.testing.assert_array_equal(outs[pakr.NN_SCAN][k], outs[pakr.NN_INDEX][k])


@pytest.mark.parametrize("name,n0,B,K,clustered", [
    ("C2", 70000, 1024, 2, False), ("C2", 300000, 2048, 1, True), ("C5", 1 << 20, 512, 1, False),
    ("C4", 60000, 4096, 1, False), ("C4", 200000, 1024, 2, True), ("N3", 90000, 2048, 1, False),
    ("C3", 150000, 2048, 1, False), ("C3", 150000, 2048, 1, True),      # heading weight 1: the cosine bound is loose
    ("N4", 120000, 1024, 1, False), ("N1", 200000, 1024, 1, True), ("N2", 200000, 1024, 1, False),
    ("C1", 65000, 2048, 1, True), ("C2", 4096, 20000, 1, False)])
def test_nn_filter_tier_equals_scan_tier(pakr, orc, name, n0, B, K, clustered):
    """The tensor-core coarse filter (pakr_nn_filter.cuh: fp16 hi/lo mma, fp32 accumulate, exact rescoring of the
    candidate chunks) must return bit-identical NN indices and distances to the brute-force fp32 scan -- on uniform
    trees, on trees squeezed into a corner with duplicated rows (many rows inside the rounding band: ties, lowest index
    wins) -- and meets the oracle bar on sampled queries.  Problems with heavy angle weights (C3, N1, N2, N4) silently
    keep the fp32 scan under PAKR_NN_FILTER; B = 20000 on a 4096-node tree is the shape that exposed an out-of-range
    shared-memory read of idle warps in the scan's last round."""
    p, _ = wl.CONFIGS[name]()
    host = wl.random_tree(p, n0, seed=n0 % 977, flat=True)
    if clustered:
        pd = p.pos_dim
        host["states"][n0 // 3:, :pd] = (p.state_lo[:pd] + 0.05 * (host["states"][n0 // 3:, :pd] - p.state_lo[:pd]))
        host["states"][n0 - 3000:] = host["states"][100:3100]       # exact duplicates, far apart in index
        host["states"][n0 // 2:n0 // 2 + 3000] = host["states"][100:3100] + np.float32(1e-4)  # near-duplicates inside the band
    outs = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_FILTER):
        tree = pl.new_tree(n0 + B * K, host)
        outs[mode] = pl.expand_step(tree, 5, 1, 4, B, K, nn_mode=mode)
        st = pl.read_stats(B, K, n0 + B * K)
        heavy_angles = float(p.nn_weight[p.dim_kind == 1].sum()) > 0.1   # those problems keep the fp32 scan
        if mode == pakr.NN_FILTER and B * n0 * p.state_dim >= 4e8 and not heavy_angles:
            assert st["nn_pairs_filtered"] == B * n0, "the filter did not run"
    pl.close()
    for k in ("x_rand", "nn_idx", "nn_d2", "child_state", "child_flags"):
        np.testing.assert_array_equal(outs[pakr.NN_SCAN][k], outs[pakr.NN_FILTER][k])
    op = orc.OracleProblem(p)
    tree64 = host["states"].astype(np.float64)
    rng = np.random.default_rng(2)
    for s_ in rng.choice(B, 12, replace=False):
        q = op.sample_state(5, 1, 4, int(s_))
        i, d2 = op.nearest(tree64, q)
        j = int(outs[pakr.NN_FILTER]["nn_idx"][s_])
        assert j == i or op.dist2(q, tree64[j]) <= (1 + 1e-6) * d2


@pytest.mark.parametrize("half_width", [0.02, 0.005])
def test_nn_filter_tier_equals_scan_tier_on_a_tiny_state_box(pakr, half_width):
    """A state box much narrower than 1 in weighted units puts every filter feature in the fp16 subnormal range of its
    lo half, where the hi/lo split is only good to an absolute 2^-25: the relative rounding band alone would then drop
    the chunk of the true nearest row.  With the absolute floor in the band the filter tier must still equal the scan
    bit for bit (and must really have run)."""
    p, _ = wl.config2()
    D = p.state_dim
    centre = np.full(D, 0.3, np.float32)
    lo, hi = centre - np.float32(half_width), centre + np.float32(half_width)
    p = dataclasses.replace(p, state_lo=lo, state_hi=hi, start=centre.copy(), obstacles=p.obstacles[:0],
                            goal_center=centre[:p.pos_dim] + np.float32(0.5 * half_width),
                            goal_radius=float(0.1 * half_width), nn_weight=np.ones(D, np.float32))
    n0, B, K = 200000, 1024, 1
    host = wl.random_tree(p, n0, seed=17, flat=True)
    host["states"][n0 - 2000:] = host["states"][100:2100]   # exact duplicates: lowest index must win
    outs = {}
    pl = pakr.Planner(p)
    for mode in (pakr.NN_SCAN, pakr.NN_FILTER):
        tree = pl.new_tree(n0 + B * K, host)
        outs[mode] = pl.expand_step(tree, 5, 1, 4, B, K, nn_mode=mode)
        if mode == pakr.NN_FILTER:
            assert pl.read_stats(B, K, n0 + B * K)["nn_pairs_filtered"] == B * n0, "the filter did not run"
    pl.close()
    for k in ("x_rand", "nn_idx", "nn_d2"):
        np.testing.assert_array_equal(outs[pakr.NN_SCAN][k], outs[pakr.NN_FILTER][k])


@pytest.mark.parametrize("name", ["C3", "C4"])
def test_step_on_planner_grown_trees(pakr, orc, name):
    """SURVEY.md 8(c) "T" on the trees the planner itself grows (every batch sees the frozen snapshot the
    previous batches left), at BASELINE's B and K: (a) replan 0 cut after 6 iterations, no bound yet; (b) the tree of a
    late replan (r = 2) grown under a finite c_best -- nodes hugging the corridor the bound leaves open.  The tree is
    read back, handed to one pakr_expand_step (the library picks the NN tier as it does in the loop) and to the oracle,
    which checks sampled queries exactly: draw, nearest node, the K children re-propagated from the chosen parent."""
    from parity_util import check_sampled
    p, cfg = wl.CONFIGS[name]()
    B, K, cap = cfg.B, cfg.K, cfg.tree_capacity
    pl = pakr.Planner(p)
    op = orc.OracleProblem(p)
    c0 = pl.plan(3, B, K, cap, 1)["cost"]
    assert np.isfinite(c0)
    grown = []
    res = pl.plan(3, B, K, cap, 1, max_iters_per_replan=6)
    grown.append((res, 0, int(res["replan_iters"][0]), float("inf")))
    res = pl.plan(3, B, K, cap, 3, max_iters_per_replan=10, initial_cost_bound=c0)
    grown.append((res, 2, int(res["replan_iters"][2]), float(min(c0, res["replan_cost"][2]))))
    rng = np.random.default_rng(11)
    for res, r, it, c_best in grown:
        n = res["final_tree_nodes"]
        assert n > 20000
        host = pl.read_tree(B, K, cap, n)
        step_cap = n + B * K
        tree = pl.new_tree(step_cap, host)
        out = pl.expand_step(tree, 3, r, it, B, K, c_best=c_best)
        share = check_sampled(op, p, host, out, 3, r, it, K, c_best, rng.choice(B, 64, replace=False))
        assert share > 0.95
        # the insert is the stable compaction of the GPU's own keep flags
        keep = np.nonzero(((out["child_flags"] & 1) != 0) & ((out["child_flags"] & 8) != 0))[0]
        assert out["n_inserted"] == len(keep) == int(tree["n_nodes"][0].item()) - n
        np.testing.assert_array_equal(tree["parents"][n:n + len(keep)].cpu().numpy(), out["nn_idx"][keep // K])
        np.testing.assert_array_equal(tree["states"][n:n + len(keep), :p.state_dim].cpu().numpy(), out["child_state"][keep])
    pl.close()
