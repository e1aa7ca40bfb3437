"""pakr_expand_step_static: the iteration for callers that cannot hand over (or allocate) a device workspace.

A planner inside a control loop with a deadline reserves its memory at start-up and may not call cudaMalloc while it
runs (the call can stall the device for an unbounded time); a plug-in inside a host whose pool owns the GPU has no
allocator to ask.  For them the library carries one fixed scratch array per GPU inside its own image and offers an
entry point that allocates nothing.  The array is shared by every call in the process and keeps the bytes of the
previous call, so the property to check is: the same inputs give the same outputs as the workspace path
(pakr_expand_step, PAKR_NN_SCAN), bit for bit -- the tolerance the tier-equality tests of test_gpu_step.py use -- on
the first call AND on calls that follow it with other shapes, whatever ran in the process before.

This file sorts last on purpose (pytest -x stops at the first failure; nothing is hidden behind this one) and must
pass both on its own in a fresh process and after the rest of the suite.
"""
import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl

pytestmark = pytest.mark.gpu

_KEYS = ("x_rand", "nn_idx", "nn_d2", "child_state", "child_ctrl", "child_cost", "child_flags")
_SCALARS = ("n_inserted", "goal_node", "new_c_best")


@pytest.fixture(scope="module")
def pakr():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2607_03987_b200 import pakr as mod
    mod.lib()  # fails loudly if the extension is missing
    return mod


def _tree_np(pl, tree):
    n = int(tree["n_nodes"][0].item())
    return dict(n=n, states=tree["states"][:n].cpu().numpy(), actions=tree["actions"][:n].cpu().numpy(),
                parents=tree["parents"][:n].cpu().numpy(), costs=tree["costs"][:n].cpu().numpy())


def _same(a, b):
    for k in _KEYS:
        np.testing.assert_array_equal(a[k], b[k], err_msg=k)
    for k in _SCALARS:
        assert a[k] == b[k] or (np.isinf(a[k]) and np.isinf(b[k])), (k, a[k], b[k])


@pytest.mark.parametrize("name,n0,shapes", [
    # two or three calls in a row on a growing tree; the later ones use other (B, K), so they find the array full of
    # another shape's leftovers.  B = 8 is below the streaming tier's threshold of the workspace path (16 queries).
    ("C1", 1500, [(256, 4), (100, 3), (256, 4)]),
    ("C2", 6000, [(1024, 16), (8, 5), (300, 7)]),        # first call at the limit B*K = 16384
    ("C4", 5000, [(512, 16), (1024, 16), (33, 1)]),      # 12-D rows: the widest scratch rows
    ("N4", 3000, [(300, 5), (300, 5)]),
])
def test_static_scratch_step_equals_workspace_step(pakr, name, n0, shapes):
    p, _ = wl.CONFIGS[name]()
    pl = pakr.Planner(p)
    host = wl.random_tree(p, n0, seed=n0 + 7)
    cap = n0 + sum(B * K for B, K in shapes)
    ref_tree = pl.new_tree(cap, host)   # grown by the existing path (caller workspace)
    sta_tree = pl.new_tree(cap, host)   # grown by the no-allocation path
    c_best = float("inf")
    for it, (B, K) in enumerate(shapes):
        ref = pl.expand_step(ref_tree, 5, 1, it, B, K, c_best=c_best, nn_mode=pakr.NN_SCAN)
        sta = pl.expand_step_static(sta_tree, 5, 1, it, B, K, c_best=c_best)
        _same(sta, ref)
        a, b = _tree_np(pl, sta_tree), _tree_np(pl, ref_tree)
        assert a["n"] == b["n"] and a["n"] > n0
        for k in ("states", "actions", "parents", "costs"):
            np.testing.assert_array_equal(a[k], b[k], err_msg=k)
        if np.isfinite(ref["new_c_best"]):
            c_best = ref["new_c_best"]  # a goal child turned up: the next call prunes against it on both sides
    pl.close()


def test_static_scratch_is_shared_between_planners(pakr):
    """Two planners of different models take turns on the one array; each call still equals its workspace twin."""
    pa, _ = wl.config1()
    pb, _ = wl.config4()
    pls = [pakr.Planner(pa), pakr.Planner(pb)]
    hosts = [wl.random_tree(pa, 2000, seed=1), wl.random_tree(pb, 2000, seed=2)]
    for rnd in range(2):
        for pl, host, (B, K) in zip(pls, hosts, [(256, 4), (384, 16)]):
            cap = 2000 + B * K
            ref = pl.expand_step(pl.new_tree(cap, host), 9, 0, rnd, B, K, nn_mode=pakr.NN_SCAN)
            sta = pl.expand_step_static(pl.new_tree(cap, host), 9, 0, rnd, B, K)
            _same(sta, ref)
    for pl in pls:
        pl.close()


def test_static_scratch_rejects_what_does_not_fit(pakr):
    """Beyond the stated maximum the call says so and launches nothing (the tree is untouched)."""
    p, _ = wl.config2()
    pl = pakr.Planner(p)
    host = wl.random_tree(p, 500, seed=3)
    tree = pl.new_tree(500 + 40000, host)
    before = _tree_np(pl, tree)
    assert 1025 * 16 > pakr.STATIC_MAX_CHILDREN
    with pytest.raises(pakr.PakrError) as e:
        pl.expand_step_static(tree, 1, 0, 0, 1025, 16)
    assert e.value.status == 1 and "exceeds the static scratch" in str(e.value)
    with pytest.raises(pakr.PakrError) as e:
        pl.expand_step_static(tree, 1, 0, 0, 256, 4, nn_mode=pakr.NN_INDEX)  # tiers with per-node copies: not here
    assert e.value.status == 2
    after = _tree_np(pl, tree)
    assert after["n"] == before["n"] == 500
    np.testing.assert_array_equal(after["states"], before["states"])
    # and the limit itself is accepted
    out = pl.expand_step_static(tree, 1, 0, 0, 1024, 16)
    assert out["n_inserted"] > 0
    pl.close()
