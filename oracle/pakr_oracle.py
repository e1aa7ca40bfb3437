"""ctypes wrapper of the fp64 CPU oracle (oracle/pakr_oracle.cpp) -- TEST INFRASTRUCTURE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
import this module.  It never imports the CUDA binding.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
# PAKR_ORACLE_SANITIZE=1: the same source built with AddressSanitizer + UBSan into a library of its own, for running
# the oracle's pins under a memory / undefined-behaviour checker.  The interpreter is not instrumented, so the ASan
# runtime has to be preloaded:
#   LD_PRELOAD=$(gcc -print-file-name=libasan.so) ASAN_OPTIONS=detect_leaks=0 PAKR_ORACLE_SANITIZE=1 \
#       python -m pytest tests -m "not gpu" -k oracle
_SANITIZE = os.environ.get("PAKR_ORACLE_SANITIZE", "") not in ("", "0")
_SO = os.path.join(_HERE, "libpakr_oracle_san.so" if _SANITIZE else "libpakr_oracle.so")
_SRC = [os.path.join(_HERE, "pakr_oracle.cpp"), os.path.join(_HERE, "pakr_oracle.h")]


def build(force: bool = False) -> str:
    """g++ -O2 -std=c++17, no -ffast-math, no OpenMP (BASELINE.md CPU-baseline plan)."""
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in _SRC)
    if force or stale:
        tmp = _SO + f".{os.getpid()}.tmp"
        opt = (["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"]
               if _SANITIZE else ["-O2"])
        subprocess.check_call(["g++"] + opt + ["-std=c++17", "-Wall", "-shared", "-fPIC", "-o", tmp, _SRC[0]])
        os.replace(tmp, _SO)
    return _SO


_dp = C.POINTER(C.c_double)
_ip = C.POINTER(C.c_int32)
_lp = C.POINTER(C.c_int64)
_up = C.POINTER(C.c_uint8)


class _Problem(C.Structure):
    _fields_ = [
        ("dynamics_id", C.c_int32), ("integrator", C.c_int32), ("state_dim", C.c_int32),
        ("control_dim", C.c_int32), ("pos_dim", C.c_int32),
        ("dyn_params", _dp), ("n_dyn_params", C.c_int32),
        ("state_lo", _dp), ("state_hi", _dp), ("dim_kind", _up), ("nn_weight", _dp),
        ("control_lo", _dp), ("control_hi", _dp),
        ("obstacle_type", C.c_int32), ("obstacles", _dp), ("n_obstacles", C.c_int32),
        ("start", _dp), ("goal_center", _dp), ("goal_radius", C.c_double),
        ("goal_angle_dim", C.c_int32), ("goal_angle", C.c_double), ("goal_angle_tol", C.c_double),
        ("dt", C.c_double), ("steps_per_edge", C.c_int32),
        ("cost_mode", C.c_int32), ("heuristic_speed", C.c_double),
        ("goal_n_dims", C.c_int32), ("goal_dims", _ip),
    ]


class _Tree(C.Structure):
    _fields_ = [("states", _dp), ("actions", _dp), ("parents", _ip), ("costs", _dp),
                ("capacity", C.c_int64), ("n", C.c_int64)]


class _IterDebug(C.Structure):
    _fields_ = [("x_rand", _dp), ("nn_idx", _ip), ("nn_d2", _dp), ("child_state", _dp),
                ("child_ctrl", _dp), ("child_cost", _dp), ("child_flags", _ip),
                ("child_margin", _dp), ("prune_margin", _dp), ("goal_margin", _dp),
                ("n_inserted", C.c_int64), ("goal_node", C.c_int64), ("new_c_best", C.c_double),
                ("phase_ms", C.c_double * 3)]


class _PlanOpts(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("B", C.c_int32), ("K", C.c_int32),
                ("tree_capacity", C.c_int64), ("n_replans", C.c_int32),
                ("time_budget_ms", C.c_double), ("max_iters_per_replan", C.c_int64),
                ("initial_cost_bound", C.c_double)]


class _PlanResult(C.Structure):
    _fields_ = [("path_nodes", _ip), ("path_states", _dp), ("path_controls", _dp),
                ("path_capacity", C.c_int32), ("path_len", C.c_int32),
                ("cost", C.c_double), ("outcome", C.c_int32),
                ("iterations", C.c_int64), ("children", C.c_int64), ("inserted", C.c_int64),
                ("replans_run", C.c_int32), ("replans_solved", C.c_int32),
                ("first_solution_ms", C.c_double), ("total_ms", C.c_double),
                ("replan_cost", _dp), ("replan_nodes", _lp), ("replan_iters", _lp), ("phase_ms", C.c_double * 3)]


F_VALID, F_INBOUNDS, F_COLLFREE, F_NOTPRUNED, F_GOAL, F_INSERTED = 1, 2, 4, 8, 16, 32

_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.orc_uniform_f32.restype = C.c_float
        L.orc_uniform_f32.argtypes = [C.c_uint32, C.c_float, C.c_float]
        L.orc_draw_word.restype = C.c_uint32
        L.orc_draw_word.argtypes = [C.c_uint64] + [C.c_uint32] * 6
        L.orc_wrap_pi.restype = C.c_double
        L.orc_wrap_pi.argtypes = [C.c_double]
        L.orc_dist2.restype = C.c_double
        L.orc_nearest.restype = C.c_int64
        L.orc_nearest.argtypes = [C.c_void_p, _dp, C.c_int64, _dp, _dp]
        L.orc_obstacle_margin.restype = C.c_double
        L.orc_bounds_margin.restype = C.c_double
        L.orc_heuristic.restype = C.c_double
        L.orc_propagate.restype = C.c_int32
        L.orc_in_goal.restype = C.c_int32
        L.orc_expand_iteration.restype = C.c_int32
        L.orc_expand_iteration.argtypes = [C.c_void_p, C.c_void_p, C.c_uint64, C.c_uint32,
                                           C.c_uint32, C.c_int32, C.c_int32, C.c_double, C.c_void_p]
        L.orc_plan.restype = C.c_int32
        L.orc_validate_plan.restype = C.c_int32
        _lib = L
    return _lib


def _d(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float64))


def _ptr(a: np.ndarray, t=_dp):
    return a.ctypes.data_as(t)


class OracleProblem:
    """Widens a workloads.Problem (fp32 arrays) to the oracle's fp64 struct and keeps it alive."""

    def __init__(self, p):
        self.p = p
        self.D, self.m, self.pos_dim = p.state_dim, p.control_dim, p.pos_dim
        f32 = lambda v: float(np.float32(v))  # scalars reach the GPU as fp32: widen the same value
        self._keep = dict(
            dyn=_d(p.dyn_params if len(p.dyn_params) else [0.0]), lo=_d(p.state_lo), hi=_d(p.state_hi),
            kind=np.ascontiguousarray(p.dim_kind, dtype=np.uint8), w=_d(p.nn_weight),
            ulo=_d(p.control_lo), uhi=_d(p.control_hi),
            obs=_d(p.obstacles.reshape(-1) if p.n_obstacles else [0.0]), start=_d(p.start),
            goal=_d(p.goal_center),
            gdims=np.ascontiguousarray(p.goal_dims if p.goal_dims is not None else [0], dtype=np.int32))
        k = self._keep
        self.c = _Problem(
            p.dynamics_id, p.integrator, p.state_dim, p.control_dim, p.pos_dim,
            _ptr(k["dyn"]), len(p.dyn_params), _ptr(k["lo"]), _ptr(k["hi"]), _ptr(k["kind"], _up),
            _ptr(k["w"]), _ptr(k["ulo"]), _ptr(k["uhi"]), p.obstacle_type, _ptr(k["obs"]),
            p.n_obstacles, _ptr(k["start"]), _ptr(k["goal"]), f32(p.goal_radius), p.goal_angle_dim,
            f32(p.goal_angle), f32(p.goal_angle_tol), f32(p.dt), p.steps_per_edge, p.cost_mode,
            f32(p.heuristic_speed), 0 if p.goal_dims is None else len(p.goal_dims), _ptr(k["gdims"], _ip))
        self.ref = C.byref(self.c)

    # ---- building blocks ----
    def sample_state(self, seed, r, it, s) -> np.ndarray:
        x = np.zeros(self.D)
        lib().orc_sample_state(self.ref, C.c_uint64(seed), C.c_uint32(r), C.c_uint32(it), C.c_uint32(s), _ptr(x))
        return x

    def sample_control(self, seed, r, it, s, k) -> np.ndarray:
        u = np.zeros(self.m)
        lib().orc_sample_control(self.ref, C.c_uint64(seed), C.c_uint32(r), C.c_uint32(it), C.c_uint32(s),
                                 C.c_uint32(k), _ptr(u))
        return u

    def dist2(self, a, b) -> float:
        a, b = _d(a), _d(b)
        return lib().orc_dist2(self.ref, _ptr(a), _ptr(b))

    def nearest(self, states, q):
        states, q = _d(states), _d(q)
        d2 = C.c_double()
        i = lib().orc_nearest(self.ref, _ptr(states), states.shape[0], _ptr(q), C.byref(d2))
        return int(i), d2.value

    def f(self, x, u) -> np.ndarray:
        x, u = _d(x), _d(u)
        out = np.zeros(self.D)
        lib().orc_f(self.ref, _ptr(x), _ptr(u), _ptr(out))
        return out

    def step(self, x, u) -> np.ndarray:
        x, u = _d(x), _d(u)
        out = np.zeros(self.D)
        lib().orc_step(self.ref, _ptr(x), _ptr(u), _ptr(out))
        return out

    def obstacle_margin(self, x) -> float:
        x = _d(x)
        return lib().orc_obstacle_margin(self.ref, _ptr(x))

    def bounds_margin(self, x) -> float:
        x = _d(x)
        return lib().orc_bounds_margin(self.ref, _ptr(x))

    def propagate(self, x0, u):
        """-> (x_new, flags, first_bad_step, min_margin, edge_cost)"""
        x0, u = _d(x0), _d(u)
        out = np.zeros(self.D)
        fb, mm, ec = C.c_int32(), C.c_double(), C.c_double()
        fl = lib().orc_propagate(self.ref, _ptr(x0), _ptr(u), _ptr(out), C.byref(fb), C.byref(mm), C.byref(ec))
        return out, int(fl), fb.value, mm.value, ec.value

    def heuristic(self, x) -> float:
        x = _d(x)
        return lib().orc_heuristic(self.ref, _ptr(x))

    def in_goal(self, x):
        x = _d(x)
        mg = C.c_double()
        r = lib().orc_in_goal(self.ref, _ptr(x), C.byref(mg))
        return bool(r), mg.value

    def validate_plan(self, path_states, path_controls, per_edge: bool = False):
        """-> (code, cost, max_state_err); code 0 = valid and in goal."""
        ps, pc = _d(path_states), _d(path_controls)
        cost, err = C.c_double(), C.c_double()
        code = lib().orc_validate_plan(self.ref, _ptr(ps), _ptr(pc), C.c_int32(ps.shape[0]),
                                       C.c_int32(1 if per_edge else 0), C.byref(cost), C.byref(err))
        return int(code), cost.value, err.value


class OracleTree:
    def __init__(self, op: OracleProblem, capacity: int):
        self.op = op
        self.capacity = int(capacity)
        self.states = np.zeros((self.capacity, op.D))
        self.actions = np.zeros((self.capacity, op.m))
        self.parents = np.zeros(self.capacity, np.int32)
        self.costs = np.zeros(self.capacity)
        self.c = _Tree(_ptr(self.states), _ptr(self.actions), _ptr(self.parents, _ip), _ptr(self.costs),
                       self.capacity, 0)
        self.ref = C.byref(self.c)
        self.reset()

    @property
    def n(self) -> int:
        return int(self.c.n)

    def reset(self):
        lib().orc_tree_reset(self.op.ref, self.ref)

    def load(self, states, actions, parents, costs):
        """Teacher forcing: overwrite the first n nodes with a (widened) snapshot."""
        n = len(parents)
        assert n <= self.capacity
        self.states[:n] = np.asarray(states, dtype=np.float64)[:, :self.op.D]
        self.actions[:n] = np.asarray(actions, dtype=np.float64)[:, :self.op.m]
        self.parents[:n] = parents
        self.costs[:n] = costs
        self.c.n = n


def expand_iteration(op: OracleProblem, tree: OracleTree, seed: int, r: int, it: int, B: int, K: int,
                     c_best: float = float("inf")) -> dict:
    """One trip of Alg. 1 l.6-17 with every debug output."""
    D, m, BK = op.D, op.m, B * K
    out = dict(x_rand=np.zeros((B, D)), nn_idx=np.zeros(B, np.int32), nn_d2=np.zeros(B),
               child_state=np.zeros((BK, D)), child_ctrl=np.zeros((BK, m)), child_cost=np.zeros(BK),
               child_flags=np.zeros(BK, np.int32), child_margin=np.zeros(BK), prune_margin=np.zeros(BK),
               goal_margin=np.zeros(BK))
    dbg = _IterDebug(_ptr(out["x_rand"]), _ptr(out["nn_idx"], _ip), _ptr(out["nn_d2"]),
                     _ptr(out["child_state"]), _ptr(out["child_ctrl"]), _ptr(out["child_cost"]),
                     _ptr(out["child_flags"], _ip), _ptr(out["child_margin"]), _ptr(out["prune_margin"]),
                     _ptr(out["goal_margin"]), 0, -1, 0.0, (C.c_double * 3)())
    goal = lib().orc_expand_iteration(op.ref, tree.ref, C.c_uint64(seed), C.c_uint32(r), C.c_uint32(it),
                                      C.c_int32(B), C.c_int32(K), C.c_double(c_best), C.byref(dbg))
    out.update(goal=bool(goal), n_inserted=int(dbg.n_inserted), goal_node=int(dbg.goal_node),
               new_c_best=float(dbg.new_c_best), phase_ms=[float(v) for v in dbg.phase_ms])  # NN / propagate / insert
    return out


def plan(op: OracleProblem, seed: int, B: int, K: int, tree_capacity: int, n_replans: int,
         time_budget_ms: float = 0.0, max_iters_per_replan: int = 0, path_capacity: int = 4096,
         tree: Optional[OracleTree] = None, initial_cost_bound: float = 0.0) -> dict:
    """Alg. 1 l.1-18.  Returns the path (nodes, states, controls), cost, stats and the final tree."""
    tree = tree or OracleTree(op, tree_capacity)
    nodes = np.zeros(path_capacity, np.int32)
    states = np.zeros((path_capacity, op.D))
    ctrls = np.zeros((path_capacity, op.m))
    rc = np.full(n_replans, np.inf)
    rn = np.zeros(n_replans, np.int64)
    ri = np.zeros(n_replans, np.int64)
    opts = _PlanOpts(seed, B, K, tree_capacity, n_replans, time_budget_ms, max_iters_per_replan, initial_cost_bound)
    res = _PlanResult(_ptr(nodes, _ip), _ptr(states), _ptr(ctrls), path_capacity, 0, 0.0, 0, 0, 0, 0, 0, 0,
                      0.0, 0.0, _ptr(rc), _ptr(rn, _lp), _ptr(ri, _lp), (C.c_double * 3)())
    status = lib().orc_plan(op.ref, C.byref(opts), tree.ref, C.byref(res))
    L = res.path_len if status == 0 else 0
    return dict(status=status, outcome=int(res.outcome), cost=float(res.cost), path_len=int(res.path_len),
                path_nodes=nodes[:L].copy(), path_states=states[:L].copy(),
                path_controls=ctrls[:max(L - 1, 0)].copy(), iterations=int(res.iterations),
                children=int(res.children), inserted=int(res.inserted), replans_run=int(res.replans_run),
                replans_solved=int(res.replans_solved), first_solution_ms=float(res.first_solution_ms),
                total_ms=float(res.total_ms), replan_cost=rc, replan_nodes=rn, replan_iters=ri, tree=tree,
                phase_ms=[float(v) for v in res.phase_ms])


def philox4x32_10(ctr, key) -> np.ndarray:
    c = (C.c_uint32 * 4)(*[int(v) & 0xFFFFFFFF for v in ctr])
    k = (C.c_uint32 * 2)(*[int(v) & 0xFFFFFFFF for v in key])
    o = (C.c_uint32 * 4)()
    lib().orc_philox4x32_10(c, k, o)
    return np.array(list(o), dtype=np.uint32)


def uniform_f32(word: int, lo: float, hi: float) -> float:
    return float(lib().orc_uniform_f32(C.c_uint32(word), C.c_float(lo), C.c_float(hi)))


def draw_word(seed, it, r, s, kind, k, j) -> int:
    return int(lib().orc_draw_word(C.c_uint64(seed), it, r, s, kind, k, j))


def wrap_pi(a: float) -> float:
    return float(lib().orc_wrap_pi(C.c_double(a)))
