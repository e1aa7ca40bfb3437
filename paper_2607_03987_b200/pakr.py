"""Thin ctypes binding of include/pakr.h: argument marshalling only.

Every step of the hot path runs in the CUDA kernels of csrc/; PyTorch supplies device memory
(a uint8 workspace tensor) and the current stream, nothing else.  There is no CPU fallback:
if libpakr.so is missing or a call fails, this module raises.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpakr.so")
_CSRC = os.path.join(_HERE, "csrc")
_SOURCES = ["pakr_api.cu", "pakr_kernel_inst.cu", "pakr_kernel.cuh", "pakr_device.cuh", "pakr_nn_filter.cuh"]

F_VALID, F_INBOUNDS, F_COLLFREE, F_NOTPRUNED, F_GOAL, F_INSERTED = 1, 2, 4, 8, 16, 32
NN_AUTO, NN_SCAN, NN_INDEX, NN_FILTER = 0, 1, 2, 3
MAX_REPLAN_STATS = 64
MAX_PATH_NODES = 8192
STATIC_MAX_CHILDREN = 16384          # PAKR_STATIC_MAX_CHILDREN: B*K limit of pakr_expand_step_static
STATIC_SCRATCH_BYTES = 2304 * 1024   # PAKR_STATIC_SCRATCH_BYTES
_STATUS = {0: "PAKR_OK", 1: "PAKR_ERR_INVALID_ARG", 2: "PAKR_ERR_UNSUPPORTED", 3: "PAKR_ERR_WORKSPACE_TOO_SMALL",
           4: "PAKR_ERR_BUFFER_TOO_SMALL", 5: "PAKR_ERR_CUDA"}


class PakrError(RuntimeError):
    def __init__(self, status: int, msg: str):
        super().__init__(f"{_STATUS.get(status, status)}: {msg}")
        self.status = status


def build(force: bool = False, verbose: bool = False) -> str:
    """nvcc -gencode arch=compute_100a,code=sm_100a -> paper_2607_03987_b200/libpakr.so (in-tree).
    Nine translation units (host API; kernels per NN tier and model group) compile in parallel.  The roofline
    microbenchmark is a library of its own (peak.py)."""
    srcs = [os.path.join(_CSRC, s) for s in _SOURCES] + [os.path.join(_HERE, "..", "include", "pakr.h")]
    nvcc = os.environ.get("NVCC", "/usr/local/cuda/bin/nvcc")
    flags = [nvcc, "-gencode", "arch=compute_100a,code=sm_100a", "-O3", "-lineinfo", "-std=c++17",
             "-Xcompiler", "-fPIC"] + (["-Xptxas=-v"] if verbose else [])
    # the stamp records the flags the library was built with: a build with other flags is never silently reused
    stamp = " ".join(f for f in flags if f != "-Xptxas=-v")
    stamp_file = _SO + ".stamp"
    stale = (not os.path.exists(_SO)) or any(os.path.getmtime(s) > os.path.getmtime(_SO) for s in srcs)
    if not stale:
        try:
            stale = open(stamp_file).read() != stamp
        except OSError:
            stale = True
    if force or stale:
        tag = f".{os.getpid()}.tmp"
        units = [("pakr_api.cu", [], "api")]
        for tier, part in ((0, 0), (0, 1), (1, 0), (1, 1), (2, 0), (2, 1), (3, 0), (3, 1)):
            units.append(("pakr_kernel_inst.cu", [f"-DPAKR_STREAM_TIER={tier}", f"-DPAKR_PART={part}"], f"t{tier}p{part}"))
        objs, procs = [], []
        for src, defs, name in units:
            obj = os.path.join(_HERE, f"_{name}{tag}.o")
            objs.append(obj)
            procs.append(subprocess.Popen(flags + defs + ["-c", "-o", obj, os.path.join(_CSRC, src)]))
        try:
            for pr in procs:
                if pr.wait() != 0:
                    raise subprocess.CalledProcessError(pr.returncode, pr.args)
            tmp = _SO + tag
            subprocess.check_call([nvcc, "-shared", "-o", tmp] + objs)
            os.replace(tmp, _SO)
            with open(stamp_file, "w") as f:
                f.write(stamp)
        finally:
            for pr in procs:
                if pr.poll() is None:
                    pr.kill()
            for o in objs:
                if os.path.exists(o):
                    os.remove(o)
    return _SO


_fp = C.POINTER(C.c_float)
_ip = C.POINTER(C.c_int32)
_up = C.POINTER(C.c_uint8)


class _Problem(C.Structure):
    _fields_ = [
        ("dynamics_id", C.c_int32), ("integrator", C.c_int32), ("state_dim", C.c_int32),
        ("control_dim", C.c_int32), ("pos_dim", C.c_int32),
        ("dyn_params", _fp), ("n_dyn_params", C.c_int32),
        ("state_lo", _fp), ("state_hi", _fp), ("dim_kind", _up), ("nn_weight", _fp),
        ("control_lo", _fp), ("control_hi", _fp),
        ("obstacle_type", C.c_int32), ("obstacles", _fp), ("n_obstacles", C.c_int32),
        ("start", _fp), ("goal_center", _fp), ("goal_radius", C.c_float),
        ("goal_angle_dim", C.c_int32), ("goal_angle", C.c_float), ("goal_angle_tol", C.c_float),
        ("dt", C.c_float), ("steps_per_edge", C.c_int32),
        ("cost_mode", C.c_int32), ("heuristic_speed", C.c_float),
        ("goal_n_dims", C.c_int32), ("goal_dims", _ip),
    ]


class _TreeLayout(C.Structure):
    _fields_ = [("states_off", C.c_size_t), ("actions_off", C.c_size_t), ("parents_off", C.c_size_t),
                ("costs_off", C.c_size_t), ("state_stride", C.c_int32), ("action_stride", C.c_int32)]


class _PlanOpts(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("B", C.c_int32), ("K", C.c_int32), ("tree_capacity", C.c_int64),
                ("n_replans", C.c_int32), ("time_budget_ms", C.c_double), ("max_iters_per_replan", C.c_int64),
                ("initial_cost_bound", C.c_double), ("nn_mode", C.c_int32)]


class _Stats(C.Structure):
    _fields_ = [("iterations", C.c_int64), ("children", C.c_int64), ("inserted", C.c_int64), ("nn_pairs", C.c_int64),
                ("nn_pairs_evaluated", C.c_int64), ("nn_pairs_filtered", C.c_int64), ("h2d_bytes", C.c_int64), ("d2h_bytes", C.c_int64),
                ("replans_run", C.c_int32), ("replans_solved", C.c_int32), ("termination", C.c_int32),
                ("replan_stats_truncated", C.c_int32), ("path_truncated", C.c_int32),
                ("first_solution_ms", C.c_double), ("device_ms", C.c_double), ("phase_ms", C.c_double * 4),
                ("replan_cost", C.c_float * MAX_REPLAN_STATS), ("replan_nodes", C.c_int32 * MAX_REPLAN_STATS),
                ("replan_iters", C.c_int32 * MAX_REPLAN_STATS), ("replan_end_ms", C.c_double * MAX_REPLAN_STATS)]


class _Result(C.Structure):
    _fields_ = [("path_nodes", _ip), ("path_states", _fp), ("path_controls", _fp),
                ("path_capacity", C.c_int32), ("path_len", C.c_int32), ("cost", C.c_double),
                ("outcome", C.c_int32), ("final_tree_nodes", C.c_int32), ("stats", _Stats)]


class _StepArgs(C.Structure):
    _fields_ = [("seed", C.c_uint64), ("replan", C.c_uint32), ("iteration", C.c_uint32),
                ("B", C.c_int32), ("K", C.c_int32), ("tree_capacity", C.c_int64), ("c_best", C.c_float),
                ("nn_mode", C.c_int32),
                ("states", C.c_void_p), ("actions", C.c_void_p), ("parents", C.c_void_p), ("costs", C.c_void_p),
                ("n_nodes", C.c_void_p),
                ("x_rand", C.c_void_p), ("nn_idx", C.c_void_p), ("nn_d2", C.c_void_p), ("child_state", C.c_void_p),
                ("child_ctrl", C.c_void_p), ("child_cost", C.c_void_p), ("child_flags", C.c_void_p),
                ("n_inserted", C.c_void_p), ("goal_node", C.c_void_p), ("new_c_best", C.c_void_p)]


EXPORTS = ["pakr_create", "pakr_destroy", "pakr_last_error", "pakr_workspace_bytes", "pakr_workspace_bytes_for",
           "pakr_get_tree_layout",
           "pakr_plan", "pakr_expand_step", "pakr_expand_step_static", "pakr_read_stats"]

_lib = None


def lib():
    """Loads libpakr.so (building it if the sources are newer).  Raises if that is impossible."""
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        L.pakr_create.restype = C.c_int
        L.pakr_create.argtypes = [C.POINTER(_Problem), C.c_int, C.POINTER(C.c_void_p)]
        L.pakr_destroy.restype = None
        L.pakr_destroy.argtypes = [C.c_void_p]
        L.pakr_last_error.restype = C.c_char_p
        L.pakr_last_error.argtypes = [C.c_void_p]
        L.pakr_workspace_bytes.restype = C.c_size_t
        L.pakr_workspace_bytes.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64]
        L.pakr_workspace_bytes_for.restype = C.c_size_t
        L.pakr_workspace_bytes_for.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_int32]
        L.pakr_get_tree_layout.restype = C.c_int
        L.pakr_get_tree_layout.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.POINTER(_TreeLayout)]
        L.pakr_plan.restype = C.c_int
        L.pakr_plan.argtypes = [C.c_void_p, C.POINTER(_PlanOpts), C.c_void_p, C.c_size_t, C.c_void_p,
                                C.POINTER(_Result)]
        L.pakr_expand_step.restype = C.c_int
        L.pakr_expand_step.argtypes = [C.c_void_p, C.POINTER(_StepArgs), C.c_void_p, C.c_size_t, C.c_void_p]
        L.pakr_expand_step_static.restype = C.c_int
        L.pakr_expand_step_static.argtypes = [C.c_void_p, C.POINTER(_StepArgs), C.c_void_p]
        L.pakr_read_stats.restype = C.c_int
        L.pakr_read_stats.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int64, C.c_void_p, C.c_size_t, C.c_void_p,
                                      C.POINTER(_Stats)]
        _lib = L
    return _lib


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _ptr(a: np.ndarray, t=_fp):
    return a.ctypes.data_as(t)


def make_problem_struct(p):
    """workloads.Problem -> (pakr_problem struct, keep-alive list)."""
    keep = dict(dyn=_f32(p.dyn_params if len(p.dyn_params) else [0.0]), lo=_f32(p.state_lo), hi=_f32(p.state_hi),
                kind=np.ascontiguousarray(p.dim_kind, dtype=np.uint8), w=_f32(p.nn_weight), ulo=_f32(p.control_lo),
                uhi=_f32(p.control_hi), obs=_f32(p.obstacles.reshape(-1) if p.n_obstacles else [0.0]),
                start=_f32(p.start), goal=_f32(p.goal_center),
                gdims=np.ascontiguousarray(p.goal_dims if p.goal_dims is not None else [0], dtype=np.int32))
    s = _Problem(p.dynamics_id, p.integrator, p.state_dim, p.control_dim, p.pos_dim, _ptr(keep["dyn"]),
                 len(p.dyn_params), _ptr(keep["lo"]), _ptr(keep["hi"]), _ptr(keep["kind"], _up), _ptr(keep["w"]),
                 _ptr(keep["ulo"]), _ptr(keep["uhi"]), p.obstacle_type, _ptr(keep["obs"]), p.n_obstacles,
                 _ptr(keep["start"]), _ptr(keep["goal"]), p.goal_radius, p.goal_angle_dim, p.goal_angle,
                 p.goal_angle_tol, p.dt, p.steps_per_edge, p.cost_mode, p.heuristic_speed,
                 0 if p.goal_dims is None else len(p.goal_dims), _ptr(keep["gdims"], _ip))
    return s, keep


class Planner:
    """pakr_create / pakr_plan / pakr_expand_step / pakr_destroy with torch-supplied memory and stream."""

    def __init__(self, problem, device: int = 0):
        import torch  # device memory and streams only
        self._torch = torch
        self.problem = problem
        self.device = device
        self.D, self.m = problem.state_dim, problem.control_dim
        self.Dp = (self.D + 3) // 4 * 4
        s, keep = make_problem_struct(problem)
        h = C.c_void_p()
        st = lib().pakr_create(C.byref(s), device, C.byref(h))
        if st != 0:
            raise PakrError(st, (lib().pakr_last_error(None) or b"").decode())
        self._h = h
        self._ws = None
        self._last_ws = None  # the workspace the last plan() ran in (read_tree's default)

    def close(self):
        if getattr(self, "_h", None):
            lib().pakr_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, st: int):
        if st != 0:
            raise PakrError(st, (lib().pakr_last_error(self._h) or b"").decode())

    def workspace_bytes(self, B: int, K: int, cap: int) -> int:
        return int(lib().pakr_workspace_bytes(self._h, B, K, cap))

    def workspace_bytes_for(self, B: int, K: int, cap: int, nn_mode: int) -> int:
        """pakr_workspace_bytes_for: what calls with this nn_mode need (no buffers of tiers the mode cannot launch)."""
        return int(lib().pakr_workspace_bytes_for(self._h, B, K, cap, nn_mode))

    def workspace(self, B: int, K: int, cap: int):
        """A cached torch.uint8 device tensor of at least pakr_workspace_bytes()."""
        need = self.workspace_bytes(B, K, cap)
        if need == 0:
            raise PakrError(1, "invalid B, K or tree_capacity")
        if self._ws is None or self._ws.numel() < need:
            self._ws = None
            self._ws = self._torch.empty(need, dtype=self._torch.uint8, device=f"cuda:{self.device}")
        return self._ws

    def _stream(self) -> int:
        return int(self._torch.cuda.current_stream(self.device).cuda_stream)

    # ---- pakr_plan ----
    def plan(self, seed: int, B: int, K: int, tree_capacity: int, n_replans: int, time_budget_ms: float = 0.0,
             max_iters_per_replan: int = 0, path_capacity: int = 8192, workspace=None,
             initial_cost_bound: float = 0.0, nn_mode: int = NN_AUTO) -> dict:
        ws = workspace if workspace is not None else self.workspace(B, K, tree_capacity)
        self._last_ws = ws
        nodes = np.zeros(path_capacity, np.int32)
        states = np.zeros((path_capacity, self.D), np.float32)
        ctrls = np.zeros((max(path_capacity - 1, 1), self.m), np.float32)
        opts = _PlanOpts(seed, B, K, tree_capacity, n_replans, time_budget_ms, max_iters_per_replan, initial_cost_bound,
                         nn_mode)
        res = _Result(_ptr(nodes, _ip), _ptr(states), _ptr(ctrls), path_capacity, 0, 0.0, 0, 0, _Stats())
        st = lib().pakr_plan(self._h, C.byref(opts), C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(self._stream()),
                             C.byref(res))
        self._check(st)
        s = res.stats
        R = min(int(s.replans_run), MAX_REPLAN_STATS)
        L = int(res.path_len)
        return dict(outcome=int(res.outcome), cost=float(res.cost), path_len=L, path_nodes=nodes[:L].copy(),
                    path_states=states[:L].copy(), path_controls=ctrls[:max(L - 1, 0)].copy(),
                    final_tree_nodes=int(res.final_tree_nodes), iterations=int(s.iterations), children=int(s.children),
                    inserted=int(s.inserted), nn_pairs=int(s.nn_pairs), nn_pairs_evaluated=int(s.nn_pairs_evaluated),
                    nn_pairs_filtered=int(s.nn_pairs_filtered),
                    h2d_bytes=int(s.h2d_bytes),
                    d2h_bytes=int(s.d2h_bytes), replans_run=int(s.replans_run), replans_solved=int(s.replans_solved),
                    termination=int(s.termination), first_solution_ms=float(s.first_solution_ms),
                    device_ms=float(s.device_ms), phase_ms=[float(v) for v in s.phase_ms], replan_cost=np.array(s.replan_cost[:R], np.float32),
                    replan_nodes=np.array(s.replan_nodes[:R], np.int64), replan_iters=np.array(s.replan_iters[:R], np.int64),
                    replan_end_ms=np.array(s.replan_end_ms[:R], np.float64),
                    replan_stats_truncated=int(s.replan_stats_truncated), path_truncated=int(s.path_truncated))

    def read_tree(self, B: int, K: int, tree_capacity: int, n: int, workspace=None) -> dict:
        """Copies the first n nodes of the tree pakr_plan left in `workspace` (default: the workspace of the last
        plan() call) to numpy."""
        torch = self._torch
        lay = _TreeLayout()
        self._check(lib().pakr_get_tree_layout(self._h, B, K, tree_capacity, C.byref(lay)))
        ws = workspace if workspace is not None else self._last_ws
        if ws is None:
            raise PakrError(1, "read_tree: no workspace given and plan() has not run")

        def view(off, count, dtype):
            nbytes = count * 4
            return ws[off:off + nbytes].view(dtype).cpu().numpy()

        return dict(states=view(lay.states_off, n * self.Dp, torch.float32).reshape(n, self.Dp)[:, :self.D].copy(),
                    actions=view(lay.actions_off, n * 4, torch.float32).reshape(n, 4)[:, :self.m].copy(),
                    parents=view(lay.parents_off, n, torch.int32).copy(),
                    costs=view(lay.costs_off, n, torch.float32).copy())

    def read_stats(self, B: int, K: int, tree_capacity: int, workspace=None) -> dict:
        """pakr_read_stats: statistics of the last launch on this workspace (synchronises the stream)."""
        ws = workspace if workspace is not None else self.workspace(B, K, tree_capacity)
        st = _Stats()
        self._check(lib().pakr_read_stats(self._h, B, K, tree_capacity, C.c_void_p(ws.data_ptr()), ws.numel(),
                                          C.c_void_p(self._stream()), C.byref(st)))
        return dict(iterations=int(st.iterations), children=int(st.children), inserted=int(st.inserted),
                    nn_pairs=int(st.nn_pairs), nn_pairs_evaluated=int(st.nn_pairs_evaluated),
                    nn_pairs_filtered=int(st.nn_pairs_filtered), device_ms=float(st.device_ms), phase_ms=[float(v) for v in st.phase_ms])

    # ---- pakr_expand_step ----
    def new_tree(self, capacity: int, host: Optional[dict] = None) -> dict:
        """Device tree buffers in the layout of include/pakr.h; optionally filled from numpy arrays."""
        torch = self._torch
        dev = f"cuda:{self.device}"
        t = dict(states=torch.zeros((capacity, self.Dp), dtype=torch.float32, device=dev),
                 actions=torch.zeros((capacity, 4), dtype=torch.float32, device=dev),
                 parents=torch.zeros(capacity, dtype=torch.int32, device=dev),
                 costs=torch.zeros(capacity, dtype=torch.float32, device=dev),
                 n_nodes=torch.zeros(1, dtype=torch.int32, device=dev), capacity=capacity)
        if host is None:
            host = dict(states=np.asarray(self.problem.start, np.float32)[None, :], actions=np.zeros((1, self.m), np.float32),
                        parents=np.array([-1], np.int32), costs=np.zeros(1, np.float32))
        n = len(host["parents"])
        t["states"][:n, :self.D] = torch.from_numpy(np.ascontiguousarray(host["states"], dtype=np.float32)).to(dev)
        t["actions"][:n, :self.m] = torch.from_numpy(np.ascontiguousarray(host["actions"], dtype=np.float32)).to(dev)
        t["parents"][:n] = torch.from_numpy(np.ascontiguousarray(host["parents"], dtype=np.int32)).to(dev)
        t["costs"][:n] = torch.from_numpy(np.ascontiguousarray(host["costs"], dtype=np.float32)).to(dev)
        t["n_nodes"][0] = n
        return t

    def expand_step(self, tree: dict, seed: int, replan: int, iteration: int, B: int, K: int,
                    c_best: float = float("inf"), debug: bool = True, workspace=None,
                    nn_mode: int = NN_AUTO) -> Optional[dict]:
        torch = self._torch
        dev = f"cuda:{self.device}"
        cap = tree["capacity"]
        ws = workspace if workspace is not None else self.workspace(B, K, cap)
        dbg = None
        ptr = lambda t: C.c_void_p(t.data_ptr())
        null = C.c_void_p(0)
        if debug:
            BK = B * K
            dbg = dict(x_rand=torch.zeros((B, self.Dp), dtype=torch.float32, device=dev),
                       nn_idx=torch.zeros(B, dtype=torch.int32, device=dev),
                       nn_d2=torch.zeros(B, dtype=torch.float32, device=dev),
                       child_state=torch.zeros((BK, self.Dp), dtype=torch.float32, device=dev),
                       child_ctrl=torch.zeros((BK, 4), dtype=torch.float32, device=dev),
                       child_cost=torch.zeros(BK, dtype=torch.float32, device=dev),
                       child_flags=torch.zeros(BK, dtype=torch.int32, device=dev),
                       n_inserted=torch.zeros(1, dtype=torch.int32, device=dev),
                       goal_node=torch.zeros(1, dtype=torch.int32, device=dev),
                       new_c_best=torch.zeros(1, dtype=torch.float32, device=dev))
        g = (lambda k: ptr(dbg[k])) if debug else (lambda k: null)
        a = _StepArgs(seed, replan, iteration, B, K, cap, c_best, nn_mode, ptr(tree["states"]), ptr(tree["actions"]),
                      ptr(tree["parents"]), ptr(tree["costs"]), ptr(tree["n_nodes"]), g("x_rand"), g("nn_idx"),
                      g("nn_d2"), g("child_state"), g("child_ctrl"), g("child_cost"), g("child_flags"),
                      g("n_inserted"), g("goal_node"), g("new_c_best"))
        st = lib().pakr_expand_step(self._h, C.byref(a), C.c_void_p(ws.data_ptr()), ws.numel(), C.c_void_p(self._stream()))
        self._check(st)
        if not debug:
            return None
        torch.cuda.synchronize(self.device)
        out = {k: v.cpu().numpy() for k, v in dbg.items()}
        out["x_rand"] = out["x_rand"][:, :self.D]
        out["child_state"] = out["child_state"][:, :self.D]
        out["child_ctrl"] = out["child_ctrl"][:, :self.m]
        for k in ("n_inserted", "goal_node", "new_c_best"):
            out[k] = out[k][0].item()
        return out

    # ---- pakr_expand_step_static ----
    def expand_step_static(self, tree: dict, seed: int, replan: int, iteration: int, B: int, K: int,
                           c_best: float = float("inf"), nn_mode: int = NN_AUTO) -> dict:
        """pakr_expand_step_static: one iteration without a workspace, for callers that may not allocate device
        memory while they run (a deadline-bound control loop, a plug-in whose host owns the pool).  The library's
        scratch is a fixed 2.25 MiB array inside libpakr.so on each GPU; B*K <= STATIC_MAX_CHILDREN, NN = tiled scan.
        The C call allocates nothing.  The tree (in/out) and the per-child output tensors are the caller's: this
        convenience wrapper makes the outputs with torch, exactly as expand_step(debug=True) does, and returns them as
        numpy.  One array per device is shared by all planners: calls on different streams must not overlap."""
        torch = self._torch
        dev = f"cuda:{self.device}"
        BK = B * K
        ptr = lambda t: C.c_void_p(t.data_ptr())
        dbg = dict(x_rand=torch.zeros((B, self.Dp), dtype=torch.float32, device=dev),
                   nn_idx=torch.zeros(B, dtype=torch.int32, device=dev),
                   nn_d2=torch.zeros(B, dtype=torch.float32, device=dev),
                   child_state=torch.zeros((BK, self.Dp), dtype=torch.float32, device=dev),
                   child_ctrl=torch.zeros((BK, 4), dtype=torch.float32, device=dev),
                   child_cost=torch.zeros(BK, dtype=torch.float32, device=dev),
                   child_flags=torch.zeros(BK, dtype=torch.int32, device=dev),
                   n_inserted=torch.zeros(1, dtype=torch.int32, device=dev),
                   goal_node=torch.zeros(1, dtype=torch.int32, device=dev),
                   new_c_best=torch.zeros(1, dtype=torch.float32, device=dev))
        a = _StepArgs(seed, replan, iteration, B, K, tree["capacity"], c_best, nn_mode, ptr(tree["states"]),
                      ptr(tree["actions"]), ptr(tree["parents"]), ptr(tree["costs"]), ptr(tree["n_nodes"]),
                      *[ptr(dbg[k]) for k in ("x_rand", "nn_idx", "nn_d2", "child_state", "child_ctrl", "child_cost",
                                              "child_flags", "n_inserted", "goal_node", "new_c_best")])
        self._check(lib().pakr_expand_step_static(self._h, C.byref(a), C.c_void_p(self._stream())))
        torch.cuda.synchronize(self.device)
        out = {k: v.cpu().numpy() for k, v in dbg.items()}
        out["x_rand"] = out["x_rand"][:, :self.D]
        out["child_state"] = out["child_state"][:, :self.D]
        out["child_ctrl"] = out["child_ctrl"][:, :self.m]
        for k in ("n_inserted", "goal_node", "new_c_best"):
            out[k] = out[k][0].item()
        return out
