"""Seeded synthetic workloads (BASELINE.json configs C1-C5) shared by the oracle and the CUDA path.

This module holds NONE of the method's arithmetic: it only draws obstacle fields with numpy's
PCG64 and fills in the problem statement of PAPER.md:59-69 (dynamics id, bounds, obstacles,
start, goal, dt/steps).  Both sides receive the same fp32 arrays (the oracle widens them).

The paper measures on Kino-PAX's Tree/Narrow/House meshes and DynoBench
problems; neither exists here, and nothing of them is reproduced.  These
analytic obstacle fields stand in for them.

Readings used: P27-P30 for start/goal/bounds/obstacle generation, P15 for the
heuristic speed cap.
"""
from __future__ import annotations

import dataclasses
import math
from typing import Optional

import numpy as np

# ABI constants (numeric values documented in DESIGN.md; restated in include/pakr.h and
# oracle/pakr_oracle.h independently).
DYN_DOUBLE_INTEGRATOR, DYN_UNICYCLE2, DYN_QUADROTOR, DYN_DUBINS_AIRPLANE, DYN_UNICYCLE1 = 0, 1, 2, 3, 4
DYN_QUADROTOR_BODY, DYN_ACROBOT = 5, 6
INT_EULER, INT_RK4 = 0, 1
OBS_CIRCLE2D, OBS_AABB, OBS_ZCYLINDER = 0, 1, 2
COST_DURATION, COST_PATH_LENGTH = 0, 1
DIM_REAL, DIM_ANGLE = 0, 1


@dataclasses.dataclass
class Problem:
    """Field-for-field the `pakr_problem` of include/pakr.h, as fp32 numpy arrays."""
    name: str
    dynamics_id: int
    integrator: int
    state_dim: int
    control_dim: int
    pos_dim: int
    dyn_params: np.ndarray
    state_lo: np.ndarray
    state_hi: np.ndarray
    dim_kind: np.ndarray
    nn_weight: np.ndarray
    control_lo: np.ndarray
    control_hi: np.ndarray
    obstacle_type: int
    obstacles: np.ndarray          # [O, 3] circles/cylinders (cx, cy, r); [O, 2*pos_dim] boxes (lo, hi)
    start: np.ndarray
    goal_center: np.ndarray
    goal_radius: float
    goal_angle_dim: int
    goal_angle: float
    goal_angle_tol: float
    dt: float
    steps_per_edge: int
    cost_mode: int
    heuristic_speed: float
    goal_dims: Optional[np.ndarray] = None   # int32 state indices the goal ball spans; None = the position dims

    @property
    def n_obstacles(self) -> int:
        return int(self.obstacles.shape[0])

    @property
    def state_stride(self) -> int:
        """Floats per node in the device tree: D rounded up to a multiple of 4 (DESIGN.md layout)."""
        return (self.state_dim + 3) // 4 * 4

    @property
    def control_stride(self) -> int:
        return 4


@dataclasses.dataclass
class PlanConfig:
    B: int
    K: int
    tree_capacity: int
    n_replans: int
    seed: int = 0
    time_budget_ms: float = 0.0
    max_iters_per_replan: int = 0


def _f32(a) -> np.ndarray:
    return np.ascontiguousarray(np.asarray(a, dtype=np.float32))


def _place(rng: np.random.Generator, n: int, draw, clear_of) -> np.ndarray:
    """P30: draw primitives until n are accepted; `clear_of(prim)` rejects one too close to start/goal."""
    out = []
    guard = 0
    while len(out) < n:
        prim = draw(rng)
        guard += 1
        if guard > 100000:
            raise RuntimeError("obstacle placement did not converge")
        if clear_of(prim):
            out.append(prim)
    return _f32(np.stack(out))


def _circles(rng, n, ws_lo, ws_hi, r_lo, r_hi, start_xy, goal_xy, goal_r, inflate=0.5):
    ws_lo = np.asarray(ws_lo, dtype=np.float64)
    ws_hi = np.asarray(ws_hi, dtype=np.float64)

    def draw(g):
        c = g.uniform(ws_lo, ws_hi)
        r = g.uniform(r_lo, r_hi)
        return np.array([c[0], c[1], r])

    def ok(p):
        c, r = p[:2], p[2]
        if np.linalg.norm(c - start_xy) <= r + inflate:
            return False
        if np.linalg.norm(c - goal_xy) <= r + inflate + goal_r:
            return False
        return True

    return _place(rng, n, draw, ok)


def _boxes(rng, n, ws_lo, ws_hi, side_lo, side_hi, start_p, goal_p, goal_r, inflate=0.5):
    ws_lo = np.asarray(ws_lo, dtype=np.float64)
    ws_hi = np.asarray(ws_hi, dtype=np.float64)
    pd = ws_lo.shape[0]

    def draw(g):
        c = g.uniform(ws_lo, ws_hi)
        side = g.uniform(side_lo, side_hi, size=pd)  # one draw per axis
        return np.concatenate([c - side / 2, c + side / 2])

    def dist_to_box(p, lo, hi):
        return np.linalg.norm(np.maximum(np.maximum(lo - p, p - hi), 0.0))

    def ok(b):
        lo, hi = b[:pd], b[pd:]
        if dist_to_box(start_p, lo, hi) <= inflate:
            return False
        if dist_to_box(goal_p, lo, hi) <= inflate + goal_r:
            return False
        return True

    return _place(rng, n, draw, ok)


def config1(env_seed: int = 101) -> tuple[Problem, PlanConfig]:
    """C1: 2D double integrator, Euler, 8 circles (BASELINE.json configs[0])."""
    rng = np.random.Generator(np.random.PCG64(env_seed))
    start = np.array([0.5, 0.5, 0.0, 0.0])
    goal = np.array([9.5, 9.5])
    obs = _circles(rng, 8, [0, 0], [10, 10], 0.5, 1.5, start[:2], goal, 0.5)
    p = Problem(
        name="C1-di2d", dynamics_id=DYN_DOUBLE_INTEGRATOR, integrator=INT_EULER, state_dim=4,
        control_dim=2, pos_dim=2, dyn_params=_f32([]), state_lo=_f32([0, 0, -1, -1]),
        state_hi=_f32([10, 10, 1, 1]), dim_kind=np.zeros(4, np.uint8), nn_weight=_f32([1, 1, 1, 1]),
        control_lo=_f32([-1, -1]), control_hi=_f32([1, 1]), obstacle_type=OBS_CIRCLE2D,
        obstacles=obs, start=_f32(start), goal_center=_f32(goal), goal_radius=0.5,
        goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0, dt=0.05, steps_per_edge=10,
        cost_mode=COST_DURATION, heuristic_speed=math.sqrt(2.0))
    return p, PlanConfig(B=256, K=4, tree_capacity=65536, n_replans=10, seed=0)


def _di3d(name: str, n_boxes: int, env_seed: int) -> Problem:
    rng = np.random.Generator(np.random.PCG64(env_seed))
    start = np.array([0.5, 0.5, 0.5, 0, 0, 0.0])
    goal = np.array([9.5, 9.5, 9.5])
    obs = _boxes(rng, n_boxes, [0, 0, 0], [10, 10, 10], 0.5, 2.0, start[:3], goal, 0.5)
    return Problem(
        name=name, dynamics_id=DYN_DOUBLE_INTEGRATOR, integrator=INT_RK4, state_dim=6,
        control_dim=3, pos_dim=3, dyn_params=_f32([]), state_lo=_f32([0, 0, 0, -1, -1, -1]),
        state_hi=_f32([10, 10, 10, 1, 1, 1]), dim_kind=np.zeros(6, np.uint8),
        nn_weight=_f32([1] * 6), control_lo=_f32([-1] * 3), control_hi=_f32([1] * 3),
        obstacle_type=OBS_AABB, obstacles=obs, start=_f32(start), goal_center=_f32(goal),
        goal_radius=0.5, goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0, dt=0.05,
        steps_per_edge=20, cost_mode=COST_DURATION, heuristic_speed=math.sqrt(3.0))


def config2(env_seed: int = 202) -> tuple[Problem, PlanConfig]:
    """C2: 3D double integrator, RK4, 32 boxes (BASELINE.json configs[1]; the bench workload)."""
    return _di3d("C2-di3d", 32, env_seed), PlanConfig(B=1024, K=8, tree_capacity=1 << 20, n_replans=20)


def config3(env_seed: int = 303) -> tuple[Problem, PlanConfig]:
    """C3: second-order unicycle, RK4, 64 circles (BASELINE.json configs[2])."""
    rng = np.random.Generator(np.random.PCG64(env_seed))
    start = np.array([1.0, 1.0, 0.0, 0.0, 0.0])
    goal = np.array([19.0, 19.0])
    obs = _circles(rng, 64, [0, 0], [20, 20], 0.3, 1.2, start[:2], goal, 0.5)
    pi = math.pi
    p = Problem(
        name="C3-unicycle2", dynamics_id=DYN_UNICYCLE2, integrator=INT_RK4, state_dim=5,
        control_dim=2, pos_dim=2, dyn_params=_f32([]), state_lo=_f32([0, 0, -pi, -1, -1]),
        state_hi=_f32([20, 20, pi, 1, 1]), dim_kind=np.array([0, 0, 1, 0, 0], np.uint8),
        nn_weight=_f32([1, 1, 1, 1, 1]), control_lo=_f32([-1, -2]), control_hi=_f32([1, 2]),
        obstacle_type=OBS_CIRCLE2D, obstacles=obs, start=_f32(start), goal_center=_f32(goal),
        goal_radius=0.5, goal_angle_dim=2, goal_angle=0.0, goal_angle_tol=0.5, dt=0.05,
        steps_per_edge=20, cost_mode=COST_DURATION, heuristic_speed=1.0)
    return p, PlanConfig(B=2048, K=8, tree_capacity=1 << 21, n_replans=20)


def config4(env_seed: int = 404) -> tuple[Problem, PlanConfig]:
    """C4: 12D quadrotor, RK4, 128 vertical cylinders (BASELINE.json configs[3])."""
    rng = np.random.Generator(np.random.PCG64(env_seed))
    m, g = 1.0, 9.81
    start = np.zeros(12)
    start[:3] = [1.0, 1.0, 2.5]
    goal = np.array([19.0, 19.0, 2.5])
    obs = _circles(rng, 128, [0, 0], [20, 20], 0.2, 0.5, start[:2], goal[:2], 0.5)
    vmax, amax, wmax = 5.0, 1.2, 6.0
    inf = np.inf
    lo = [0, 0, 0, -vmax, -vmax, -vmax, -amax, -amax, -inf, -wmax, -wmax, -wmax]
    hi = [20, 20, 5, vmax, vmax, vmax, amax, amax, inf, wmax, wmax, wmax]
    kind = np.zeros(12, np.uint8)
    kind[8] = DIM_ANGLE  # yaw; roll/pitch are real dims with finite bounds (P13)
    w = [1, 1, 1, 0.1, 0.1, 0.1, 0.2, 0.2, 0.02, 0.02, 0.02, 0.02]
    p = Problem(
        name="C4-quadrotor", dynamics_id=DYN_QUADROTOR, integrator=INT_RK4, state_dim=12,
        control_dim=4, pos_dim=3, dyn_params=_f32([m, 0.01, 0.01, 0.02, g]), state_lo=_f32(lo),
        state_hi=_f32(hi), dim_kind=kind, nn_weight=_f32(w),
        control_lo=_f32([0.0, -0.1, -0.1, -0.1]), control_hi=_f32([2 * m * g, 0.1, 0.1, 0.1]),
        obstacle_type=OBS_ZCYLINDER, obstacles=obs, start=_f32(start), goal_center=_f32(goal),
        goal_radius=0.5, goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0, dt=0.02,
        steps_per_edge=25, cost_mode=COST_DURATION, heuristic_speed=math.sqrt(3.0) * vmax)
    return p, PlanConfig(B=4096, K=16, tree_capacity=1 << 22, n_replans=30)


def config5(B: int = 1024, K: int = 16, env_seed: int = 505,
            tree_capacity: Optional[int] = None) -> tuple[Problem, PlanConfig]:
    """C5: scaling sweep point on the 6D double integrator with 128 boxes (BASELINE.json configs[4])."""
    cap = tree_capacity if tree_capacity is not None else 1 << 23
    return _di3d("C5-di3d-128", 128, env_seed), PlanConfig(B=B, K=K, tree_capacity=cap, n_replans=1)


def config6(env_seed: int = 606) -> tuple[Problem, PlanConfig]:
    """N1 (not a BASELINE config): 6D Dubins airplane [x,y,z,yaw,pitch,v]
    among 32 boxes in [0,10]^3; level start and goal, speed in [0.5, 1.5], pitch within +-0.6 rad."""
    rng = np.random.Generator(np.random.PCG64(env_seed))
    start = np.array([0.5, 0.5, 5.0, 0.0, 0.0, 1.0])
    goal = np.array([9.5, 9.5, 5.0])
    obs = _boxes(rng, 32, [0, 0, 0], [10, 10, 10], 0.5, 2.0, start[:3], goal, 0.7)
    pi = math.pi
    p = Problem(
        name="N1-dubins-airplane", dynamics_id=DYN_DUBINS_AIRPLANE, integrator=INT_RK4, state_dim=6,
        control_dim=3, pos_dim=3, dyn_params=_f32([]), state_lo=_f32([0, 0, 0, -pi, -0.6, 0.5]),
        state_hi=_f32([10, 10, 10, pi, 0.6, 1.5]), dim_kind=np.array([0, 0, 0, 1, 0, 0], np.uint8),
        nn_weight=_f32([1, 1, 1, 0.5, 0.5, 0.5]), control_lo=_f32([-1.0, -0.5, -0.5]),
        control_hi=_f32([1.0, 0.5, 0.5]), obstacle_type=OBS_AABB, obstacles=obs, start=_f32(start),
        goal_center=_f32(goal), goal_radius=0.7, goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0,
        dt=0.05, steps_per_edge=20, cost_mode=COST_DURATION, heuristic_speed=1.5)
    return p, PlanConfig(B=1024, K=8, tree_capacity=1 << 20, n_replans=10)


def config7(env_seed: int = 707) -> tuple[Problem, PlanConfig]:
    """N2 (NEXT-2, not a BASELINE config): first-order unicycle [x,y,theta], control (v, omega)
    among 40 circles in [0,20]^2 (the paper's custom problem has 40 obstacles)."""
    rng = np.random.Generator(np.random.PCG64(env_seed))
    start = np.array([1.0, 1.0, 0.0])
    goal = np.array([19.0, 19.0])
    obs = _circles(rng, 40, [0, 0], [20, 20], 0.3, 1.2, start[:2], goal, 0.5)
    pi = math.pi
    p = Problem(
        name="N2-unicycle1", dynamics_id=DYN_UNICYCLE1, integrator=INT_RK4, state_dim=3, control_dim=2,
        pos_dim=2, dyn_params=_f32([]), state_lo=_f32([0, 0, -pi]), state_hi=_f32([20, 20, pi]),
        dim_kind=np.array([0, 0, 1], np.uint8), nn_weight=_f32([1, 1, 0.5]), control_lo=_f32([-0.5, -1.5]),
        control_hi=_f32([1.0, 1.5]), obstacle_type=OBS_CIRCLE2D, obstacles=obs, start=_f32(start),
        goal_center=_f32(goal), goal_radius=0.5, goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0,
        dt=0.05, steps_per_edge=20, cost_mode=COST_DURATION, heuristic_speed=1.0)
    return p, PlanConfig(B=1024, K=8, tree_capacity=1 << 20, n_replans=10)


def config8(env_seed: int = 404) -> tuple[Problem, PlanConfig]:
    """N3 (NEXT-2, not a BASELINE config): the quadcopter exactly as the paper states it: state
    [x,y,z, phi,theta,psi, u,v,w, p,q,r] with body-frame linear velocities; C4's cylinder forest, limits and sizes."""
    c4, cfg = config4(env_seed)
    start = np.zeros(12)
    start[:3] = c4.start[:3]
    vmax, amax, wmax = 5.0, 1.2, 6.0
    inf = np.inf
    lo = [0, 0, 0, -amax, -amax, -inf, -vmax, -vmax, -vmax, -wmax, -wmax, -wmax]
    hi = [20, 20, 5, amax, amax, inf, vmax, vmax, vmax, wmax, wmax, wmax]
    kind = np.zeros(12, np.uint8)
    kind[5] = DIM_ANGLE
    w = [1, 1, 1, 0.2, 0.2, 0.02, 0.1, 0.1, 0.1, 0.02, 0.02, 0.02]
    p = dataclasses.replace(c4, name="N3-quadcopter-body", dynamics_id=DYN_QUADROTOR_BODY, state_lo=_f32(lo),
                            state_hi=_f32(hi), dim_kind=kind, nn_weight=_f32(w), start=_f32(start))
    return p, cfg


def config9() -> tuple[Problem, PlanConfig]:
    """N4 (NEXT-2, not a BASELINE config): Acrobot swing-up -- state [theta1, theta2, theta1_dot,
    theta2_dot], elbow torque; both angles are angle dims, no obstacles, start hanging at rest, goal a ball in angle
    space around the upright pose (theta1 = pi, theta2 = 0), velocities free like every other goal here (P18).
    Uniform unit rods (P35): m = 1, l = 1, lc = 0.5, I = m l^2 / 12, g = 9.81."""
    pi = math.pi
    wmax = 10.0
    p = Problem(
        name="N4-acrobot", dynamics_id=DYN_ACROBOT, integrator=INT_RK4, state_dim=4, control_dim=1, pos_dim=2,
        dyn_params=_f32([1.0, 1.0, 1.0, 0.5, 0.5, 1.0 / 12.0, 1.0 / 12.0, 9.81]),
        state_lo=_f32([-pi, -pi, -wmax, -wmax]), state_hi=_f32([pi, pi, wmax, wmax]),
        dim_kind=np.array([1, 1, 0, 0], np.uint8), nn_weight=_f32([1, 1, 0.1, 0.1]),
        control_lo=_f32([-10.0]), control_hi=_f32([10.0]), obstacle_type=OBS_CIRCLE2D,
        obstacles=np.zeros((0, 3), np.float32), start=_f32([0, 0, 0, 0]), goal_center=_f32([pi, 0.0]),
        goal_radius=0.3, goal_angle_dim=-1, goal_angle=0.0, goal_angle_tol=0.0, dt=0.02, steps_per_edge=10,
        cost_mode=COST_DURATION, heuristic_speed=math.sqrt(2.0) * wmax,
        goal_dims=np.array([0, 1], np.int32))
    return p, PlanConfig(B=1024, K=8, tree_capacity=1 << 20, n_replans=10)


CONFIGS = {"C1": config1, "C2": config2, "C3": config3, "C4": config4, "C5": config5, "N1": config6, "N2": config7, "N3": config8,
           "N4": config9}


def random_tree(problem: Problem, n: int, seed: int, flat: bool = False) -> dict[str, np.ndarray]:
    """Teacher-forcing / NN-microbench input: n nodes uniform in the state box.

    Node 0 is the start.  Parents point to a uniformly random earlier node, costs grow by one
    edge duration along parents, so the tree invariants hold by construction.  Positions are NOT
    filtered against obstacles (the NN scan and the propagation do not care).  flat=True makes every node a
    child of the root (vectorised; for multi-million-node microbenchmark trees).
    """
    rng = np.random.Generator(np.random.PCG64(seed))
    D, m = problem.state_dim, problem.control_dim
    lo = np.where(np.isfinite(problem.state_lo), problem.state_lo, -math.pi).astype(np.float64)
    hi = np.where(np.isfinite(problem.state_hi), problem.state_hi, math.pi).astype(np.float64)
    states = rng.uniform(lo, hi, size=(n, D)).astype(np.float32)
    states[0] = problem.start
    actions = rng.uniform(problem.control_lo, problem.control_hi, size=(n, m)).astype(np.float32)
    actions[0] = 0
    parents = np.full(n, -1, np.int32)
    if n > 1 and not flat:
        parents[1:] = (rng.random(n - 1) * np.arange(1, n)).astype(np.int32)
    elif n > 1:
        parents[1:] = 0
    edge = np.float32(problem.steps_per_edge) * np.float32(problem.dt)
    costs = np.zeros(n, np.float32)
    if flat:
        costs[1:] = edge
    else:
        for i in range(1, n):
            costs[i] = costs[parents[i]] + edge
    return {"states": states, "actions": actions, "parents": parents, "costs": costs}
