"""Pins of the oracle's Acrobot (reading P35) and of the goal ball over listed dims.

The paper prints no equations for the Acrobot, so the pins come from mechanics that is independent of the
D(q) qdd + c = -dV/dq + B u form the oracle evaluates: total energy rebuilt from the CARTESIAN velocities of the two
centres of mass (conserved at zero torque; changed by exactly tau * delta(theta2) under a constant elbow torque),
the parallel-axis theorem for the straight arm, the two normal modes of the hanging pendulum (numpy's eigen-solver),
and the two equilibria.  A flipped Coriolis or gravity sign, a wrong d12, or a torque applied to the wrong joint
turns one of them red (each was mutation-checked).
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl


def _acrobot(orc, dt=None, **kw):
    p, cfg = wl.CONFIGS["N4"]()
    big = np.float32(1e6)
    p = dataclasses.replace(p, state_lo=np.array([-math.pi, -math.pi, -big, -big], np.float32),
                            state_hi=np.array([math.pi, math.pi, big, big], np.float32), **kw)
    if dt is not None:
        p = dataclasses.replace(p, dt=dt)
    return p, orc.OracleProblem(p)


def _energy(par, x):
    """Kinetic energy from the Cartesian velocities of the centres of mass plus the spin of each link about it;
    potential m g y.  theta1 from the downward vertical, theta2 relative to link 1."""
    m1, m2, l1, lc1, lc2, I1, I2, g = par
    t1, t2, w1, w2 = x
    a = t1 + t2
    v1 = lc1 * w1 * np.array([math.cos(t1), math.sin(t1)])
    v2 = l1 * w1 * np.array([math.cos(t1), math.sin(t1)]) + lc2 * (w1 + w2) * np.array([math.cos(a), math.sin(a)])
    kin = 0.5 * m1 * v1 @ v1 + 0.5 * I1 * w1 ** 2 + 0.5 * m2 * v2 @ v2 + 0.5 * I2 * (w1 + w2) ** 2
    y1 = -lc1 * math.cos(t1)
    y2 = -l1 * math.cos(t1) - lc2 * math.cos(a)
    return kin + m1 * g * y1 + m2 * g * y2


def _roll(op, x, u, steps):
    x = np.asarray(x, dtype=np.float64)
    for _ in range(steps):
        x = op.step(x, u)   # no wrap inside: theta2 stays continuous
    return x


def test_acrobot_equilibria_and_straight_arm_inertia(orc):
    p, op = _acrobot(orc)
    par = p.dyn_params.astype(np.float64)
    m1, m2, l1, lc1, lc2, I1, I2, g = par
    for eq in ([0, 0, 0, 0], [math.pi, 0, 0, 0], [0, math.pi, 0, 0], [math.pi, math.pi, 0, 0]):
        np.testing.assert_allclose(op.f(eq, [0.0]), 0.0, atol=1e-12)
    # hanging straight at rest (gravity torque 0), elbow torque tau: D0 qdd = (0, tau) with D0 from the parallel-axis
    # theorem: the whole arm about the shoulder, link 2 about the shoulder through the elbow coupling, link 2 about the elbow
    tau = 3.0
    D0 = np.array([[I1 + m1 * lc1 ** 2 + I2 + m2 * (l1 + lc2) ** 2, I2 + m2 * lc2 * (l1 + lc2)],
                   [I2 + m2 * lc2 * (l1 + lc2), I2 + m2 * lc2 ** 2]])
    qdd = np.linalg.solve(D0, [0.0, tau])
    xd = op.f([0, 0, 0, 0], [tau])
    np.testing.assert_allclose(xd, [0, 0, qdd[0], qdd[1]], rtol=1e-12, atol=1e-12)
    assert xd[3] > 0 > xd[2]  # the elbow follows the torque, the shoulder recoils
    # state slots: velocities feed the angles
    xd = op.f([0.3, -0.2, 0.7, -0.4], [0.0])
    assert xd[0] == 0.7 and xd[1] == -0.4


def test_acrobot_energy_is_conserved_without_torque(orc):
    p, op = _acrobot(orc, dt=1e-3)
    par = p.dyn_params.astype(np.float64)
    x0 = np.array([1.9, -1.1, 2.5, -3.0])   # fast, far from the linear regime: Coriolis terms matter
    e0 = _energy(par, x0)
    x = _roll(op, x0, [0.0], 3000)
    assert np.abs(x - x0).max() > 1.0
    assert abs(_energy(par, x) - e0) < 1e-8 * max(1.0, abs(e0))


def test_acrobot_elbow_torque_does_work_on_theta2(orc):
    """dE/dt = tau * theta2_dot: the torque acts at the elbow, on the RELATIVE angle."""
    p, op = _acrobot(orc, dt=1e-3)
    par = p.dyn_params.astype(np.float64)
    for tau, x0 in ((4.0, [0.4, 0.3, 0.0, 0.0]), (-7.5, [-1.0, 2.0, 1.0, -2.0])):
        x0 = np.array(x0)
        x = _roll(op, x0, [tau], 600)
        work = tau * (x[1] - x0[1])
        assert abs(work) > 0.5
        assert _energy(par, x) - _energy(par, x0) == pytest.approx(work, rel=1e-7)


def test_acrobot_normal_modes_of_the_hanging_pendulum(orc):
    """Small oscillations about theta = 0: D0 qdd + G q = 0, G the Hessian of m g y.  Started along an eigenvector of
    D0^-1 G (numpy) the motion is q(t) = v cos(w t) up to O(amplitude^3)."""
    p, op = _acrobot(orc, dt=1e-3)
    m1, m2, l1, lc1, lc2, I1, I2, g = p.dyn_params.astype(np.float64)
    D0 = np.array([[I1 + m1 * lc1 ** 2 + I2 + m2 * (l1 + lc2) ** 2, I2 + m2 * lc2 * (l1 + lc2)],
                   [I2 + m2 * lc2 * (l1 + lc2), I2 + m2 * lc2 ** 2]])
    G = g * np.array([[m1 * lc1 + m2 * (l1 + lc2), m2 * lc2], [m2 * lc2, m2 * lc2]])
    lam, vec = np.linalg.eig(np.linalg.solve(D0, G))
    assert (lam.real > 0).all() and abs(lam[0] - lam[1]) > 1.0
    amp = 1e-4
    for k in range(2):
        w = math.sqrt(lam[k].real)
        v = vec[:, k].real / np.abs(vec[:, k].real).max() * amp
        steps = int(round(0.8 * 2 * math.pi / w / 1e-3))   # 0.8 of a period
        x = _roll(op, [v[0], v[1], 0, 0], [0.0], steps)
        t = steps * float(np.float32(1e-3))
        np.testing.assert_allclose(x[:2], v * math.cos(w * t), atol=2e-4 * amp)
        np.testing.assert_allclose(x[2:], -v * w * math.sin(w * t), atol=2e-4 * amp * w)


def test_acrobot_upright_is_unstable(orc):
    p, op = _acrobot(orc, dt=1e-3)
    x = _roll(op, [math.pi - 1e-6, 0, 0, 0], [0.0], 2000)
    assert abs(x[0] - math.pi) > 1e-4


def test_goal_ball_over_listed_dims_wraps_angles(orc):
    """X_goal of N4: ball of radius 0.3 in (theta1, theta2) around (pi, 0), differences wrapped (P18 / P35)."""
    p, op = _acrobot(orc)
    r = float(np.float32(p.goal_radius))
    inside, mg = op.in_goal([-math.pi + 0.1, 0.2, 5.0, -5.0])   # 0.1 past the seam from +pi; velocities are free
    assert inside and mg == pytest.approx(r - math.hypot(0.1, 0.2), abs=1e-6)
    assert not op.in_goal([math.pi - 0.25, 0.25, 0, 0])[0]      # 0.354 away
    assert op.in_goal([float(p.goal_center[0]), r, 0, 0])[0]     # closed ball: on the rim is inside
    assert not op.in_goal([0.0, 0.0, 0, 0])[0]
    # heuristic: (distance over the goal dims - r) / speed, wrapped the same way
    h = op.heuristic([-math.pi + 1.0, 0.0, 0, 0])
    assert h == pytest.approx((1.0 - r) / float(np.float32(p.heuristic_speed)), rel=1e-6)
    # a goal over a subset that includes a velocity: rest-to-rest style ball on (theta1, theta1_dot)
    p2 = dataclasses.replace(p, goal_dims=np.array([0, 2], np.int32), goal_center=np.array([math.pi, 0.0], np.float32),
                             heuristic_speed=float("inf"))
    op2 = orc.OracleProblem(p2)
    assert op2.in_goal([math.pi - 0.1, 2.0, 0.2, 9.0])[0]
    assert not op2.in_goal([math.pi - 0.1, 2.0, 0.4, 9.0])[0]
    assert op2.heuristic([0, 0, 0, 0]) == 0.0
    # default (goal_dims None) is still the position ball: C1
    p1, _ = wl.config1()
    op1 = orc.OracleProblem(p1)
    assert op1.in_goal([9.5, 9.2, 1, 1])[0] and not op1.in_goal([9.5, 8.9, 0, 0])[0]


def test_acrobot_plan_swings_up_and_validates(orc):
    """Alg. 1 on N4 with a small batch: the returned plan, re-propagated from the hanging start, ends in the goal ball
    and every edge keeps the angular rates inside the box."""
    p, _ = wl.CONFIGS["N4"]()
    op = orc.OracleProblem(p)
    res = orc.plan(op, 0, 64, 8, 60000, 1)
    assert res["outcome"] == 1
    code, cost, err = op.validate_plan(res["path_states"], res["path_controls"])
    assert code == 0 and cost == pytest.approx(res["cost"], rel=1e-9) and err < 1e-9
    assert op.in_goal(res["path_states"][-1])[0]
    assert np.abs(res["path_states"][:, 2:]).max() <= 10.0
