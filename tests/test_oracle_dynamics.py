"""Pins of the oracle's integrators and dynamics against closed forms (SURVEY.md 8(c) pin table).

Each test fixes something a plausible mistake would break: a dropped term, a wrong sign, a
transposed state slot, a wrong RK4 weight.
"""
import dataclasses
import math

import numpy as np
import pytest

from paper_2607_03987_b200 import workloads as wl


def _free(p, **kw):
    """Same problem without obstacles and with wide bounds, so closed forms are not cut short."""
    lo = np.where(np.isfinite(p.state_lo), -1e6, p.state_lo).astype(np.float32)
    hi = np.where(np.isfinite(p.state_hi), 1e6, p.state_hi).astype(np.float32)
    return dataclasses.replace(p, obstacles=p.obstacles[:0], state_lo=lo, state_hi=hi, **kw)


def test_euler_double_integrator_closed_form(orc):
    """C1 (P9): explicit Euler, position updated with the OLD velocity:
    v_S = v0 + S dt a ; p_S = p0 + S dt v0 + dt^2 a S(S-1)/2."""
    p, _ = wl.config1()
    op = orc.OracleProblem(_free(p))
    x0 = np.array([1.0, 2.0, 0.3, -0.2])
    u = np.array([0.7, -0.4])
    S, dt = p.steps_per_edge, float(np.float32(p.dt))
    x, flags, fb, _, ec = op.propagate(x0, u)
    v = x0[2:] + S * dt * u
    pos = x0[:2] + S * dt * x0[2:] + dt * dt * u * S * (S - 1) / 2
    np.testing.assert_allclose(x, np.concatenate([pos, v]), rtol=0, atol=1e-13)
    assert flags & orc.F_VALID and fb == 0
    assert ec == pytest.approx(S * dt, abs=1e-15)


def test_rk4_double_integrator_exact(orc):
    """C2: RK4 is exact for constant acceleration: p = p0 + v0 T + a T^2/2, v = v0 + a T."""
    p, _ = wl.config2()
    op = orc.OracleProblem(_free(p))
    x0 = np.array([1.0, 2.0, 3.0, 0.3, -0.2, 0.1])
    u = np.array([0.7, -0.4, 0.9])
    T = p.steps_per_edge * float(np.float32(p.dt))
    x, *_ = op.propagate(x0, u)
    np.testing.assert_allclose(x[:3], x0[:3] + x0[3:] * T + 0.5 * u * T * T, atol=1e-13)
    np.testing.assert_allclose(x[3:], x0[3:] + u * T, atol=1e-13)
    # one step, too: catches a wrong (h/6)(k1+2k2+2k3+k4) weight that only cancels over an edge
    dt = float(np.float32(p.dt))
    x1 = op.step(x0, u)
    np.testing.assert_allclose(x1[:3], x0[:3] + x0[3:] * dt + 0.5 * u * dt * dt, atol=1e-15)


def test_rk4_unicycle_closed_forms(orc):
    p, _ = wl.config3()
    op = orc.OracleProblem(_free(p))
    T = p.steps_per_edge * float(np.float32(p.dt))
    # straight line with constant acceleration: omega0 = alpha = 0
    x, *_ = op.propagate([2, 3, 0.6, 0.5, 0.0], [0.4, 0.0])
    s = 0.5 * T + 0.5 * 0.4 * T * T
    np.testing.assert_allclose(x, [2 + s * math.cos(0.6), 3 + s * math.sin(0.6), 0.6, 0.5 + 0.4 * T, 0.0], atol=1e-12)
    # constant-turn arc: a = alpha = 0
    v, w, th0 = 0.8, 0.7, -0.3
    x, *_ = op.propagate([2, 3, th0, v, w], [0.0, 0.0])
    ex = [2 + v / w * (math.sin(th0 + w * T) - math.sin(th0)), 3 - v / w * (math.cos(th0 + w * T) - math.cos(th0)),
          th0 + w * T, v, w]
    np.testing.assert_allclose(x, ex, atol=2e-9)
    # theta integrates omega which integrates alpha: theta = th0 + w T + alpha T^2 / 2 (exact for RK4)
    x, *_ = op.propagate([2, 3, 0.1, 0.0, 0.2], [0.0, 1.5])
    assert x[2] == pytest.approx(0.1 + 0.2 * T + 0.75 * T * T, abs=1e-13)
    assert x[4] == pytest.approx(0.2 + 1.5 * T, abs=1e-13)


def test_rk4_fourth_order_convergence(orc):
    """General unicycle / quadrotor edge vs the same RK4 at dt/16; halving dt cuts the error ~16x."""
    for cfg, x0, u in [
        (wl.config3, [2, 3, 0.4, 0.6, -0.5], [0.8, 1.7]),
        (wl.config4, [5, 5, 2, 1, -1, 0.5, 0.2, -0.3, 0.4, 0.5, -0.4, 0.3], [11.0, 0.05, -0.08, 0.03]),
    ]:
        p, _ = cfg()
        base = _free(p)
        T = p.steps_per_edge * float(np.float32(p.dt))

        def run(S):
            q = dataclasses.replace(base, dt=T / S, steps_per_edge=S)
            op = orc.OracleProblem(q)
            # dt passes through fp32 on the way in; use the widened value so S*dt == T only approximately
            return op.propagate(x0, u)[0], S * float(np.float32(T / S))

        ref, _ = run(p.steps_per_edge * 16)
        e1 = np.abs(run(p.steps_per_edge)[0] - ref).max()
        e2 = np.abs(run(p.steps_per_edge * 2)[0] - ref).max()
        assert e1 < 2e-5
        # fp32 rounding of dt makes T differ by ~1e-8 between runs; only assert the order when visible
        if e1 > 1e-7:
            assert 8.0 < e1 / e2 < 32.0


def test_quadrotor_fixed_points_and_axes(orc):
    p, _ = wl.config4()
    op = orc.OracleProblem(_free(p))
    m, Ixx, Iyy, Izz, g = [float(v) for v in p.dyn_params]
    T = p.steps_per_edge * float(np.float32(p.dt))
    x0 = np.zeros(12)
    x0[:3] = [3, 4, 2]
    # hover is a fixed point
    x, *_ = op.propagate(x0, [m * g, 0, 0, 0])
    np.testing.assert_allclose(x, x0, atol=1e-12)
    # free fall / pure vertical thrust: exact parabola in z, nothing else moves
    for thrust in (0.0, 1.5 * m * g):
        x, *_ = op.propagate(x0, [thrust, 0, 0, 0])
        az = thrust / m - g
        ex = x0.copy()
        ex[2] += 0.5 * az * T * T
        ex[5] += az * T
        np.testing.assert_allclose(x, ex, atol=1e-12)
    # pure tau_z from level: psi = r0 t + tau_z t^2 / (2 Izz); stays level
    xr = x0.copy()
    xr[11] = 0.3
    x, *_ = op.propagate(xr, [m * g, 0, 0, 0.05])
    assert x[8] == pytest.approx(0.3 * T + 0.05 * T * T / (2 * Izz), abs=1e-12)
    assert x[11] == pytest.approx(0.3 + 0.05 * T / Izz, abs=1e-12)
    np.testing.assert_allclose(x[[6, 7, 9, 10]], 0, atol=1e-14)
    # pure tau_x from level with zero thrust: phi = tau_x t^2 / (2 Ixx), p = tau_x t / Ixx
    x, *_ = op.propagate(x0, [0.0, 0.02, 0, 0])
    assert x[6] == pytest.approx(0.02 * T * T / (2 * Ixx), abs=1e-12)
    assert x[9] == pytest.approx(0.02 * T / Ixx, abs=1e-12)
    # pure tau_y: theta, q  (catches swapped torque axes / inertia slots)
    x, *_ = op.propagate(x0, [0.0, 0, 0.03, 0])
    assert x[7] == pytest.approx(0.03 * T * T / (2 * Iyy), abs=1e-12)
    assert x[10] == pytest.approx(0.03 * T / Iyy, abs=1e-12)


def test_quadrotor_thrust_direction_and_euler_rates(orc):
    """f(x,u) at hand-picked attitudes: R e3 columns and the ZYX Euler-rate matrix."""
    p, _ = wl.config4()
    op = orc.OracleProblem(_free(p))
    m, g = float(p.dyn_params[0]), float(p.dyn_params[4])
    a = 2.0 * g
    x = np.zeros(12)
    # pitch +90deg-ish (theta = 0.5): thrust tilts toward +x when psi = 0
    x[7] = 0.5
    xd = op.f(x, [a * m, 0, 0, 0])
    np.testing.assert_allclose(xd[3:6], [a * math.sin(0.5), 0.0, a * math.cos(0.5) - g], atol=1e-12)
    # roll phi = 0.5: thrust tilts toward -y
    x[:] = 0
    x[6] = 0.5
    xd = op.f(x, [a * m, 0, 0, 0])
    np.testing.assert_allclose(xd[3:6], [0.0, -a * math.sin(0.5), a * math.cos(0.5) - g], atol=1e-12)
    # yaw rotates the pitched thrust: psi = pi/2 sends +x tilt to +y
    x[:] = 0
    x[7], x[8] = 0.5, math.pi / 2
    xd = op.f(x, [a * m, 0, 0, 0])
    np.testing.assert_allclose(xd[3:6], [0.0, a * math.sin(0.5), a * math.cos(0.5) - g], atol=1e-12)
    # general attitude: R = Rz(psi) Ry(theta) Rx(phi), third column
    phi, th, psi = 0.3, -0.4, 1.1
    Rx = np.array([[1, 0, 0], [0, math.cos(phi), -math.sin(phi)], [0, math.sin(phi), math.cos(phi)]])
    Ry = np.array([[math.cos(th), 0, math.sin(th)], [0, 1, 0], [-math.sin(th), 0, math.cos(th)]])
    Rz = np.array([[math.cos(psi), -math.sin(psi), 0], [math.sin(psi), math.cos(psi), 0], [0, 0, 1]])
    x[:] = 0
    x[6:9] = [phi, th, psi]
    x[9:12] = [0.2, -0.5, 0.7]
    xd = op.f(x, [a * m, 0, 0, 0])
    np.testing.assert_allclose(xd[3:6], a * (Rz @ Ry @ Rx)[:, 2] - [0, 0, g], atol=1e-12)
    # Euler rates: omega_body = W(phi,theta) * euler_dot  <=>  check by inverting
    W = np.array([[1, 0, -math.sin(th)], [0, math.cos(phi), math.sin(phi) * math.cos(th)],
                  [0, -math.sin(phi), math.cos(phi) * math.cos(th)]])
    np.testing.assert_allclose(W @ xd[6:9], x[9:12], atol=1e-12)
    # position derivative is the world-frame velocity
    x[3:6] = [1, 2, 3]
    np.testing.assert_allclose(op.f(x, [0, 0, 0, 0])[:3], [1, 2, 3])


def test_quadrotor_torque_free_invariants(orc):
    """Torque-free rigid body: kinetic energy and |I w| are conserved (to O(dt^4))."""
    p, _ = wl.config4()
    op = orc.OracleProblem(_free(p))
    I = np.array([float(v) for v in p.dyn_params[1:4]])
    x0 = np.zeros(12)
    x0[9:12] = [1.0, -2.0, 1.5]
    x, *_ = op.propagate(x0, [0, 0, 0, 0])
    w0, w1 = x0[9:12], x[9:12]
    assert np.abs(w1 - w0).max() > 1e-2  # the gyroscopic term does something (Izz != Ixx)
    assert 0.5 * (I * w1 * w1).sum() == pytest.approx(0.5 * (I * w0 * w0).sum(), rel=1e-8)
    assert np.linalg.norm(I * w1) == pytest.approx(np.linalg.norm(I * w0), rel=1e-8)


def test_angle_wrap(orc):
    assert orc.wrap_pi(0.0) == 0.0
    assert orc.wrap_pi(math.pi) == pytest.approx(-math.pi)
    assert orc.wrap_pi(-math.pi) == pytest.approx(-math.pi)
    assert orc.wrap_pi(3 * math.pi + 0.25) == pytest.approx(-math.pi + 0.25)
    assert orc.wrap_pi(-7.0) == pytest.approx(-7.0 + 2 * math.pi)
    # P13: propagate wraps angle dims once, at the end of the edge
    p, _ = wl.config3()
    op = orc.OracleProblem(_free(p))
    T = p.steps_per_edge * float(np.float32(p.dt))
    x, *_ = op.propagate([2, 3, 3.0, 0.0, 1.0], [0.0, 0.0])  # theta -> 3 + T ~ 4.0 -> 4 - 2pi
    assert x[2] == pytest.approx(3.0 + T - 2 * math.pi, abs=1e-12)


def test_rk4_unicycle1_closed_forms(orc):
    """NEXT-2 model: straight line exact; constant (v, omega) is a circular arc
    x = x0 + (v/w)(sin(th0 + wT) - sin th0), y = y0 - (v/w)(cos(th0 + wT) - cos th0); heading th0 + wT (wrapped)."""
    p, _ = wl.config7()
    op = orc.OracleProblem(_free(p))
    T = p.steps_per_edge * float(np.float32(p.dt))
    x, *_ = op.propagate([2, 3, 0.6], [0.8, 0.0])
    np.testing.assert_allclose(x, [2 + 0.8 * T * math.cos(0.6), 3 + 0.8 * T * math.sin(0.6), 0.6], atol=1e-13)
    v, w, th0 = 0.9, -1.3, 2.9
    x, *_ = op.propagate([5, 6, th0], [v, w])
    np.testing.assert_allclose(x[0], 5 + (v / w) * (math.sin(th0 + w * T) - math.sin(th0)), atol=2e-8)
    np.testing.assert_allclose(x[1], 6 - (v / w) * (math.cos(th0 + w * T) - math.cos(th0)), atol=2e-8)
    assert x[2] == pytest.approx(orc.wrap_pi(th0 + w * T), abs=1e-13)
    # reversing (v < 0) moves against the heading: catches a dropped sign / swapped sin-cos
    x, *_ = op.propagate([5, 6, math.pi / 2], [-0.5, 0.0])
    np.testing.assert_allclose(x[:2], [5, 6 - 0.5 * T], atol=1e-13)


def test_rk4_dubins_airplane_closed_forms(orc):
    """NEXT-2 model (reading P33): velocity of magnitude v along (yaw, pitch).
    Zero rates + constant acceleration: straight line of length v0 T + a T^2/2 (RK4 exact for a quadratic);
    yaw rate only at level flight: horizontal circular arc; pitch rate only at yaw 0: vertical arc."""
    p, _ = wl.config6()
    op = orc.OracleProblem(_free(p))
    T = p.steps_per_edge * float(np.float32(p.dt))
    yaw, pitch, v0, a = 0.7, -0.3, 1.1, 0.4
    x, *_ = op.propagate([1, 2, 3, yaw, pitch, v0], [0.0, 0.0, a])
    s = v0 * T + 0.5 * a * T * T
    d = np.array([math.cos(pitch) * math.cos(yaw), math.cos(pitch) * math.sin(yaw), math.sin(pitch)])
    np.testing.assert_allclose(x[:3], np.array([1, 2, 3]) + s * d, atol=1e-13)
    np.testing.assert_allclose(x[3:], [yaw, pitch, v0 + a * T], atol=1e-13)
    w = 0.8  # level turn
    x, *_ = op.propagate([1, 2, 3, yaw, 0.0, v0], [w, 0.0, 0.0])
    np.testing.assert_allclose(x[0], 1 + (v0 / w) * (math.sin(yaw + w * T) - math.sin(yaw)), atol=2e-8)
    np.testing.assert_allclose(x[1], 2 - (v0 / w) * (math.cos(yaw + w * T) - math.cos(yaw)), atol=2e-8)
    assert x[2] == pytest.approx(3.0, abs=1e-13) and x[3] == pytest.approx(yaw + w * T, abs=1e-13)
    q = -0.45  # pull-down in the x-z plane
    x, *_ = op.propagate([1, 2, 3, 0.0, 0.2, v0], [0.0, q, 0.0])
    np.testing.assert_allclose(x[0], 1 + (v0 / q) * (math.sin(0.2 + q * T) - math.sin(0.2)), atol=2e-8)
    np.testing.assert_allclose(x[2], 3 - (v0 / q) * (math.cos(0.2 + q * T) - math.cos(0.2)), atol=2e-8)
    assert x[1] == pytest.approx(2.0, abs=1e-13) and x[4] == pytest.approx(0.2 + q * T, abs=1e-13)


def test_rk4_convergence_new_models(orc):
    """General motion of both NEXT-2 models against the same RK4 at dt/16: 4th-order (error ratio ~16 per halving)."""
    for cfgf, x0, u in ((wl.config6, [1, 2, 3, 0.4, 0.1, 1.0], [0.9, -0.4, 0.3]), (wl.config7, [1, 2, 0.4], [0.9, 1.2])):
        p, _ = cfgf()
        errs = []
        fine = orc.OracleProblem(_free(p, dt=p.dt / 16, steps_per_edge=p.steps_per_edge * 16)).propagate(x0, u)[0]
        for k in (1, 2):
            x = orc.OracleProblem(_free(p, dt=p.dt / k, steps_per_edge=p.steps_per_edge * k)).propagate(x0, u)[0]
            errs.append(np.abs(x - fine).max())
        assert errs[0] < 1e-6 and 10 < errs[0] / errs[1] < 24, errs


def _rot_zyx(phi, th, psi):
    cz, sz, cy, sy, cx, sx = math.cos(psi), math.sin(psi), math.cos(th), math.sin(th), math.cos(phi), math.sin(phi)
    Rz = np.array([[cz, -sz, 0], [sz, cz, 0], [0, 0, 1]])
    Ry = np.array([[cy, 0, sy], [0, 1, 0], [-sy, 0, cy]])
    Rx = np.array([[1, 0, 0], [0, cx, -sx], [0, sx, cx]])
    return Rz @ Ry @ Rx


def test_quadcopter_body_frame_model(orc):
    """NEXT-2 model exactly as PAPER.md:174 (body-frame velocities, reading P34).
    (i) hover is a fixed point; (ii) free fall from level rest: w_b = -g t, z = z0 - g t^2/2 (RK4 exact);
    (iii) forward body speed at yaw psi moves along the heading; (iv) the SAME physical motion as the
    world-frame model of config 4 (pinned separately): equivalent initial states (v_world = R v_b) and equal
    controls give equal position, angles, rates and world velocity after an edge."""
    pb, _ = wl.config8()
    pw, _ = wl.config4()
    ob, ow = orc.OracleProblem(_free(pb)), orc.OracleProblem(_free(pw))
    m, g = 1.0, float(np.float32(9.81))
    T = pb.steps_per_edge * float(np.float32(pb.dt))
    x0 = np.zeros(12)
    x0[:3] = [3, 4, 2]
    x, *_ = ob.propagate(x0, [m * g, 0, 0, 0])
    np.testing.assert_allclose(x, x0, atol=1e-12)
    x, *_ = ob.propagate(x0, [0, 0, 0, 0])
    assert x[8] == pytest.approx(-g * T, abs=1e-12) and x[2] == pytest.approx(2 - 0.5 * g * T * T, abs=1e-12)
    x1 = x0.copy()
    x1[5], x1[6] = 0.9, 1.5  # yaw, forward body speed
    x, *_ = ob.propagate(x1, [m * g, 0, 0, 0])
    np.testing.assert_allclose(x[:3], [3 + 1.5 * T * math.cos(0.9), 4 + 1.5 * T * math.sin(0.9), 2], atol=1e-12)
    # both are 4th-order discretisations of the same ODE: compare at dt/4, where their truncation errors (a few
    # 1e-6 at the config's dt) are ~256 times smaller
    fine = dict(dt=pb.dt / 4, steps_per_edge=pb.steps_per_edge * 4)
    ob, ow = orc.OracleProblem(_free(pb, **fine)), orc.OracleProblem(_free(pw, **fine))
    rng = np.random.default_rng(5)
    for _ in range(4):
        ang = rng.uniform([-0.5, -0.5, -3], [0.5, 0.5, 3])
        vb = rng.uniform(-2, 2, 3)
        rates = rng.uniform(-1, 1, 3)
        u = [rng.uniform(5, 15), *rng.uniform(-0.1, 0.1, 3)]
        R0 = _rot_zyx(*ang)
        xb = np.concatenate([[3, 4, 2], ang, vb, rates])
        xw = np.concatenate([[3, 4, 2], R0 @ vb, ang, rates])
        yb, *_ = ob.propagate(xb, u)
        yw, *_ = ow.propagate(xw, u)
        np.testing.assert_allclose(yb[:3], yw[:3], atol=1e-7)           # position
        np.testing.assert_allclose(yb[3:6], yw[6:9], atol=1e-7)         # Euler angles
        np.testing.assert_allclose(yb[9:], yw[9:], atol=1e-7)           # body rates
        np.testing.assert_allclose(_rot_zyx(*yb[3:6]) @ yb[6:9], yw[3:6], atol=1e-7)  # world velocity
