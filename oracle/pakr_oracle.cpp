/*
 * pakr_oracle.cpp -- TEST INFRASTRUCTURE, NOT THE PRODUCT (see pakr_oracle.h).
 *
 * Single-threaded fp64 restatement of PAKR's batched tree-expansion iteration inside AO-x
 * replanning, step by step in the order of PAPER.md Alg. 1.  No blocking,
 * fusion or reordering: every loop is the loop the paper's listing states.  "P<n>" are the
 * readings listed in DESIGN.md (taken from SURVEY.md Sec. 8(c)).
 *
 * Build: g++ -O2 -std=c++17 -shared -fPIC (no -ffast-math, no OpenMP).
 */
#include "pakr_oracle.h"

#include <chrono>
#include <cmath>
#include <cstring>
#include <limits>
#include <vector>

namespace {
const double kPi = 3.14159265358979323846;
const double kInf = std::numeric_limits<double>::infinity();
}  // namespace

/* ------------------------------------------------------------------------------------------
 * Philox4x32-10 (Salmon et al., "Parallel random numbers: as easy as 1, 2, 3", SC'11).
 * Reading P4: the paper is silent on the generator; BASELINE.json north_star (1) fixes a
 * Philox counter-based sampler keyed by (seed, replan, iteration, sample, branch).
 * ------------------------------------------------------------------------------------------ */
extern "C" void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]) {
  uint32_t c0 = ctr[0], c1 = ctr[1], c2 = ctr[2], c3 = ctr[3];
  uint32_t k0 = key[0], k1 = key[1];
  for (int round = 0; round < 10; ++round) {
    if (round > 0) {  // key schedule: Weyl sequence bump before every round but the first
      k0 += 0x9E3779B9u;
      k1 += 0xBB67AE85u;
    }
    const uint64_t p0 = (uint64_t)0xD2511F53u * c0;
    const uint64_t p1 = (uint64_t)0xCD9E8D57u * c2;
    const uint32_t hi0 = (uint32_t)(p0 >> 32), lo0 = (uint32_t)p0;
    const uint32_t hi1 = (uint32_t)(p1 >> 32), lo1 = (uint32_t)p1;
    const uint32_t n0 = hi1 ^ c1 ^ k0;
    const uint32_t n1 = lo1;
    const uint32_t n2 = hi0 ^ c3 ^ k1;
    const uint32_t n3 = lo0;
    c0 = n0; c1 = n1; c2 = n2; c3 = n3;
  }
  out[0] = c0; out[1] = c1; out[2] = c2; out[3] = c3;
}

/* P4: u = (word>>8) * 2^-24 is exact in fp32; the affine map is ONE fp32 fma on both sides. */
extern "C" float orc_uniform_f32(uint32_t word, float lo, float hi) {
  const float u = (float)(word >> 8) * 5.9604644775390625e-08f;  // 2^-24
  const float span = hi - lo;                                    // fp32 rounding, as on the GPU
  return std::fmaf(u, span, lo);
}

/* P4: counter = (it, r, s, (kind<<31) | (k<<4) | blk), key = (seed_lo, seed_hi). */
extern "C" uint32_t orc_draw_word(uint64_t seed, uint32_t it, uint32_t r, uint32_t s,
                                  uint32_t kind, uint32_t k, uint32_t j) {
  const uint32_t blk = j >> 2;
  const uint32_t ctr[4] = {it, r, s, (kind << 31) | (k << 4) | blk};
  const uint32_t key[2] = {(uint32_t)(seed & 0xffffffffu), (uint32_t)(seed >> 32)};
  uint32_t out[4];
  orc_philox4x32_10(ctr, key, out);
  return out[j & 3];
}

/* Alg. 1 l.6 SampleStates; P3: uniform over the state box, angle dims over
 * [-pi_f, pi_f), a dim with infinite bounds (only legal with nn_weight 0) is sampled as 0. */
extern "C" void orc_sample_state(const orc_problem* P, uint64_t seed, uint32_t r, uint32_t it,
                                 uint32_t s, double* x) {
  const float pif = 3.14159274101257324f;  // (float)pi
  for (int d = 0; d < P->state_dim; ++d) {
    const uint32_t w = orc_draw_word(seed, it, r, s, 0u, 0u, (uint32_t)d);
    if (P->dim_kind[d] == ORC_DIM_ANGLE) {
      x[d] = (double)orc_uniform_f32(w, -pif, pif);
    } else if (std::isfinite(P->state_lo[d]) && std::isfinite(P->state_hi[d])) {
      x[d] = (double)orc_uniform_f32(w, (float)P->state_lo[d], (float)P->state_hi[d]);
    } else {
      x[d] = 0.0;
    }
  }
}

/* Alg. 1 l.8 SampleControls ("uniform distribution"); P7. */
extern "C" void orc_sample_control(const orc_problem* P, uint64_t seed, uint32_t r, uint32_t it,
                                   uint32_t s, uint32_t k, double* u) {
  for (int j = 0; j < P->control_dim; ++j) {
    const uint32_t w = orc_draw_word(seed, it, r, s, 1u, k, (uint32_t)j);
    double v = (double)orc_uniform_f32(w, (float)P->control_lo[j], (float)P->control_hi[j]);
    if (v < P->control_lo[j]) v = P->control_lo[j];  // clamp (north_star (3)); no-op by construction
    if (v > P->control_hi[j]) v = P->control_hi[j];
    u[j] = v;
  }
}

/* ------------------------------------------------------------------------------------------ */
extern "C" double orc_wrap_pi(double a) {  // -> [-pi, pi)
  double w = a - 2.0 * kPi * std::floor((a + kPi) / (2.0 * kPi));
  if (w >= kPi) w -= 2.0 * kPi;  // guard the rounding case floor() lands one short
  if (w < -kPi) w += 2.0 * kPi;
  return w;
}

/* P5: d^2 = sum_d w_d * delta_d^2, delta wrapped on angle dims ("distance calculations",
 * PAPER.md:142; subset of dims via zero weights). */
extern "C" double orc_dist2(const orc_problem* P, const double* a, const double* b) {
  double acc = 0.0;
  for (int d = 0; d < P->state_dim; ++d) {
    double delta = a[d] - b[d];
    if (P->dim_kind[d] == ORC_DIM_ANGLE) delta = orc_wrap_pi(delta);
    acc += P->nn_weight[d] * delta * delta;
  }
  return acc;
}

/* Alg. 1 l.7 NearestNeighbor: brute force over the snapshot [0,n), ascending
 * scan, replace on strict '<' => lowest index on ties (P6). */
extern "C" int64_t orc_nearest(const orc_problem* P, const double* states, int64_t n,
                               const double* q, double* d2_out) {
  int64_t best = -1;
  double best_d2 = kInf;
  for (int64_t i = 0; i < n; ++i) {
    const double d2 = orc_dist2(P, q, states + i * P->state_dim);
    if (d2 < best_d2) {
      best_d2 = d2;
      best = i;
    }
  }
  if (d2_out) *d2_out = best_d2;
  return best;
}

/* Eq. (1) xdot = f(x,u) for the model families of the configs and of PAPER.md Sec. V. */
extern "C" void orc_f(const orc_problem* P, const double* x, const double* u, double* xd) {
  switch (P->dynamics_id) {
    case ORC_DYN_DOUBLE_INTEGRATOR: {  // [p, pdot], control = accelerations
      const int pd = P->pos_dim;
      for (int i = 0; i < pd; ++i) {
        xd[i] = x[pd + i];
        xd[pd + i] = u[i];
      }
      break;
    }
    case ORC_DYN_UNICYCLE2: {  // [x,y,theta,v,omega], control [a, alpha]
      xd[0] = x[3] * std::cos(x[2]);
      xd[1] = x[3] * std::sin(x[2]);
      xd[2] = x[4];
      xd[3] = u[0];
      xd[4] = u[1];
      break;
    }
    case ORC_DYN_QUADROTOR: {
      // Reading Q: state [p(3), v(3) world, (phi,theta,psi) ZYX Euler, (p,q,r) body rates],
      // control (T, tau_x, tau_y, tau_z); BASELINE.json config 4 layout (PAPER.md:174 names
      // the same 12 quantities with body-frame velocities; the config's layout binds).
      const double m = P->dyn_params[0], Ixx = P->dyn_params[1], Iyy = P->dyn_params[2],
                   Izz = P->dyn_params[3], g = P->dyn_params[4];
      const double phi = x[6], th = x[7], psi = x[8];
      const double p = x[9], q = x[10], r = x[11];
      const double sphi = std::sin(phi), cphi = std::cos(phi);
      const double sth = std::sin(th), cth = std::cos(th);
      const double spsi = std::sin(psi), cpsi = std::cos(psi);
      const double tth = sth / cth;
      const double a = u[0] / m;
      xd[0] = x[3]; xd[1] = x[4]; xd[2] = x[5];
      xd[3] = a * (cpsi * sth * cphi + spsi * sphi);  // (T/m) R e3
      xd[4] = a * (spsi * sth * cphi - cpsi * sphi);
      xd[5] = a * (cth * cphi) - g;
      xd[6] = p + sphi * tth * q + cphi * tth * r;     // ZYX Euler-rate kinematics
      xd[7] = cphi * q - sphi * r;
      xd[8] = (sphi * q + cphi * r) / cth;
      xd[9] = (u[1] - (Izz - Iyy) * q * r) / Ixx;      // I wdot = tau - w x (I w)
      xd[10] = (u[2] - (Ixx - Izz) * p * r) / Iyy;
      xd[11] = (u[3] - (Iyy - Ixx) * p * q) / Izz;
      break;
    }
    case ORC_DYN_DUBINS_AIRPLANE: {
      // state [x, y, z, phi (yaw), theta (pitch), v], control [phi_dot, theta_dot, v_dot].
      // The paper gives no equations; reading (P33): the velocity vector has magnitude v along
      // the heading given by yaw and pitch.
      const double yaw = x[3], pitch = x[4], v = x[5];
      xd[0] = v * std::cos(pitch) * std::cos(yaw);
      xd[1] = v * std::cos(pitch) * std::sin(yaw);
      xd[2] = v * std::sin(pitch);
      xd[3] = u[0];
      xd[4] = u[1];
      xd[5] = u[2];
      break;
    }
    case ORC_DYN_UNICYCLE1: {  // [x, y, theta], control [v, omega]
      xd[0] = u[0] * std::cos(x[2]);
      xd[1] = u[0] * std::sin(x[2]);
      xd[2] = u[1];
      break;
    }
    case ORC_DYN_QUADROTOR_BODY: {
      // state [x,y,z, phi,theta,psi, u,v,w, p,q,r] with linear and angular velocities in the body
      // frame, control [T, tau_x, tau_y, tau_z].  Rigid body in body axes (reading P34: phi roll, theta pitch,
      // psi yaw, ZYX; thrust along body z):  p_dot = R v_b;  v_b_dot = -w x v_b + R^T (0,0,-g) + (0,0,T/m).
      const double m = P->dyn_params[0], Ixx = P->dyn_params[1], Iyy = P->dyn_params[2],
                   Izz = P->dyn_params[3], g = P->dyn_params[4];
      const double phi = x[3], th = x[4], psi = x[5];
      const double ub = x[6], vb = x[7], wb = x[8], p = x[9], q = x[10], r = x[11];
      const double sphi = std::sin(phi), cphi = std::cos(phi), sth = std::sin(th), cth = std::cos(th),
                   spsi = std::sin(psi), cpsi = std::cos(psi);
      const double R[3][3] = {
          {cpsi * cth, cpsi * sth * sphi - spsi * cphi, cpsi * sth * cphi + spsi * sphi},
          {spsi * cth, spsi * sth * sphi + cpsi * cphi, spsi * sth * cphi - cpsi * sphi},
          {-sth, cth * sphi, cth * cphi}};
      for (int i = 0; i < 3; ++i) xd[i] = R[i][0] * ub + R[i][1] * vb + R[i][2] * wb;
      xd[3] = p + sphi * (sth / cth) * q + cphi * (sth / cth) * r;
      xd[4] = cphi * q - sphi * r;
      xd[5] = (sphi * q + cphi * r) / cth;
      // -w x v_b = (r v - q w, p w - r u, q u - p v);  R^T (0,0,-g) = -g * third row of R
      xd[6] = r * vb - q * wb - g * R[2][0];
      xd[7] = p * wb - r * ub - g * R[2][1];
      xd[8] = q * ub - p * vb - g * R[2][2] + u[0] / m;
      xd[9] = (u[1] - (Izz - Iyy) * q * r) / Ixx;
      xd[10] = (u[2] - (Ixx - Izz) * p * r) / Iyy;
      xd[11] = (u[3] - (Iyy - Ixx) * p * q) / Izz;
      break;
    }
    case ORC_DYN_ACROBOT: {
      // state [theta1, theta2, theta1_dot, theta2_dot], two-link pendulum actuated at the elbow,
      // control = elbow torque.  The paper prints no equations (it points to DynoBench); reading P35:
      // the planar double pendulum of rigid links from Lagrange's equations, theta1 measured from the downward
      // vertical, theta2 relative to link 1, I1 and I2 about each link's centre of mass:
      //   T = 1/2 qd^T D(q) qd,   V = -m1 g lc1 cos(th1) - m2 g (l1 cos(th1) + lc2 cos(th1 + th2))
      //   D(q) qdd + c(q, qd) = -dV/dq + (0, tau)
      const double m1 = P->dyn_params[0], m2 = P->dyn_params[1], l1 = P->dyn_params[2], lc1 = P->dyn_params[3],
                   lc2 = P->dyn_params[4], I1 = P->dyn_params[5], I2 = P->dyn_params[6], g = P->dyn_params[7];
      const double th1 = x[0], th2 = x[1], w1 = x[2], w2 = x[3];
      const double c2 = std::cos(th2), s2 = std::sin(th2);
      const double d11 = I1 + I2 + m1 * lc1 * lc1 + m2 * (l1 * l1 + lc2 * lc2 + 2.0 * l1 * lc2 * c2);
      const double d12 = I2 + m2 * (lc2 * lc2 + l1 * lc2 * c2);
      const double d22 = I2 + m2 * lc2 * lc2;
      const double hh = m2 * l1 * lc2 * s2;
      const double cor1 = -hh * (2.0 * w1 * w2 + w2 * w2);  // Coriolis / centrifugal terms c(q, qd)
      const double cor2 = hh * w1 * w1;
      const double grav1 = -(m1 * lc1 + m2 * l1) * g * std::sin(th1) - m2 * lc2 * g * std::sin(th1 + th2);  // -dV/dth1
      const double grav2 = -m2 * lc2 * g * std::sin(th1 + th2);                                              // -dV/dth2
      const double r1 = grav1 - cor1;
      const double r2 = grav2 - cor2 + u[0];
      const double det = d11 * d22 - d12 * d12;
      xd[0] = w1;
      xd[1] = w2;
      xd[2] = (d22 * r1 - d12 * r2) / det;
      xd[3] = (d11 * r2 - d12 * r1) / det;
      break;
    }
    default:
      for (int d = 0; d < P->state_dim; ++d) xd[d] = 0.0;
  }
}

/* One fixed step (PAPER.md:144 "fourth-order Runge-Kutta", :158 fixed dt); P9: classical RK4,
 * or explicit forward Euler when the config says so (config 1). */
extern "C" void orc_step(const orc_problem* P, const double* x, const double* u, double* xn) {
  const int D = P->state_dim;
  const double h = P->dt;
  double k1[16], k2[16], k3[16], k4[16], t[16];
  if (P->integrator == ORC_INT_EULER) {
    orc_f(P, x, u, k1);
    for (int d = 0; d < D; ++d) xn[d] = x[d] + h * k1[d];
    return;
  }
  orc_f(P, x, u, k1);
  for (int d = 0; d < D; ++d) t[d] = x[d] + 0.5 * h * k1[d];
  orc_f(P, t, u, k2);
  for (int d = 0; d < D; ++d) t[d] = x[d] + 0.5 * h * k2[d];
  orc_f(P, t, u, k3);
  for (int d = 0; d < D; ++d) t[d] = x[d] + h * k3[d];
  orc_f(P, t, u, k4);
  for (int d = 0; d < D; ++d) xn[d] = x[d] + (h / 6.0) * (k1[d] + 2.0 * k2[d] + 2.0 * k3[d] + k4[d]);
}

/* P11: point robot; circle / vertical cylinder: collision iff |p_xy - c| <= r; AABB: iff
 * lo <= p <= hi on every position axis.  Closed sets.  Returns min over obstacles of a margin
 * that is > 0 iff outside: circle |p-c| - r; box: max over axes of max(lo-p, p-hi). */
extern "C" double orc_obstacle_margin(const orc_problem* P, const double* x) {
  double m = kInf;
  for (int o = 0; o < P->n_obstacles; ++o) {
    double mo;
    if (P->obstacle_type == ORC_OBS_AABB) {
      const int pd = P->pos_dim;
      const double* lo = P->obstacles + (size_t)o * 2 * pd;
      const double* hi = lo + pd;
      mo = -kInf;
      for (int a = 0; a < pd; ++a) {
        const double ma = std::fmax(lo[a] - x[a], x[a] - hi[a]);
        if (ma > mo) mo = ma;
      }
    } else {  // CIRCLE2D and ZCYLINDER: (cx, cy, r), distance in the xy plane
      const double* c = P->obstacles + (size_t)o * 3;
      const double dx = x[0] - c[0], dy = x[1] - c[1];
      mo = std::sqrt(dx * dx + dy * dy) - c[2];
    }
    if (mo < m) m = mo;
  }
  return m;
}

/* P12: closed box on every non-angle dim with a finite bound; >= 0 iff inside. */
extern "C" double orc_bounds_margin(const orc_problem* P, const double* x) {
  double m = kInf;
  for (int d = 0; d < P->state_dim; ++d) {
    if (P->dim_kind[d] == ORC_DIM_ANGLE) continue;  // P13: angles are never bounds-tested
    if (std::isfinite(P->state_lo[d])) m = std::fmin(m, x[d] - P->state_lo[d]);
    if (std::isfinite(P->state_hi[d])) m = std::fmin(m, P->state_hi[d] - x[d]);
  }
  return m;
}

/* Alg. 1 l.9 Propagate + l.12 CollisionFree: S steps with the control
 * held, validity at each step-end state j=1..S (P8, P10); angles wrapped once at the end (P13). */
extern "C" int32_t orc_propagate(const orc_problem* P, const double* x0, const double* u,
                                 double* x_new, int32_t* first_bad_step, double* min_margin,
                                 double* edge_cost) {
  const int D = P->state_dim;
  double x[16], xn[16];
  for (int d = 0; d < D; ++d) x[d] = x0[d];
  int32_t flags = ORC_F_VALID | ORC_F_INBOUNDS | ORC_F_COLLFREE;
  int32_t first_bad = 0;
  double mm = kInf, length = 0.0;
  for (int j = 1; j <= P->steps_per_edge; ++j) {
    orc_step(P, x, u, xn);
    double seg = 0.0;
    for (int a = 0; a < P->pos_dim; ++a) seg += (xn[a] - x[a]) * (xn[a] - x[a]);
    length += std::sqrt(seg);
    for (int d = 0; d < D; ++d) x[d] = xn[d];
    const double bm = orc_bounds_margin(P, x);
    const double om = orc_obstacle_margin(P, x);
    if (bm < 0.0) flags &= ~(ORC_F_INBOUNDS | ORC_F_VALID);
    if (om <= 0.0) flags &= ~(ORC_F_COLLFREE | ORC_F_VALID);
    if (!(flags & ORC_F_VALID) && first_bad == 0) first_bad = j;
    mm = std::fmin(mm, std::fmin(std::fabs(bm), std::fabs(om)));
  }
  for (int d = 0; d < D; ++d)
    x_new[d] = (P->dim_kind[d] == ORC_DIM_ANGLE) ? orc_wrap_pi(x[d]) : x[d];
  if (first_bad_step) *first_bad_step = first_bad;
  if (min_margin) *min_margin = mm;
  if (edge_cost)  // P14: J = T, or path length over the step-end positions
    *edge_cost = (P->cost_mode == ORC_COST_PATH_LENGTH) ? length
                                                         : (double)P->steps_per_edge * P->dt;
  return flags;
}

/* Euclidean distance to the goal centre over the goal dims (default: the position dims), the difference wrapped on
 * angle dims (P18; Acrobot's goal lives in angle space, "swing-up"). */
static double goal_distance(const orc_problem* P, const double* x) {
  double s = 0.0;
  const int ng = P->goal_n_dims > 0 ? P->goal_n_dims : P->pos_dim;
  for (int i = 0; i < ng; ++i) {
    const int d = P->goal_n_dims > 0 ? P->goal_dims[i] : i;
    double delta = x[d] - P->goal_center[i];
    if (P->dim_kind[d] == ORC_DIM_ANGLE) delta = orc_wrap_pi(delta);
    s += delta * delta;
  }
  return std::sqrt(s);
}

/* P15: h(x) = max(0, |p - p_goal| - r_goal) / v_cap  ("Euclidean heuristic",
 * made admissible for the duration cost as BASELINE.json demands). */
extern "C" double orc_heuristic(const orc_problem* P, const double* x) {
  if (std::isinf(P->heuristic_speed)) return 0.0;
  return std::fmax(0.0, goal_distance(P, x) - P->goal_radius) / P->heuristic_speed;
}

/* P18: x_new in X_goal (Alg. 1 l.14): position ball (closed) and optional heading tolerance. */
extern "C" int32_t orc_in_goal(const orc_problem* P, const double* x, double* margin) {
  const double dpos = goal_distance(P, x);
  int32_t in = dpos <= P->goal_radius;
  double mg = std::fabs(dpos - P->goal_radius);
  if (P->goal_angle_dim >= 0) {
    const double da = std::fabs(orc_wrap_pi(x[P->goal_angle_dim] - P->goal_angle));
    in = in && (da <= P->goal_angle_tol);
    mg = std::fmin(mg, std::fabs(da - P->goal_angle_tol));
  }
  if (margin) *margin = mg;
  return in;
}

/* Alg. 1 l.4: T <- {(x_init, empty, 0)}; P24: parent[0] = -1, action[0] = 0. */
extern "C" void orc_tree_reset(const orc_problem* P, orc_tree* T) {
  for (int d = 0; d < P->state_dim; ++d) T->states[d] = P->start[d];
  for (int j = 0; j < P->control_dim; ++j) T->actions[j] = 0.0;
  T->parents[0] = -1;
  T->costs[0] = 0.0;
  T->n = 1;
}

/* Alg. 1 l.6-17, one trip of the inner loop, in the listing's order. */
extern "C" int32_t orc_expand_iteration(const orc_problem* P, orc_tree* T, uint64_t seed,
                                        uint32_t r, uint32_t it, int32_t B, int32_t K,
                                        double c_best, orc_iter_debug* dbg) {
  const int D = P->state_dim, m = P->control_dim;
  const int64_t n_snapshot = T->n;  // frozen snapshot for every query of the batch
  const int64_t BK = (int64_t)B * K;
  std::vector<double> x_rand((size_t)B * D), xs((size_t)BK * D), us((size_t)BK * m), cs(BK);
  std::vector<int64_t> nn(B);
  std::vector<int32_t> flags(BK);
  using clk = std::chrono::steady_clock;  // timing only (bench.py's cpu_baseline reports per-phase shares)
  const auto t_begin = clk::now();

  // l.6  X_rand <- SampleStates(B)
  for (int s = 0; s < B; ++s) orc_sample_state(P, seed, r, it, (uint32_t)s, &x_rand[(size_t)s * D]);
  // l.7  X_near <- NearestNeighbor(T, X_rand)
  for (int s = 0; s < B; ++s) {
    double d2;
    nn[s] = orc_nearest(P, T->states, n_snapshot, &x_rand[(size_t)s * D], &d2);
    if (dbg && dbg->nn_idx) dbg->nn_idx[s] = (int32_t)nn[s];
    if (dbg && dbg->nn_d2) dbg->nn_d2[s] = d2;
  }
  if (dbg && dbg->x_rand) std::memcpy(dbg->x_rand, x_rand.data(), sizeof(double) * B * D);
  const auto t_nn = clk::now();
  // l.8  U <- SampleControls(B, K);  l.9  X_new, C_new <- Propagate(X_near, U, dt)
  for (int s = 0; s < B; ++s) {
    for (int k = 0; k < K; ++k) {
      const int64_t c = (int64_t)s * K + k;
      orc_sample_control(P, seed, r, it, (uint32_t)s, (uint32_t)k, &us[(size_t)c * m]);
      double mm, ec;
      int32_t fb;
      int32_t f = orc_propagate(P, T->states + nn[s] * D, &us[(size_t)c * m], &xs[(size_t)c * D],
                                &fb, &mm, &ec);
      cs[c] = T->costs[nn[s]] + ec;  // additivity of J
      // l.11  c_new + h(x_new) < c_best  (strict, P16);  l.12 CollisionFree;  P17: the AND
      const double fcost = cs[c] + orc_heuristic(P, &xs[(size_t)c * D]);
      if (fcost < c_best) f |= ORC_F_NOTPRUNED;
      double gm;
      const int32_t ing = orc_in_goal(P, &xs[(size_t)c * D], &gm);
      if ((f & ORC_F_VALID) && (f & ORC_F_NOTPRUNED) && ing) f |= ORC_F_GOAL;
      flags[c] = f;
      if (dbg && dbg->child_margin) dbg->child_margin[c] = mm;
      if (dbg && dbg->prune_margin) dbg->prune_margin[c] = std::fabs(fcost - c_best);
      if (dbg && dbg->goal_margin) dbg->goal_margin[c] = gm;
    }
  }
  const auto t_prop = clk::now();
  // l.13  T <- T u {(x_new, u, c_new)} in ascending child index while n < cap (P20)
  int64_t inserted = 0, goal_node = -1;
  double goal_cost = kInf;
  for (int64_t c = 0; c < BK; ++c) {
    const bool keep = (flags[c] & ORC_F_VALID) && (flags[c] & ORC_F_NOTPRUNED);
    if (!keep || T->n >= T->capacity) continue;
    const int64_t i = T->n++;
    for (int d = 0; d < D; ++d) T->states[i * D + d] = xs[(size_t)c * D + d];
    for (int j = 0; j < m; ++j) T->actions[i * m + j] = us[(size_t)c * m + j];
    T->parents[i] = (int32_t)nn[c / K];
    T->costs[i] = cs[c];
    flags[c] |= ORC_F_INSERTED;
    ++inserted;
    // l.14-15: goal winner = min c_new, ties -> lowest child index (P19)
    if ((flags[c] & ORC_F_GOAL) && cs[c] < goal_cost) {
      goal_cost = cs[c];
      goal_node = i;
    }
  }
  if (dbg) {
    if (dbg->child_state) std::memcpy(dbg->child_state, xs.data(), sizeof(double) * BK * D);
    if (dbg->child_ctrl) std::memcpy(dbg->child_ctrl, us.data(), sizeof(double) * BK * m);
    if (dbg->child_cost) std::memcpy(dbg->child_cost, cs.data(), sizeof(double) * BK);
    if (dbg->child_flags) std::memcpy(dbg->child_flags, flags.data(), sizeof(int32_t) * BK);
    dbg->n_inserted = inserted;
    dbg->goal_node = goal_node;
    dbg->new_c_best = goal_node >= 0 ? goal_cost : c_best;
    const auto t_end = clk::now();
    dbg->phase_ms[0] = std::chrono::duration<double, std::milli>(t_nn - t_begin).count();
    dbg->phase_ms[1] = std::chrono::duration<double, std::milli>(t_prop - t_nn).count();
    dbg->phase_ms[2] = std::chrono::duration<double, std::milli>(t_end - t_prop).count();
  }
  return goal_node >= 0 ? 1 : 0;
}

/* Alg. 1 l.16 ExtractPath: walk parents to the root, reverse. */
static int32_t extract_path(const orc_problem* P, const orc_tree* T, int64_t goal_node,
                            orc_plan_result* R) {
  int32_t len = 0;
  for (int64_t i = goal_node; i >= 0; i = T->parents[i]) ++len;
  R->path_len = len;
  if (len > R->path_capacity) return 1;
  const int D = P->state_dim, m = P->control_dim;
  int32_t pos = len - 1;
  for (int64_t i = goal_node; i >= 0; i = T->parents[i], --pos) {
    if (R->path_nodes) R->path_nodes[pos] = (int32_t)i;
    if (R->path_states)
      for (int d = 0; d < D; ++d) R->path_states[(size_t)pos * D + d] = T->states[i * D + d];
    if (R->path_controls && pos > 0)  // P25: action[i] produced node i from parent[i]
      for (int j = 0; j < m; ++j) R->path_controls[(size_t)(pos - 1) * m + j] = T->actions[i * m + j];
  }
  return 0;
}

/* Alg. 1 l.1-3,18: AO-x meta loop (c_best monotone). */
extern "C" int32_t orc_plan(const orc_problem* P, const orc_plan_opts* O, orc_tree* T,
                            orc_plan_result* R) {
  using clk = std::chrono::steady_clock;
  const auto t0 = clk::now();
  auto ms_since = [&]() { return std::chrono::duration<double, std::milli>(clk::now() - t0).count(); };
  const int64_t BK = (int64_t)O->B * O->K;
  int64_t max_iters = O->max_iters_per_replan;
  if (max_iters <= 0) max_iters = std::max<int64_t>(32, O->tree_capacity / BK);  // P21
  double c_best = kInf;  // l.1
  if (O->initial_cost_bound > 0.0 && std::isfinite(O->initial_cost_bound)) c_best = O->initial_cost_bound;
  R->path_len = 0;       // l.2
  R->outcome = 0;
  R->cost = kInf;
  R->iterations = R->children = R->inserted = 0;
  R->replans_run = R->replans_solved = 0;
  R->first_solution_ms = -1.0;
  R->phase_ms[0] = R->phase_ms[1] = R->phase_ms[2] = 0.0;
  int32_t status = 0;
  for (int32_t r = 0; r < O->n_replans; ++r) {  // l.3 (P22: a failed replan counts against R)
    if (O->time_budget_ms > 0 && ms_since() >= O->time_budget_ms) break;
    orc_tree_reset(P, T);  // l.4
    int64_t it = 0;
    bool solved = false;
    for (; it < max_iters; ++it) {  // l.5
      orc_iter_debug dbg;
      std::memset(&dbg, 0, sizeof(dbg));
      const int32_t goal = orc_expand_iteration(P, T, O->seed, (uint32_t)r, (uint32_t)it, O->B,
                                                O->K, c_best, &dbg);
      R->iterations += 1;
      R->children += BK;
      R->inserted += dbg.n_inserted;
      for (int ph = 0; ph < 3; ++ph) R->phase_ms[ph] += dbg.phase_ms[ph];
      if (goal) {  // l.14-17
        c_best = dbg.new_c_best;
        if (extract_path(P, T, dbg.goal_node, R)) status = 1;
        R->outcome = 1;
        R->cost = c_best;
        solved = true;
        ++it;
        break;
      }
      if (T->n >= T->capacity) { ++it; break; }  // P20: full tree ends the replan
      if (O->time_budget_ms > 0 && ms_since() >= O->time_budget_ms) { ++it; break; }
    }
    if (solved) {
      R->replans_solved += 1;
      if (R->first_solution_ms < 0) R->first_solution_ms = ms_since();
    }
    if (R->replan_cost) R->replan_cost[r] = c_best;
    if (R->replan_nodes) R->replan_nodes[r] = T->n;
    if (R->replan_iters) R->replan_iters[r] = it;
    R->replans_run += 1;
  }
  R->total_ms = ms_since();
  return status;  // l.18 return sigma*
}

extern "C" int32_t orc_validate_plan(const orc_problem* P, const double* path_states,
                                     const double* path_controls, int32_t path_len,
                                     int32_t per_edge, double* cost_out, double* max_state_err) {
  const int D = P->state_dim, m = P->control_dim;
  double x[16], xn[16];
  for (int d = 0; d < D; ++d) x[d] = P->start[d];
  double err = 0.0, cost = 0.0;
  int32_t code = 0;
  for (int d = 0; d < D; ++d) err = std::fmax(err, std::fabs(x[d] - path_states[d]));
  for (int e = 0; e + 1 < path_len; ++e) {
    const double* u = path_controls + (size_t)e * m;
    for (int j = 0; j < m; ++j)
      if (u[j] < P->control_lo[j] || u[j] > P->control_hi[j]) code = code ? code : 3;
    int32_t fb;
    double mm, ec;
    if (per_edge)  // restart every edge from the stored node (tree invariant form)
      for (int d = 0; d < D; ++d) x[d] = path_states[(size_t)e * D + d];
    const int32_t f = orc_propagate(P, x, u, xn, &fb, &mm, &ec);
    if (!(f & ORC_F_VALID)) code = code ? code : 1;
    cost += ec;
    for (int d = 0; d < D; ++d) {
      x[d] = xn[d];
      double de = x[d] - path_states[(size_t)(e + 1) * D + d];
      if (P->dim_kind[d] == ORC_DIM_ANGLE) de = orc_wrap_pi(de);
      err = std::fmax(err, std::fabs(de));
    }
  }
  if (!orc_in_goal(P, x, nullptr)) code = code ? code : 2;
  if (cost_out) *cost_out = cost;
  if (max_state_err) *max_state_err = err;
  return code;
}
