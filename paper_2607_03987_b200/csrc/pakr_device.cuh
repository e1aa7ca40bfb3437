// pakr_device.cuh -- device building blocks of the PAKR expansion iteration (sm_100a).
//
// Philox sampler (reading P4), dynamics f(x,u) (Eq. (1), :172, :208,
// BASELINE.json config 4), fixed-step Euler / RK4, per-step validity,
// heuristic and goal test (Alg. 1 l.11,14).  fp32 throughout; the state of a child
// lives in registers for its whole edge.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace pakr {

constexpr int kMaxD = 12;
constexpr int kMaxM = 4;
constexpr float kPiF = 3.14159274101257324f;   // (float)pi
constexpr float kTwoPiF = 6.28318548202514648f;

// ---- compile-time description of a dynamics model -------------------------------------------
enum DynKind { DYN_DI2 = 0, DYN_DI3 = 1, DYN_UNI2 = 2, DYN_QUAD = 3, DYN_DA = 4, DYN_UNI1 = 5, DYN_QUADB = 6, DYN_ACRO = 7 };
enum ObsKind { OBS_CIRCLE = 0, OBS_BOX = 1 };

// ANGLES: bit d set = state dim d is an angle (wrapped to [-pi, pi), never bounds-tested; P13)
template <int DYN> struct DynTraits;
template <> struct DynTraits<DYN_DI2> { static constexpr int D = 4, M = 2, PD = 2, DP = 4; static constexpr unsigned ANGLES = 0u; };
template <> struct DynTraits<DYN_DI3> { static constexpr int D = 6, M = 3, PD = 3, DP = 8; static constexpr unsigned ANGLES = 0u; };
template <> struct DynTraits<DYN_UNI2> { static constexpr int D = 5, M = 2, PD = 2, DP = 8; static constexpr unsigned ANGLES = 1u << 2; };
template <> struct DynTraits<DYN_QUAD> { static constexpr int D = 12, M = 4, PD = 3, DP = 12; static constexpr unsigned ANGLES = 1u << 8; };
template <> struct DynTraits<DYN_DA> { static constexpr int D = 6, M = 3, PD = 3, DP = 8; static constexpr unsigned ANGLES = 1u << 3; };
template <> struct DynTraits<DYN_UNI1> { static constexpr int D = 3, M = 2, PD = 2, DP = 4; static constexpr unsigned ANGLES = 1u << 2; };
template <> struct DynTraits<DYN_QUADB> { static constexpr int D = 12, M = 4, PD = 3, DP = 12; static constexpr unsigned ANGLES = 1u << 5; };
template <> struct DynTraits<DYN_ACRO> { static constexpr int D = 4, M = 1, PD = 2, DP = 4; static constexpr unsigned ANGLES = 3u; };
template <int DYN> __host__ __device__ constexpr bool is_angle(int d) { return (DynTraits<DYN>::ANGLES >> d) & 1u; }

// Problem constants, passed by value in the kernel parameter block.
struct DevProblem {
  float lo[kMaxD], hi[kMaxD];          // state box (+-inf = unbounded)
  float w[kMaxD];                      // NN weights
  float samp_lo[kMaxD], samp_span[kMaxD];  // sampling: fmaf(u, span, lo), span = fl32(hi - lo)
  float ulo[kMaxM], uhi[kMaxM], uspan[kMaxM];
  float start[kMaxD];
  float goal_c[kMaxD], goal_m[kMaxD];  // goal ball: centre per state dim, mask 1 on the goal dims (0 elsewhere)
  float goal_r, goal_angle, goal_angle_tol;
  int goal_angle_dim;
  float dyn[12];                       // quadrotor: m, Ixx, Iyy, Izz, g, then 1/m, 1/Ixx, 1/Iyy, 1/Izz
                                       // Acrobot: the five lumped constants of dyn_f (set by the host)
  float dt;
  int S;
  int integrator;                      // 0 Euler, 1 RK4
  int cost_mode;                       // 0 duration, 1 path length
  float inv_hspeed;                    // 1 / heuristic_speed (0 if +inf)
  int unit_weights;                    // all w == 1: skip the weight multiply in the NN scan
  int n_obs;
  const float* obstacles;              // DEVICE, rows of OBS_STRIDE floats
  // obstacle broad phase: uniform grid over the position box, CSR lists of obstacle ids per cell
  int grid_on;                         // 0: test every obstacle
  int gdim[3];                         // cells per axis (gdim[2] == 1 for circle / cylinder fields)
  float gorg[3], ginv[3];              // cell(x) = clamp(floor((x - gorg) * ginv), 0, gdim - 1)
  int g_cells, g_list;                 // number of cells, total list entries
  const uint32_t* grid_cells;          // DEVICE [g_cells]: cell words, see cell_margin()
  const uint16_t* grid_list;           // DEVICE [g_list] obstacle ids
  // tensor-core NN filter (pakr_nn_filter.cuh): feature u_d = (x_d - f_ctr[d]) * f_scale[d], f_scale = sqrt(w)
  float f_ctr[kMaxD], f_scale[kMaxD];
  float f_qn_ang;                      // 2 * sum of the angle dims' weights
  float f_eps;                         // |approximate key - true key| <= f_eps * sum_i |c_i u_i| (host: 2^-17)
  // NN index: Morton key layout over the weighted state box (pakr_api.cu: idx_key_layout)
  float idx_scale[kMaxD];              // quantised coordinate = floor((x - lo) * scale), 0 .. 2^bits - 1
  uint8_t idx_bits[kMaxD];             // key bits of every dimension (0: not keyed)
  uint8_t idx_pos[kMaxD][16];          // key position of bit b of the dimension's quantised coordinate
};

// ---- Philox4x32-10 ---------------------------------------------------------------------------
__device__ __forceinline__ uint4 philox4x32_10(uint4 c, uint2 k) {
#pragma unroll
  for (int i = 0; i < 10; ++i) {
    const uint32_t hi0 = __umulhi(0xD2511F53u, c.x), lo0 = 0xD2511F53u * c.x;
    const uint32_t hi1 = __umulhi(0xCD9E8D57u, c.z), lo1 = 0xCD9E8D57u * c.z;
    c = make_uint4(hi1 ^ c.y ^ k.x, lo1, hi0 ^ c.w ^ k.y, lo0);
    k.x += 0x9E3779B9u;
    k.y += 0xBB67AE85u;
  }
  return c;
}

// counter = (it, r, s, (kind<<31) | (k<<4) | blk), key = seed (P4)
__device__ __forceinline__ uint4 draw_block(uint64_t seed, uint32_t it, uint32_t r, uint32_t s,
                                            uint32_t kind, uint32_t k, uint32_t blk) {
  return philox4x32_10(make_uint4(it, r, s, (kind << 31) | (k << 4) | blk),
                       make_uint2((uint32_t)seed, (uint32_t)(seed >> 32)));
}

__device__ __forceinline__ float u01(uint32_t w) { return (float)(w >> 8) * 5.9604644775390625e-08f; }

// Alg. 1 l.6: one sampled state, D draws (word j&3 of block j>>2).
template <int D>
__device__ __forceinline__ void sample_state(const DevProblem& pb, uint64_t seed, uint32_t r,
                                             uint32_t it, uint32_t s, float (&x)[D]) {
#pragma unroll
  for (int blk = 0; blk < (D + 3) / 4; ++blk) {
    const uint4 v = draw_block(seed, it, r, s, 0u, 0u, blk);
    const uint32_t wd[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
    for (int j = 0; j < 4; ++j) {
      const int d = blk * 4 + j;
      if (d < D) x[d] = fmaf(u01(wd[j]), pb.samp_span[d], pb.samp_lo[d]);
    }
  }
}

// Alg. 1 l.8: one control vector (M <= 4 draws: one Philox block), clamped to the control box.
template <int M>
__device__ __forceinline__ void sample_control(const DevProblem& pb, uint64_t seed, uint32_t r,
                                               uint32_t it, uint32_t s, uint32_t k, float (&u)[M]) {
  const uint4 v = draw_block(seed, it, r, s, 1u, k, 0u);
  const uint32_t wd[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
  for (int j = 0; j < M; ++j) {
    const float t = fmaf(u01(wd[j]), pb.uspan[j], pb.ulo[j]);
    u[j] = fminf(fmaxf(t, pb.ulo[j]), pb.uhi[j]);
  }
}

// ---- angles ----------------------------------------------------------------------------------
__device__ __forceinline__ float wrap_pi(float a) {  // -> [-pi, pi)
  float w = a - kTwoPiF * floorf((a + kPiF) * (1.0f / kTwoPiF));
  if (w >= kPiF) w -= kTwoPiF;
  if (w < -kPiF) w += kTwoPiF;
  return w;
}
// |wrap(a - b)| for a, b in [-pi, pi]: min(|a-b|, 2pi - |a-b|); exact whenever no wrap happens
__device__ __forceinline__ float angle_absdiff(float a, float b) {
  const float d = fabsf(a - b);
  return fminf(d, kTwoPiF - d);
}

// ---- dynamics xdot = f(x, u) -----------------------------------------------------------------
template <int DYN>
__device__ __forceinline__ void dyn_f(const DevProblem& pb, const float (&x)[DynTraits<DYN>::D],
                                      const float (&u)[DynTraits<DYN>::M],
                                      float (&xd)[DynTraits<DYN>::D]) {
  if constexpr (DYN == DYN_DI2 || DYN == DYN_DI3) {
    constexpr int PD = DynTraits<DYN>::PD;
#pragma unroll
    for (int i = 0; i < PD; ++i) {
      xd[i] = x[PD + i];
      xd[PD + i] = u[i];
    }
  } else if constexpr (DYN == DYN_UNI2) {
    float s, c;
    sincosf(x[2], &s, &c);
    xd[0] = x[3] * c;
    xd[1] = x[3] * s;
    xd[2] = x[4];
    xd[3] = u[0];
    xd[4] = u[1];
  } else if constexpr (DYN == DYN_DA) {  // Dubins airplane [x,y,z,yaw,pitch,v], u = (yaw rate, pitch rate, accel)
    float sy, cy, sp, cp;
    sincosf(x[3], &sy, &cy);
    sincosf(x[4], &sp, &cp);
    xd[0] = x[5] * cp * cy;
    xd[1] = x[5] * cp * sy;
    xd[2] = x[5] * sp;
    xd[3] = u[0];
    xd[4] = u[1];
    xd[5] = u[2];
  } else if constexpr (DYN == DYN_UNI1) {  // first-order unicycle [x,y,theta], u = (v, omega)
    float s, c;
    sincosf(x[2], &s, &c);
    xd[0] = u[0] * c;
    xd[1] = u[0] * s;
    xd[2] = u[1];
  } else if constexpr (DYN == DYN_QUADB) {
    // [x,y,z, phi,theta,psi, u,v,w (body), p,q,r (body)], control (T, tau).  Same rigid body as
    // DYN_QUAD written in body axes: pdot = R v_b, v_b dot = -w x v_b + R^T (0,0,-g) + (0,0,T/m).
    const float Ixx = pb.dyn[1], Iyy = pb.dyn[2], Izz = pb.dyn[3], g = pb.dyn[4];
    float sphi, cphi, sth, cth, spsi, cpsi;
    __sincosf(x[3], &sphi, &cphi);
    __sincosf(x[4], &sth, &cth);
    __sincosf(x[5] - kTwoPiF * rintf(x[5] * (1.0f / kTwoPiF)), &spsi, &cpsi);
    const float ub = x[6], vb = x[7], wb = x[8];
    const float p = x[9], q = x[10], r = x[11];
    const float icth = __frcp_rn(cth);
    const float tth = sth * icth;
    // rows of R = Rz(psi) Ry(theta) Rx(phi)
    xd[0] = cpsi * cth * ub + (cpsi * sth * sphi - spsi * cphi) * vb + (cpsi * sth * cphi + spsi * sphi) * wb;
    xd[1] = spsi * cth * ub + (spsi * sth * sphi + cpsi * cphi) * vb + (spsi * sth * cphi - cpsi * sphi) * wb;
    xd[2] = -sth * ub + cth * sphi * vb + cth * cphi * wb;
    const float sq_cr = sphi * q + cphi * r;
    xd[3] = p + tth * sq_cr;
    xd[4] = cphi * q - sphi * r;
    xd[5] = sq_cr * icth;
    xd[6] = r * vb - q * wb + g * sth;
    xd[7] = p * wb - r * ub - g * sphi * cth;
    xd[8] = q * ub - p * vb - g * cphi * cth + u[0] * pb.dyn[5];
    xd[9] = (u[1] - (Izz - Iyy) * q * r) * pb.dyn[6];
    xd[10] = (u[2] - (Ixx - Izz) * p * r) * pb.dyn[7];
    xd[11] = (u[3] - (Iyy - Ixx) * p * q) * pb.dyn[8];
  } else if constexpr (DYN == DYN_ACRO) {
    // PAPER.md:209 (P35): D(q) qdd + c(q, qd) = -dV/dq + (0, tau), theta1 from the downward vertical.
    // Host-lumped constants: A = I1 + I2 + m1 lc1^2 + m2 (l1^2 + lc2^2), Bc = m2 l1 lc2, C = I2 + m2 lc2^2,
    // Ga = (m1 lc1 + m2 l1) g, Gb = m2 lc2 g.
    const float A = pb.dyn[0], Bc = pb.dyn[1], C = pb.dyn[2], Ga = pb.dyn[3], Gb = pb.dyn[4];
    float s2, c2;
    sincosf(x[1], &s2, &c2);
    const float s1 = sinf(x[0]), s12 = sinf(x[0] + x[1]);
    const float w1 = x[2], w2 = x[3];
    const float d11 = fmaf(2.0f * Bc, c2, A), d12 = fmaf(Bc, c2, C), d22 = C;
    const float hh = Bc * s2;
    const float r1 = fmaf(hh * w2, fmaf(2.0f, w1, w2), -fmaf(Ga, s1, Gb * s12));  // -dV/dth1 - c1
    const float r2 = u[0] - fmaf(hh * w1, w1, Gb * s12);                         // tau - dV/dth2 - c2
    const float idet = __frcp_rn(fmaf(d11, d22, -d12 * d12));
    xd[0] = w1;
    xd[1] = w2;
    xd[2] = (d22 * r1 - d12 * r2) * idet;
    xd[3] = (d11 * r2 - d12 * r1) * idet;
  } else {
    const float Ixx = pb.dyn[1], Iyy = pb.dyn[2], Izz = pb.dyn[3], g = pb.dyn[4];
    float sphi, cphi, sth, cth, spsi, cpsi;
#ifndef PAKR_ACCURATE_SINCOS
    // MUFU-based sin/cos (abs error <= 2^-21.4 on [-pi, pi]; roll and pitch are bounded by the state box, yaw is
    // folded into [-pi, pi] first): 2.2x faster quadrotor edges than sincosf, whose inlined slow path also evicts
    // the edge loop from the instruction cache.  State error vs the fp64 oracle stays ~1e-5 (tolerance 1e-4).
    __sincosf(x[6], &sphi, &cphi);
    __sincosf(x[7], &sth, &cth);
    __sincosf(x[8] - kTwoPiF * rintf(x[8] * (1.0f / kTwoPiF)), &spsi, &cpsi);
#else
    sincosf(x[6], &sphi, &cphi);
    sincosf(x[7], &sth, &cth);
    sincosf(x[8], &spsi, &cpsi);
#endif
    const float p = x[9], q = x[10], r = x[11];
    const float icth = __frcp_rn(cth);
    const float tth = sth * icth;
    const float a = u[0] * pb.dyn[5];  // 1/m
    xd[0] = x[3];
    xd[1] = x[4];
    xd[2] = x[5];
    xd[3] = a * (cpsi * sth * cphi + spsi * sphi);
    xd[4] = a * (spsi * sth * cphi - cpsi * sphi);
    xd[5] = a * (cth * cphi) - g;
    const float sq_cr = sphi * q + cphi * r;
    xd[6] = p + tth * sq_cr;
    xd[7] = cphi * q - sphi * r;
    xd[8] = sq_cr * icth;
    xd[9] = (u[1] - (Izz - Iyy) * q * r) * pb.dyn[6];   // 1/Ixx, 1/Iyy, 1/Izz (set by the host)
    xd[10] = (u[2] - (Ixx - Izz) * p * r) * pb.dyn[7];
    xd[11] = (u[3] - (Iyy - Ixx) * p * q) * pb.dyn[8];
  }
}

// One fixed step of dt: forward Euler or classical RK4 (P9).
// RK4 is a rolled loop over the four stages (t = x + a_s h k, acc += b_s k with a = 0, 1/2, 1/2, 1 and
// b = 1, 2, 2, 1): ONE inlined copy of f instead of four keeps the quadrotor edge inside the instruction cache.
// Every operation rounds exactly like the unrolled textbook form (a_0 = 0 and b = 1 cases are exact).
template <int DYN>
__device__ __forceinline__ void dyn_step(const DevProblem& pb, float (&x)[DynTraits<DYN>::D],
                                         const float (&u)[DynTraits<DYN>::M]) {
  constexpr int D = DynTraits<DYN>::D;
  const float h = pb.dt;
  float k[D], t[D], acc[D];
  if (pb.integrator == 0) {
    dyn_f<DYN>(pb, x, u, k);
#pragma unroll
    for (int d = 0; d < D; ++d) x[d] = fmaf(h, k[d], x[d]);
    return;
  }
#pragma unroll
  for (int d = 0; d < D; ++d) { k[d] = 0.0f; acc[d] = 0.0f; }
  constexpr bool kRoll = (DYN == DYN_QUAD) || (DYN == DYN_QUADB);  // measured: rolling slows the unicycle (less ILP), f of the others is tiny
#pragma unroll 1
  for (int s = 0; s < (kRoll ? 4 : 1); ++s) {
    if constexpr (kRoll) {
      const float a = (s == 0) ? 0.0f : (s == 3) ? h : 0.5f * h;
      const float b = (s == 1 || s == 2) ? 2.0f : 1.0f;
#pragma unroll
      for (int d = 0; d < D; ++d) t[d] = fmaf(a, k[d], x[d]);
      dyn_f<DYN>(pb, t, u, k);
#pragma unroll
      for (int d = 0; d < D; ++d) acc[d] = fmaf(b, k[d], acc[d]);
    } else {
      dyn_f<DYN>(pb, x, u, k);
#pragma unroll
      for (int d = 0; d < D; ++d) { acc[d] = k[d]; t[d] = fmaf(0.5f * h, k[d], x[d]); }
      dyn_f<DYN>(pb, t, u, k);
#pragma unroll
      for (int d = 0; d < D; ++d) { acc[d] = fmaf(2.0f, k[d], acc[d]); t[d] = fmaf(0.5f * h, k[d], x[d]); }
      dyn_f<DYN>(pb, t, u, k);
#pragma unroll
      for (int d = 0; d < D; ++d) { acc[d] = fmaf(2.0f, k[d], acc[d]); t[d] = fmaf(h, k[d], x[d]); }
      dyn_f<DYN>(pb, t, u, k);
#pragma unroll
      for (int d = 0; d < D; ++d) acc[d] = acc[d] + k[d];
    }
  }
#pragma unroll
  for (int d = 0; d < D; ++d) x[d] = fmaf(h * (1.0f / 6.0f), acc[d], x[d]);
}

// ---- validity ("validity checked at each step"; P10-P13) ----------------
// Both tests return a margin whose SIGN is exact (a difference of two fp32 values has the exact
// sign), so "margin >= 0" / "margin > 0" decide exactly like the comparisons they replace, while
// the min/max trees keep the per-step dependency chain short and free of predicate registers.

// >= 0 iff lo <= x <= hi on every non-angle dim (closed box, P12)
template <int DYN>
__device__ __forceinline__ float bounds_margin(const DevProblem& pb, const float (&x)[DynTraits<DYN>::D]) {
  float m0 = __int_as_float(0x7f800000), m1 = m0;
#pragma unroll
  for (int d = 0; d < DynTraits<DYN>::D; ++d)
    if (!is_angle<DYN>(d)) {
      m0 = fminf(m0, x[d] - pb.lo[d]);
      m1 = fminf(m1, pb.hi[d] - x[d]);
    }
  return fminf(m0, m1);
}

// obstacles in shared memory: circle rows (cx, cy, r*r, pad); box rows (lo[3], pad, hi[3], pad)
// (2D boxes carry lo/hi z = -inf/+inf).  > 0 iff the position is outside every obstacle of the
// strided subset first, first+step, ... (closed sets, P11).  circle: |p-c|^2 - r^2; box: max over
// axes of max(lo - p, p - hi).
template <int OBS, int PD>
__device__ __forceinline__ float obstacle_margin(const float* __restrict__ sm_obs, int n_obs,
                                                 const float* pos, int first, int step) {
  const float4* o4 = reinterpret_cast<const float4*>(sm_obs);
  float m0 = __int_as_float(0x7f800000), m1 = m0;
  if constexpr (OBS == OBS_CIRCLE) {
    int o = first;
#pragma unroll 4
    for (; o + step < n_obs; o += 2 * step) {
      const float4 a = o4[o], b = o4[o + step];
      const float ax = pos[0] - a.x, ay = pos[1] - a.y, bx = pos[0] - b.x, by = pos[1] - b.y;
      m0 = fminf(m0, fmaf(ax, ax, ay * ay) - a.z);
      m1 = fminf(m1, fmaf(bx, bx, by * by) - b.z);
    }
    if (o < n_obs) {
      const float4 a = o4[o];
      const float ax = pos[0] - a.x, ay = pos[1] - a.y;
      m0 = fminf(m0, fmaf(ax, ax, ay * ay) - a.z);
    }
  } else {
    const float pz = (PD == 3) ? pos[2] : 0.0f;
    int o = first;
#pragma unroll 4
    for (; o + step < n_obs; o += 2 * step) {
      const float4 alo = o4[2 * o], ahi = o4[2 * o + 1], blo = o4[2 * (o + step)], bhi = o4[2 * (o + step) + 1];
      const float ma = fmaxf(fmaxf(fmaxf(alo.x - pos[0], pos[0] - ahi.x), fmaxf(alo.y - pos[1], pos[1] - ahi.y)),
                             fmaxf(alo.z - pz, pz - ahi.z));
      const float mb = fmaxf(fmaxf(fmaxf(blo.x - pos[0], pos[0] - bhi.x), fmaxf(blo.y - pos[1], pos[1] - bhi.y)),
                             fmaxf(blo.z - pz, pz - bhi.z));
      m0 = fminf(m0, ma);
      m1 = fminf(m1, mb);
    }
    if (o < n_obs) {
      const float4 alo = o4[2 * o], ahi = o4[2 * o + 1];
      const float ma = fmaxf(fmaxf(fmaxf(alo.x - pos[0], pos[0] - ahi.x), fmaxf(alo.y - pos[1], pos[1] - ahi.y)),
                             fmaxf(alo.z - pz, pz - ahi.z));
      m0 = fminf(m0, ma);
    }
  }
  return fminf(m0, m1);
}

// Margin of one obstacle (same formulas as obstacle_margin above).
template <int OBS, int PD>
__device__ __forceinline__ float one_obstacle_margin(const float4* __restrict__ o4, int o, const float* pos) {
  if constexpr (OBS == OBS_CIRCLE) {
    const float4 a = o4[o];
    const float ax = pos[0] - a.x, ay = pos[1] - a.y;
    return fmaf(ax, ax, ay * ay) - a.z;
  } else {
    const float pz = (PD == 3) ? pos[2] : 0.0f;
    const float4 alo = o4[2 * o], ahi = o4[2 * o + 1];
    return fmaxf(fmaxf(fmaxf(alo.x - pos[0], pos[0] - ahi.x), fmaxf(alo.y - pos[1], pos[1] - ahi.y)),
                 fmaxf(alo.z - pz, pz - ahi.z));
  }
}

// Broad phase (exact): only the obstacles registered in the grid cell of `pos` can contain it, because the
// host registers an obstacle in every cell its (slightly inflated) bounding box touches and cell() is
// monotone per axis; positions outside the box clamp into the border cells, whose lists hold everything
// that sticks out of the box.  The SIGN of the resulting margin equals that of the full scan.
// Cell word: bits 0-7 count; count <= 2: ids inline in bits 8-19 and 20-31; else bits 8-31 = list offset.
template <int OBS, int PD>
__device__ __forceinline__ int grid_cell(const DevProblem& pb, const float* pos) {
  constexpr int GD = (OBS == OBS_CIRCLE) ? 2 : PD;  // circles / vertical cylinders: xy grid
  int cell = 0, mul = 1;
#pragma unroll
  for (int a = 0; a < GD; ++a) {
    int c = __float2int_rd((pos[a] - pb.gorg[a]) * pb.ginv[a]);
    c = min(max(c, 0), pb.gdim[a] - 1);
    cell += c * mul;
    mul *= pb.gdim[a];
  }
  return cell;
}

template <int OBS, int PD>
__device__ __forceinline__ float cell_margin(uint32_t hdr, const uint16_t* __restrict__ sm_list,
                                             const float* __restrict__ sm_obs, const float* pos) {
  const float4* o4 = reinterpret_cast<const float4*>(sm_obs);
  const int cnt = (int)(hdr & 0xffu);
  float m = __int_as_float(0x7f800000);
  if (cnt == 0) return m;
  if (cnt <= 2) {
    m = one_obstacle_margin<OBS, PD>(o4, (int)((hdr >> 8) & 0xfffu), pos);
    if (cnt == 2) m = fminf(m, one_obstacle_margin<OBS, PD>(o4, (int)(hdr >> 20), pos));
    return m;
  }
  const uint16_t* lst = sm_list + (hdr >> 8);
  for (int k = 0; k < cnt; ++k) m = fminf(m, one_obstacle_margin<OBS, PD>(o4, (int)lst[k], pos));
  return m;
}

// Distance to the goal centre over the goal dims (mask 1; a masked-out dim adds an exact +0), wrapped on angle dims.
// `x` has its angle dims already wrapped to [-pi, pi).
template <int DYN>
__device__ __forceinline__ float goal_dist(const DevProblem& pb, const float (&x)[DynTraits<DYN>::D]) {
  float s = 0.0f;
#pragma unroll
  for (int d = 0; d < DynTraits<DYN>::D; ++d) {
    float e = x[d] - pb.goal_c[d];
    if (is_angle<DYN>(d)) e = wrap_pi(e);
    s = fmaf(e * pb.goal_m[d], e, s);
  }
  return sqrtf(s);
}

}  // namespace pakr
