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
enum DynKind { DYN_DI2 = 0, DYN_DI3 = 1, DYN_UNI2 = 2, DYN_QUAD = 3 };
enum ObsKind { OBS_CIRCLE = 0, OBS_BOX = 1 };

template <int DYN> struct DynTraits;
template <> struct DynTraits<DYN_DI2> { static constexpr int D = 4, M = 2, PD = 2, DP = 4, ANGLE = -1; };
template <> struct DynTraits<DYN_DI3> { static constexpr int D = 6, M = 3, PD = 3, DP = 8, ANGLE = -1; };
template <> struct DynTraits<DYN_UNI2> { static constexpr int D = 5, M = 2, PD = 2, DP = 8, ANGLE = 2; };
template <> struct DynTraits<DYN_QUAD> { static constexpr int D = 12, M = 4, PD = 3, DP = 12, ANGLE = 8; };

// Problem constants, passed by value in the kernel parameter block.
struct DevProblem {
  float lo[kMaxD], hi[kMaxD];          // state box (+-inf = unbounded)
  float w[kMaxD];                      // NN weights
  float samp_lo[kMaxD], samp_span[kMaxD];  // sampling: fmaf(u, span, lo), span = fl32(hi - lo)
  float ulo[kMaxM], uhi[kMaxM], uspan[kMaxM];
  float start[kMaxD];
  float goal[3];
  float goal_r, goal_angle, goal_angle_tol;
  int goal_angle_dim;
  float dyn[8];                        // quadrotor: m, Ixx, Iyy, Izz, g
  float dt;
  int S;
  int integrator;                      // 0 Euler, 1 RK4
  int cost_mode;                       // 0 duration, 1 path length
  float inv_hspeed;                    // 1 / heuristic_speed (0 if +inf)
  int unit_weights;                    // all w == 1: skip the weight multiply in the NN scan
  int n_obs;
  const float* obstacles;              // DEVICE, rows of OBS_STRIDE floats
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
  } else {
    const float m = pb.dyn[0], Ixx = pb.dyn[1], Iyy = pb.dyn[2], Izz = pb.dyn[3], g = pb.dyn[4];
    float sphi, cphi, sth, cth, spsi, cpsi;
    sincosf(x[6], &sphi, &cphi);
    sincosf(x[7], &sth, &cth);
    sincosf(x[8], &spsi, &cpsi);
    const float p = x[9], q = x[10], r = x[11];
    const float icth = 1.0f / cth;
    const float tth = sth * icth;
    const float a = u[0] / m;
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
    xd[9] = (u[1] - (Izz - Iyy) * q * r) / Ixx;
    xd[10] = (u[2] - (Ixx - Izz) * p * r) / Iyy;
    xd[11] = (u[3] - (Iyy - Ixx) * p * q) / Izz;
  }
}

// One fixed step of dt: forward Euler or classical RK4 (P9).
template <int DYN>
__device__ __forceinline__ void dyn_step(const DevProblem& pb, float (&x)[DynTraits<DYN>::D],
                                         const float (&u)[DynTraits<DYN>::M]) {
  constexpr int D = DynTraits<DYN>::D;
  const float h = pb.dt;
  float k[D], t[D], acc[D];
  dyn_f<DYN>(pb, x, u, k);
  if (pb.integrator == 0) {
#pragma unroll
    for (int d = 0; d < D; ++d) x[d] = fmaf(h, k[d], x[d]);
    return;
  }
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
  for (int d = 0; d < D; ++d) x[d] = fmaf(h * (1.0f / 6.0f), acc[d] + k[d], x[d]);
}

// ---- validity ("validity checked at each step"; P10-P13) ----------------
template <int DYN>
__device__ __forceinline__ bool in_bounds(const DevProblem& pb, const float (&x)[DynTraits<DYN>::D]) {
  bool ok = true;
#pragma unroll
  for (int d = 0; d < DynTraits<DYN>::D; ++d)
    if (d != DynTraits<DYN>::ANGLE) ok = ok && (x[d] >= pb.lo[d]) && (x[d] <= pb.hi[d]);
  return ok;
}

template <int OBS, int PD> struct ObsStride { static constexpr int value = (OBS == OBS_CIRCLE) ? 4 : 8; };

// obstacles in shared memory: circle rows (cx, cy, r*r, pad); box rows (lo[3], pad, hi[3], pad)
// (2D boxes carry lo/hi z = -inf/+inf).  Closed sets.  Lanes of a child group may each take a
// strided subset (first, step).
template <int OBS, int PD>
__device__ __forceinline__ bool collision_free(const float* __restrict__ sm_obs, int n_obs,
                                               const float* pos, int first, int step) {
  bool hit = false;
  if constexpr (OBS == OBS_CIRCLE) {
    const float4* o4 = reinterpret_cast<const float4*>(sm_obs);
#pragma unroll 4
    for (int o = first; o < n_obs; o += step) {
      const float4 c = o4[o];
      const float dx = pos[0] - c.x, dy = pos[1] - c.y;
      hit = hit || (fmaf(dx, dx, dy * dy) <= c.z);
    }
  } else {
    const float4* o4 = reinterpret_cast<const float4*>(sm_obs);
    const float pz = (PD == 3) ? pos[2] : 0.0f;
#pragma unroll 4
    for (int o = first; o < n_obs; o += step) {
      const float4 lo = o4[2 * o], hi = o4[2 * o + 1];
      const bool in = (pos[0] >= lo.x) && (pos[0] <= hi.x) && (pos[1] >= lo.y) && (pos[1] <= hi.y) &&
                      (pz >= lo.z) && (pz <= hi.z);
      hit = hit || in;
    }
  }
  return !hit;
}

template <int PD>
__device__ __forceinline__ float goal_dist(const DevProblem& pb, const float* x) {
  float s = 0.0f;
#pragma unroll
  for (int a = 0; a < PD; ++a) { const float d = x[a] - pb.goal[a]; s = fmaf(d, d, s); }
  return sqrtf(s);
}

}  // namespace pakr
