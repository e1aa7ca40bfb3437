// pakr_nn_filter.cuh -- tensor-core coarse filter of the nearest-neighbour scan.
//
// Alg. 1 l.7 asks for argmin_p d2(q, p) over the frozen tree snapshot for B queries: B*n squared
// distances of D = 3..12 dimensions.  On CUDA cores that costs 2D FMA-pipe lane-ops per pair.  Here the bilinear part of
//     d2(q, p) = |v|^2 + |u|^2 - 2 v.u,      u = sqrt(w) (p - centre), v = sqrt(w) (q - centre)
// (an angle dim contributes w (2 - 2 cos q cos p - 2 sin q sin p) <= w delta^2, a LOWER bound of its wrapped term) is
// one small GEMM, [queries x K] x [K x rows], on the tensor cores:
//   * every tree row has a FILTER ROW of K = 32 or 48 halves: the features u (real dims, cos / sin of angle dims, and
//     |u_real|^2) split into fp16 hi + lo, laid out as [u_hi | u_lo | u_hi]; a query's coefficient vector c = (-2 v, 1)
//     is laid out as [c_hi | c_hi | c_lo], so one K-long dot product gives c_hi.u_hi + c_hi.u_lo + c_lo.u_hi = c.u up
//     to ~2^-21 relative: the approximate key a(p) = d2_lower(q, p) - qn,  qn = |v_real|^2 + 2 sum_angle w.
//   * phase 1 (nn_filter_scan): a warp holds 64 queries as A fragments and streams its row range through TMA tiles;
//     per 8 rows one conflict-free LDS.128 yields the B fragments, 4 x K/16 mma.sync.m16n8k16 (fp32 accumulate) give 512
//     approximate keys in registers and 16 FMNMX fold them into running minima: the MINIMUM approximate key of every
//     (query, row range) goes to `chunkmin`.  No threshold, no divergence.
//   * phase 2 (nn_filter_refine), after a barrier: one warp per query rescans EXACTLY (the scan tiers' dist2 arithmetic
//     on the fp32 tree rows, same (d2 bits, lowest index) key) the range with the smallest minimum, which gives a real
//     upper bound UB, then every other range whose minimum is <= UB - qn + band, tightening UB as it goes.
// Exactness: the true nearest row p* has a(p*) <= d2(p*) - qn + band <= UB - qn + band at all times, so its range is
// always rescanned; ranges are rescanned with the exact arithmetic, so the result is bit-identical to the brute-force
// scan tiers (ties included).  band = 2^-17 * S with S >= sum |c_i u_i| of the pair, bounded per query by
// 3 V^2 + 4 V sqrt(UB) + UB (V = |v|; rows that matter have |u| <= V + sqrt(UB)); 2^-17 covers the fp16 hi/lo
// truncation (3 * 2^-22 S), the tensor core's fp32 accumulation (K * 2^-24 S) and the fp32 feature arithmetic with a
// margin of ~5, plus an absolute floor of 2^-24 (2 + 8 V + 4 R + R^2), R = V + sqrt(UB), for the fp16 subnormal range
// (see nn_filter_refine).
//
// Why mma.sync and not tcgen05 here: the epilogue must look at EVERY accumulator (a min over the row axis), and K is
// only 32..48.  tcgen05.mma would finish a 128 x 256 x 32 tile in ~256 cycles but draining its 128 KB of accumulators
// through tcgen05.ld takes >= 2048 cycles at the measured 64 B/clk/SM (B300_MICROARCH.md "TMEM"); mma.sync leaves the
// accumulators in registers where the FMNMX fold is free, and sustains 750 MAC/clk/SM with the fold (measured,
// profiles/r02_fp32_peak.md) = 23 (K = 32) / 15 (K = 48) pairs/clk/SM against 10.7 / 3.6 for the FFMA2 scan.
#pragma once
#include <cuda_fp16.h>

namespace pakr {

constexpr int kFilterMinRows = 4096;   // shorter row ranges go through the exact scan ...
constexpr long long kFilterMinWork = 400000000ll;  // ... and so do scans of fewer than B*n*D lane-pairs (~40 us exact)
constexpr int kFilterGiveUp = 24;      // the exact scan takes over once phase 2 rescans more than 1/24 of the pairs
constexpr int kFilterMaxChunks = 4104; // chunkmin row stride (chunks per query <= 4096, stored four at a time)
constexpr int kFilterQ = 64;           // queries per warp (4 m-tiles of 16)

__host__ __device__ constexpr int popcount_c(unsigned v) { return v ? (int)(v & 1u) + popcount_c(v >> 1) : 0; }

template <int DYN> struct FilterCfg {
  using T = DynTraits<DYN>;
  static constexpr int NANG = popcount_c(T::ANGLES);
  static constexpr int NREAL = T::D - NANG;
  static constexpr int NF = NREAL + 2 * NANG + 1;        // features: real dims, (cos, sin) per angle dim, |u_real|^2
  static constexpr int K = (3 * NF <= 32) ? 32 : 48;     // halves per filter row
  static constexpr int KS = K / 16;                      // mma k-steps
  static constexpr int ROW_BYTES = K * 2;
  static constexpr int TILE_ROWS = (K == 32) ? 64 : 40;  // rows per 4 KB TMA tile buffer (a multiple of 8)
  static_assert(3 * NF <= 48, "filter row too long");
};

struct FilterPlan {
  int G;     // query groups of 64
  int CH;    // rows per chunk: the granularity of chunkmin and of the exact rescoring (a whole number of TMA tiles)
  int NC;    // chunks over the scanned rows
  int CPR;   // chunks per work range (1, 2, 4, 8 or 16)
  int Reff;  // work ranges per query group
  int U;     // work units of phase 1: (query group, row range)
};
// The same plan indexes chunkmin in both phases.  Chunks are as small as one TMA tile (64 / 40 rows) while that keeps
// NC <= 4096, so a candidate costs 64 exact distances, not a whole range.
template <int DYN>
__host__ __device__ __forceinline__ FilterPlan filter_plan(int B, int n, int W) {
  FilterPlan f;
  f.G = (B + kFilterQ - 1) / kFilterQ;
  f.CH = FilterCfg<DYN>::TILE_ROWS;
  while ((n + f.CH - 1) / f.CH > 4096) f.CH *= 2;
  f.NC = (n + f.CH - 1) / f.CH;
  int R0 = W / f.G;  // ranges per group that fill the machine once
  if (R0 < 8) R0 = 8;
  const int cpr = f.NC / R0;
  f.CPR = cpr >= 16 ? 16 : cpr >= 8 ? 8 : cpr >= 4 ? 4 : cpr >= 2 ? 2 : 1;
  f.Reff = (f.NC + f.CPR - 1) / f.CPR;
  f.U = f.G * f.Reff;
  return f;
}

// features of a state (a tree row or a query)
template <int DYN>
__device__ __forceinline__ void filter_features(const DevProblem& pb, const float (&x)[DynTraits<DYN>::D],
                                                float (&f)[FilterCfg<DYN>::NF]) {
  using C = FilterCfg<DYN>;
  int sr = 0, sa = C::NREAL;  // compile-time after unrolling
  float pn = 0.0f;
#pragma unroll
  for (int d = 0; d < DynTraits<DYN>::D; ++d) {
    if (is_angle<DYN>(d)) {
      float s, c;
      sincosf(x[d], &s, &c);
      f[sa++] = pb.f_scale[d] * c;
      f[sa++] = pb.f_scale[d] * s;
    } else {
      const float u = (x[d] - pb.f_ctr[d]) * pb.f_scale[d];
      f[sr++] = u;
      pn = fmaf(u, u, pn);
    }
  }
  f[C::NF - 1] = pn;
}

__device__ __forceinline__ void split_half(float v, __half& hi, __half& lo) {
  hi = __float2half_rn(v);
  lo = __float2half_rn(v - __half2float(hi));
}
__device__ __forceinline__ uint32_t pack_half2(__half a, __half b) {
  return (uint32_t)__half_as_ushort(a) | ((uint32_t)__half_as_ushort(b) << 16);
}

// Stores the filter row of features f.  K order [u_hi | u_lo | u_hi | 0]; storage order: the 2*KS words thread t
// (t = lane & 3) of an mma needs as B fragments are contiguous -- word (t, j = 2 ks + r) holds K indices
// ks*16 + 8r + 2t, +1 -- so that 8 consecutive rows are one conflict-free LDS.128 / 3 x LDS.64 per lane.
template <int DYN>
__device__ __forceinline__ void filter_store_row(__half* frow, size_t row, const float (&f)[FilterCfg<DYN>::NF]) {
  using C = FilterCfg<DYN>;
  __half kv[C::K];
#pragma unroll
  for (int i = 0; i < C::K; ++i) kv[i] = __ushort_as_half(0);
#pragma unroll
  for (int i = 0; i < C::NF; ++i) {
    __half hi, lo;
    split_half(f[i], hi, lo);
    kv[i] = hi;
    kv[C::NF + i] = lo;
    kv[2 * C::NF + i] = hi;
  }
  uint32_t w[C::K / 2];
#pragma unroll
  for (int t = 0; t < 4; ++t) {
#pragma unroll
    for (int j = 0; j < 2 * C::KS; ++j) {
      const int kidx = (j >> 1) * 16 + 8 * (j & 1) + 2 * t;
      w[t * 2 * C::KS + j] = pack_half2(kv[kidx], kv[kidx + 1]);
    }
  }
  uint4* dst = reinterpret_cast<uint4*>(frow + row * C::K);
#pragma unroll
  for (int v = 0; v < C::K / 8; ++v) dst[v] = make_uint4(w[4 * v], w[4 * v + 1], w[4 * v + 2], w[4 * v + 3]);
}

template <int DYN>
__device__ __forceinline__ void filter_write_row(const DevProblem& pb, __half* frow, size_t row,
                                                 const float (&x)[DynTraits<DYN>::D]) {
  float f[FilterCfg<DYN>::NF];
  filter_features<DYN>(pb, x, f);
  filter_store_row<DYN>(frow, row, f);
}
// a row no query can be near: |u|^2 = 60000 (the largest round fp16 value below overflow), everything else 0
template <int DYN>
__device__ __forceinline__ void filter_write_sentinel(__half* frow, size_t row) {
  float f[FilterCfg<DYN>::NF];
#pragma unroll
  for (int i = 0; i < FilterCfg<DYN>::NF; ++i) f[i] = 0.0f;
  f[FilterCfg<DYN>::NF - 1] = 60000.0f;
  filter_store_row<DYN>(frow, row, f);
}

// coefficient vector of a query, natural K order [c_hi | c_hi | c_lo | 0], c = (-2 v, 1)
template <int DYN>
__device__ __forceinline__ void filter_query_kvec(const DevProblem& pb, const float (&q)[DynTraits<DYN>::D], __half* dst) {
  using C = FilterCfg<DYN>;
  float f[C::NF];
  filter_features<DYN>(pb, q, f);
  __half kv[C::K];
#pragma unroll
  for (int i = 0; i < C::K; ++i) kv[i] = __ushort_as_half(0);
#pragma unroll
  for (int i = 0; i < C::NF; ++i) {
    const float c = (i == C::NF - 1) ? 1.0f : -2.0f * f[i];
    __half hi, lo;
    split_half(c, hi, lo);
    kv[i] = hi;
    kv[C::NF + i] = hi;
    kv[2 * C::NF + i] = lo;
  }
  uint32_t* d32 = reinterpret_cast<uint32_t*>(dst);
#pragma unroll
  for (int i = 0; i < C::K / 2; ++i) d32[i] = pack_half2(kv[2 * i], kv[2 * i + 1]);
}

__device__ __forceinline__ void mma_f16_16816(float (&c)[4], const uint32_t (&a)[4], uint32_t b0, uint32_t b1) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b0), "r"(b1));
}

// ---- phase 1: minimum approximate key of every (query, chunk of rows) -> chunkmin[query][chunk] ------------------
// Rows [nbeg, nend), queries of iteration `it`.  CTAs vb = 0..vbcount-1 take part (CTA-uniform call).
// sm_qk: 128 * K halves (the coefficient vectors of the <= 2 query groups a CTA round touches);
// sm_cm: kWarps * 4 * 64 floats (a warp's chunk minima of one range, stored as one float4 per query).
template <int DYN>
__device__ __noinline__ void nn_filter_scan(const Params& P, int nbeg, int nend, uint32_t r, uint32_t it, int vb,
                                            int vbcount, const FilterPlan& fp, float* sm_tile, uint64_t* sm_bar,
                                            __half* sm_qk, float* sm_cm, uint32_t& par0, uint32_t& par1) {
  using C = FilterCfg<DYN>;
  constexpr int D = DynTraits<DYN>::D, K = C::K, KS = C::KS;
  constexpr int TG = C::TILE_ROWS / 8;             // 8-row groups per tile
  constexpr int TILE_BYTES = C::TILE_ROWS * C::ROW_BYTES;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int gq = lane >> 2, t4 = lane & 3;
  const int W = vbcount * kWarps;
  const float inf = __int_as_float(0x7f800000);
  unsigned char* tile_bytes = reinterpret_cast<unsigned char*>(sm_tile);
  float* my_cm = sm_cm + warp * (4 * kFilterQ);
  const int tiles_per_chunk = fp.CH / C::TILE_ROWS;
  for (int ub = vb * kWarps; ub < fp.U; ub += W) {
    const int u = ub + warp;
    const bool has = u < fp.U;
    const int g_lo = ub / fp.Reff, g_hi = min(fp.U - 1, ub + kWarps - 1) / fp.Reff;  // g_hi <= g_lo + 1 (Reff >= 8)
    const int g = has ? u / fp.Reff : g_lo, rr = has ? u - g * fp.Reff : 0;
    __syncthreads();  // the previous round's readers are done with sm_qk
    for (int t = threadIdx.x; t < (g_hi - g_lo + 1) * kFilterQ; t += kThreads) {
      float x[D];
      sample_state<D>(P.pb, P.seed, r, it, (uint32_t)min(g_lo * kFilterQ + t, P.B - 1), x);
      filter_query_kvec<DYN>(P.pb, x, sm_qk + (size_t)t * K);
    }
    __syncthreads();
    if (!has) continue;
    uint32_t a[4][KS][4];
    {
      const uint32_t* qw = reinterpret_cast<const uint32_t*>(sm_qk + (size_t)(g - g_lo) * kFilterQ * K);
#pragma unroll
      for (int mt = 0; mt < 4; ++mt) {
#pragma unroll
        for (int ks = 0; ks < KS; ++ks) {
          const int q0 = (mt * 16 + gq) * (K / 2), q1 = q0 + 8 * (K / 2), wb = ks * 8 + t4;
          a[mt][ks][0] = qw[q0 + wb];
          a[mt][ks][1] = qw[q1 + wb];
          a[mt][ks][2] = qw[q0 + wb + 4];
          a[mt][ks][3] = qw[q1 + wb + 4];
        }
      }
    }
    const int c_first = rr * fp.CPR;                              // first chunk of the range
    const int beg = nbeg + c_first * fp.CH, end = min(nend, beg + fp.CPR * fp.CH);
    const int groups = (end - beg + 7) >> 3;  // the last group may reach past `end`: extra rows only lower a minimum
    const int ntiles = (groups + TG - 1) / TG;
    const unsigned char* src = reinterpret_cast<const unsigned char*>(P.frow) + (size_t)beg * C::ROW_BYTES;
    for (int i = lane; i < 4 * kFilterQ; i += 32) my_cm[i] = inf;
    __syncwarp();
    if (lane == 0) {
      const uint32_t bytes = (uint32_t)min(TG, groups) * 8 * C::ROW_BYTES;
      mbar_expect_tx(&sm_bar[0], bytes);
      tma_load_1d(tile_bytes, src, bytes, &sm_bar[0]);
    }
    float m[4][2];
#pragma unroll
    for (int mt = 0; mt < 4; ++mt) m[mt][0] = m[mt][1] = inf;
    for (int t = 0; t < ntiles; ++t) {
      const int ng = min(TG, groups - t * TG);
      if (t + 1 < ntiles && lane == 0) {  // prefetch the next tile into the other buffer
        const int nb = (t + 1) & 1;
        const uint32_t bytes = (uint32_t)min(TG, groups - (t + 1) * TG) * 8 * C::ROW_BYTES;
        mbar_expect_tx(&sm_bar[nb], bytes);
        tma_load_1d(tile_bytes + nb * 4096, src + (size_t)(t + 1) * TILE_BYTES, bytes, &sm_bar[nb]);
      }
      if (t & 1) { mbar_wait(&sm_bar[1], par1); par1 ^= 1; }
      else { mbar_wait(&sm_bar[0], par0); par0 ^= 1; }
      const unsigned char* tp = tile_bytes + (t & 1) * 4096 + lane * (2 * KS * 4);
#pragma unroll 2
      for (int gi = 0; gi < ng; ++gi) {
        uint32_t b[KS][2];
        if constexpr (K == 32) {
          const uint4 w = *reinterpret_cast<const uint4*>(tp + gi * (8 * C::ROW_BYTES));
          b[0][0] = w.x; b[0][1] = w.y; b[1][0] = w.z; b[1][1] = w.w;
        } else {
          const uint2* p2 = reinterpret_cast<const uint2*>(tp + gi * (8 * C::ROW_BYTES));
#pragma unroll
          for (int ks = 0; ks < KS; ++ks) { const uint2 w = p2[ks]; b[ks][0] = w.x; b[ks][1] = w.y; }
        }
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
          float c[4] = {0.0f, 0.0f, 0.0f, 0.0f};
#pragma unroll
          for (int ks = 0; ks < KS; ++ks) mma_f16_16816(c, a[mt][ks], b[ks][0], b[ks][1]);
          m[mt][0] = fminf(m[mt][0], fminf(c[0], c[1]));  // query mt*16 + gq      against rows 2 t4, 2 t4 + 1
          m[mt][1] = fminf(m[mt][1], fminf(c[2], c[3]));  // query mt*16 + gq + 8
        }
      }
      __syncwarp();  // every lane is done with this buffer before lane 0 refills it
      if ((t + 1) % tiles_per_chunk == 0 || t + 1 == ntiles) {  // end of a chunk: fold the quad, park the minima
        const int j = t / tiles_per_chunk;
#pragma unroll
        for (int mt = 0; mt < 4; ++mt) {
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            float v = m[mt][h];
            v = fminf(v, __shfl_xor_sync(0xffffffffu, v, 1));
            v = fminf(v, __shfl_xor_sync(0xffffffffu, v, 2));
            if (t4 == 0) my_cm[(mt * 16 + gq + 8 * h) * 4 + (j & 3)] = v;
            m[mt][h] = inf;
          }
        }
        if ((j & 3) == 3 || t + 1 == ntiles) {
          // four chunk minima (or the range's CPR < 4) of every query in one store; slots past the last chunk hold
          // +inf and are never read
          __syncwarp();
#pragma unroll
          for (int h = 0; h < 2; ++h) {
            const int qi = lane + 32 * h, s = g * kFilterQ + qi;
            if (s < P.B) {
              float* dst = &P.chunkmin[(size_t)s * kFilterMaxChunks + c_first + (j & ~3)];  // c_first: a multiple of CPR
              if (fp.CPR >= 4) __stcg(reinterpret_cast<float4*>(dst), *reinterpret_cast<const float4*>(&my_cm[qi * 4]));
              else if (fp.CPR == 2) __stcg(reinterpret_cast<float2*>(dst), *reinterpret_cast<const float2*>(&my_cm[qi * 4]));
              else __stcg(dst, my_cm[qi * 4]);
            }
          }
          __syncwarp();
          for (int i = lane; i < 4 * kFilterQ; i += 32) my_cm[i] = inf;
          __syncwarp();
        }
      }
    }
  }
}

// exact (d2 bits, row) minimum of query q over tree rows [beg, end): the scan tiers' arithmetic and tie rule
template <int DYN, bool UNIT_W>
__device__ __forceinline__ unsigned long long filter_rescan(const Params& P, int beg, int end,
                                                            const float (&q)[DynTraits<DYN>::D]) {
  constexpr int DP = DynTraits<DYN>::DP;
  const int lane = threadIdx.x & 31;
  unsigned long long best = kKeyNone;
  for (int i = beg + lane; i < end; i += 32) {
    float p[DP];
    const float4* sp = reinterpret_cast<const float4*>(P.states + (size_t)i * DP);
#pragma unroll
    for (int v = 0; v < DP / 4; ++v) {
      const float4 a = __ldcg(sp + v);
      p[4 * v] = a.x; p[4 * v + 1] = a.y; p[4 * v + 2] = a.z; p[4 * v + 3] = a.w;
    }
    const float d2 = dist2<DYN, UNIT_W>(P.pb, q, p);
    if (d2 >= 0.0f)  // not NaN; ascending rows per lane + min over (bits, row): lowest index wins ties
      best = min(best, ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned)i);
  }
  return warp_min_key(best);
}

__device__ __forceinline__ unsigned float_orderable(float v) {  // monotone float -> uint (NaN sorts last)
  const unsigned b = __float_as_uint(v);
  if (v != v) return 0xffffffffu;
  return (b & 0x80000000u) ? ~b : (b | 0x80000000u);
}

// ---- phase 2: exact rescoring of the candidate chunks, one warp per query -------------------------------------------
// sm_list: kWarps * kFilterList ints (a warp's pending candidate chunks).
constexpr int kFilterList = 64;

template <int DYN, bool UNIT_W>
__device__ __noinline__ void nn_filter_refine(const Params& P, int nbeg, int nend, uint32_t r, uint32_t it,
                                              unsigned long long* key, int vb, int vbcount, const FilterPlan& fp,
                                              unsigned long long* rescored, int* sm_list) {
  using C = FilterCfg<DYN>;
  constexpr int D = DynTraits<DYN>::D, DP = DynTraits<DYN>::DP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int Wp = vbcount * kWarps;
  const float inf = __int_as_float(0x7f800000);
  int* list = sm_list + warp * kFilterList;
  int rows = 0;  // rows this warp rescanned (warp-uniform)
  for (int s = vb * kWarps + warp; s < P.B; s += Wp) {
    float q[D];
    sample_state<D>(P.pb, P.seed, r, it, (uint32_t)s, q);
    if (lane == 0 && P.dbg_x_rand && nbeg == 0) {
#pragma unroll
      for (int d = 0; d < DP; ++d) P.dbg_x_rand[(size_t)s * DP + d] = d < D ? q[d] : 0.0f;
    }
    float f[C::NF];
    filter_features<DYN>(P.pb, q, f);
    const float qn = f[C::NF - 1] + P.pb.f_qn_ang;
    // Rounding band of THIS query: |approximate - true key| <= eps * sum_i |c_i u_i| <= eps (|u|^2 + 2 |v| |u|) with
    // |u| <= |v| + sqrt(d2) for the rows that matter (d2 <= UB): eps (3 V^2 + 4 V sqrt(UB) + UB), V^2 = qn / ... >= |v|^2.
    // f_eps = 2^-17 carries the same margin over the nominal 2^-19.5 as the box-wide band did.
    // Absolute floor on top of the relative band: a feature or coefficient below 2^-3 has an fp16-SUBNORMAL lo half
    // (and below 2^-14 a subnormal hi half), whose rounding error is an absolute 2^-25 whatever the value.  That adds at
    // most 2^-25 (sum_i |c_i| + sum_i |u_i|) to |approximate - true key|, with sum |c_i| <= 1 + 2 sqrt(NF) V and, for the
    // rows that matter, sum |u_i| <= R^2 + sqrt(NF) R, R = V + sqrt(UB); sqrt(NF) < 4.  Taken with 2^-24.  It matters
    // for queries near the centre of the box and for state boxes much narrower than 1 in weighted units, where the
    // relative band alone shrinks below the subnormal spacing.
    const float v2 = f[C::NF - 1] + 0.5f * P.pb.f_qn_ang, vn = sqrtf(v2);
    auto threshold = [&](float ub) {
      const float su = sqrtf(ub), rr = vn + su;
      return ub < inf ? ub - qn + P.pb.f_eps * (3.0f * v2 + 4.0f * vn * su + ub) +
                            5.9604645e-8f * (2.0f + 8.0f * vn + 4.0f * rr + rr * rr)
                      : inf;
    };
    const float* cm = P.chunkmin + (size_t)s * kFilterMaxChunks;
    // the chunk with the smallest approximate key first: its exact minimum is a real upper bound
    unsigned long long near = kKeyNone;
    for (int c = lane; c < fp.NC; c += 32)
      near = min(near, ((unsigned long long)float_orderable(__ldcg(&cm[c])) << 32) | (unsigned)c);
    near = warp_min_key(near);
    const int c0 = (int)(unsigned)(near & 0xffffffffu);
    unsigned long long best = filter_rescan<DYN, UNIT_W>(P, nbeg + c0 * fp.CH, min(nend, nbeg + (c0 + 1) * fp.CH), q);
    float ub = best != kKeyNone ? __uint_as_float((unsigned)(best >> 32)) : inf;
    rows += fp.CH;
    // every other chunk whose minimum could still hide a nearer row: collected into a list, rescored together (the
    // loads of different chunks are independent), the bound tightened between batches
    int cnt = 0;
    unsigned long long mine = kKeyNone;  // this lane's best over the batch
    auto flush = [&]() {
      __syncwarp();
      for (int e = 0; e < cnt; ++e) {
        const int cc = list[e];
        const int rb = nbeg + cc * fp.CH, re = min(nend, rb + fp.CH);
        for (int i = rb + lane; i < re; i += 32) {
          float p[DP];
          const float4* sp = reinterpret_cast<const float4*>(P.states + (size_t)i * DP);
#pragma unroll
          for (int v = 0; v < DP / 4; ++v) {
            const float4 a = __ldcg(sp + v);
            p[4 * v] = a.x; p[4 * v + 1] = a.y; p[4 * v + 2] = a.z; p[4 * v + 3] = a.w;
          }
          const float d2 = dist2<DYN, UNIT_W>(P.pb, q, p);
          if (d2 >= 0.0f) mine = min(mine, ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned)i);
        }
      }
      rows += cnt * fp.CH;
      cnt = 0;
      best = min(best, warp_min_key(mine));
      if (best != kKeyNone) ub = __uint_as_float((unsigned)(best >> 32));
      __syncwarp();
    };
    for (int cb = 0; cb < fp.NC; cb += 32) {
      const int c = cb + lane;
      const float v = c < fp.NC ? __ldcg(&cm[c]) : inf;
      const bool is = c < fp.NC && c != c0 && v <= threshold(ub);
      const unsigned cand = __ballot_sync(0xffffffffu, is);
      if (cand == 0) continue;
      if (cnt + __popc(cand) > kFilterList) flush();  // keeps `is` as decided with the older, looser bound: still exact
      if (is) list[cnt + __popc(cand & ((1u << lane) - 1u))] = c;
      cnt += __popc(cand);
    }
    if (cnt > 0) flush();
    if (lane == 0 && best != kKeyNone) atomicMin(&key[s], best);
  }
  if (lane == 0 && rows) atomicAdd(rescored, (unsigned long long)rows);
}

}  // namespace pakr
