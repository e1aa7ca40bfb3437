// pakr_peak.cu -- measured fp32 peaks of the device, the denominators of the ALU roofline.
// "the builder must measure a sustained FFMA microbenchmark ... and use that as the denominator next
// to the nominal one".  Three register-only kernels, every thread a long run of independent chains:
//   FFMA            scalar fused multiply-add                         (1 lane-op per lane per instruction)
//   FFMA2           packed fma.rn.f32x2, the NN scan's instruction    (2 lane-ops per lane per instruction)
//   FADD2 + FFMA2   the scan's own mix: one packed subtract per packed fma
//   HMMA            mma.sync.m16n8k16 f16 x f16 -> f32, the tensor-core NN filter's instruction (pakr_nn_filter.cuh),
//                   alone (accumulating) and with the filter's epilogue: fresh accumulators folded into running minima
// A lane-op is one fp32 add, multiply or fused multiply-add on one lane.  Not on the planning path and not in libpakr.so:
// this file is libpakr_peak.so, loaded by bench.py alone (paper_2607_03987_b200/peak.py).
#include <algorithm>
#include <cuda_runtime.h>

#include "pakr_peak.h"

namespace {

constexpr int kChains = 16, kIters = 4096, kThreads = 1024, kCtasPerSm = 2;

__global__ void __launch_bounds__(kThreads) peak_ffma(float* out, float a, float b) {
  float x[kChains];
#pragma unroll
  for (int i = 0; i < kChains; ++i) x[i] = (float)(threadIdx.x + i);
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int i = 0; i < kChains; ++i) asm volatile("fma.rn.f32 %0, %0, %1, %2;" : "+f"(x[i]) : "f"(a), "f"(b));
  }
  float s = 0.0f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) s += x[i];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <bool MIX>
__global__ void __launch_bounds__(kThreads) peak_ffma2(float* out, float a, float b) {
  unsigned long long x[kChains], A, Bv;
  asm("mov.b64 %0, {%1, %1};" : "=l"(A) : "f"(a));
  asm("mov.b64 %0, {%1, %1};" : "=l"(Bv) : "f"(b));
#pragma unroll
  for (int i = 0; i < kChains; ++i) {
    const float f = (float)(threadIdx.x + i);
    asm("mov.b64 %0, {%1, %1};" : "=l"(x[i]) : "f"(f));
  }
  for (int it = 0; it < kIters; ++it) {
#pragma unroll
    for (int i = 0; i < kChains; ++i) {
      if (MIX && (i & 1)) asm volatile("sub.rn.f32x2 %0, %0, %1;" : "+l"(x[i]) : "l"(Bv));
      else asm volatile("fma.rn.f32x2 %0, %0, %1, %2;" : "+l"(x[i]) : "l"(A), "l"(Bv));
    }
  }
  float s = 0.0f;
#pragma unroll
  for (int i = 0; i < kChains; ++i) {
    float lo, hi;
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(x[i]));
    s += lo + hi;
  }
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

__device__ __forceinline__ void mma_16816(float (&c)[4], const unsigned (&a)[4], const unsigned (&b)[2]) {
  asm volatile("mma.sync.aligned.m16n8k16.row.col.f32.f16.f16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
               : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
               : "r"(a[0]), "r"(a[1]), "r"(a[2]), "r"(a[3]), "r"(b[0]), "r"(b[1]));
}
constexpr int kMmaChains = 8, kMmaIters = 8192;

template <bool MIN_FOLD>
__global__ void __launch_bounds__(kThreads) peak_mma(float* out, float a0, float b0) {
  unsigned a[kMmaChains][4], b[2] = {__float_as_uint(b0) + threadIdx.x, 0x3c003c00u};
#pragma unroll
  for (int i = 0; i < kMmaChains; ++i) {
    a[i][0] = __float_as_uint(a0) + i; a[i][1] = 0x3c003c00u + threadIdx.x; a[i][2] = 0x38003800u; a[i][3] = 0x34003400u + i;
  }
  float acc[kMmaChains][4], m[kMmaChains][2];
#pragma unroll
  for (int i = 0; i < kMmaChains; ++i) {
    acc[i][0] = acc[i][1] = acc[i][2] = acc[i][3] = 0.0f;
    m[i][0] = m[i][1] = 3.0e38f;
  }
  for (int it = 0; it < kMmaIters; ++it) {
    if (MIN_FOLD) b[0] += 0x00010001u;
#pragma unroll
    for (int i = 0; i < kMmaChains; ++i) {
      if (MIN_FOLD) {
        float c[4] = {0.0f, 0.0f, 0.0f, 0.0f};
        mma_16816(c, a[i], b);
        m[i][0] = fminf(m[i][0], fminf(c[0], c[1]));
        m[i][1] = fminf(m[i][1], fminf(c[2], c[3]));
      } else {
        mma_16816(acc[i], a[i], b);
      }
    }
  }
  float s = 0.0f;
#pragma unroll
  for (int i = 0; i < kMmaChains; ++i) s += acc[i][0] + acc[i][1] + acc[i][2] + acc[i][3] + m[i][0] + m[i][1];
  out[blockIdx.x * blockDim.x + threadIdx.x] = s;
}

template <class K>
cudaError_t time_kernel(K kernel, int sms, float* out, int reps, double lane_ops_per_thread, double* rate) {
  cudaEvent_t e0, e1;
  cudaError_t e = cudaEventCreate(&e0);
  if (e != cudaSuccess) return e;
  e = cudaEventCreate(&e1);
  if (e != cudaSuccess) { cudaEventDestroy(e0); return e; }
  const int grid = sms * kCtasPerSm;
  kernel<<<grid, kThreads>>>(out, 1.0001f, 0.5f);  // warm-up
  float best = 1e30f;
  for (int r = 0; r < reps && e == cudaSuccess; ++r) {
    cudaEventRecord(e0);
    kernel<<<grid, kThreads>>>(out, 1.0001f, 0.5f);
    cudaEventRecord(e1);
    e = cudaEventSynchronize(e1);
    float ms = 0.0f;
    if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, e0, e1);
    best = std::min(best, ms);
  }
  if (e == cudaSuccess) e = cudaGetLastError();
  *rate = (double)grid * kThreads * lane_ops_per_thread / ((double)best * 1e-3);
  cudaEventDestroy(e0);
  cudaEventDestroy(e1);
  return e;
}

}  // namespace

extern "C" int pakr_measure_fp32_peak(int cuda_device, pakr_fp32_peak* out) {
  if (!out) return 1;
  int prev = -1;
  if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
  cudaError_t e = cudaSetDevice(cuda_device);
  cudaDeviceProp prop;
  if (e == cudaSuccess) e = cudaGetDeviceProperties(&prop, cuda_device);
  float* buf = nullptr;
  if (e == cudaSuccess) e = cudaMalloc(&buf, (size_t)prop.multiProcessorCount * kCtasPerSm * kThreads * sizeof(float));
  const double per_thread = (double)kChains * kIters;
  if (e == cudaSuccess) e = time_kernel(peak_ffma, prop.multiProcessorCount, buf, 5, per_thread, &out->ffma_lane_ops_per_s);
  if (e == cudaSuccess) e = time_kernel(peak_ffma2<false>, prop.multiProcessorCount, buf, 5, 2.0 * per_thread, &out->ffma2_lane_ops_per_s);
  if (e == cudaSuccess) e = time_kernel(peak_ffma2<true>, prop.multiProcessorCount, buf, 5, 2.0 * per_thread, &out->scan_mix_lane_ops_per_s);
  // one warp instruction = 16 x 8 x 16 multiply-accumulates: 64 per lane
  const double mma_per_thread = (double)kMmaChains * kMmaIters * 64.0;
  if (e == cudaSuccess) e = time_kernel(peak_mma<false>, prop.multiProcessorCount, buf, 5, mma_per_thread, &out->mma_f16_mac_per_s);
  if (e == cudaSuccess) e = time_kernel(peak_mma<true>, prop.multiProcessorCount, buf, 5, mma_per_thread, &out->mma_f16_minfold_mac_per_s);
  if (e == cudaSuccess) {
    out->sm_count = prop.multiProcessorCount;
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, cuda_device);
    out->sm_clock_mhz = khz / 1000.0;
  }
  if (buf) cudaFree(buf);
  if (prev >= 0) cudaSetDevice(prev);
  return e == cudaSuccess ? 0 : 5;
}
