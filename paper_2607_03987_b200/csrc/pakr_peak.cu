// pakr_peak.cu -- measured fp32 peaks of the device, the denominators of the ALU roofline.
// "the builder must measure a sustained FFMA microbenchmark ... and use that as the denominator next
// to the nominal one".  Three register-only kernels, every thread a long run of independent chains:
//   FFMA            scalar fused multiply-add                         (1 lane-op per lane per instruction)
//   FFMA2           packed fma.rn.f32x2, the NN scan's instruction    (2 lane-ops per lane per instruction)
//   FADD2 + FFMA2   the scan's own mix: one packed subtract per packed fma
// A lane-op is one fp32 add, multiply or fused multiply-add on one lane.  Not on the planning path.
#include <algorithm>
#include <cuda_runtime.h>

#include "../../include/pakr.h"

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

extern "C" pakr_status pakr_measure_fp32_peak(int cuda_device, pakr_fp32_peak* out) {
  if (!out) return PAKR_ERR_INVALID_ARG;
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
  if (e == cudaSuccess) {
    out->sm_count = prop.multiProcessorCount;
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, cuda_device);
    out->sm_clock_mhz = khz / 1000.0;
  }
  if (buf) cudaFree(buf);
  if (prev >= 0) cudaSetDevice(prev);
  return e == cudaSuccess ? PAKR_OK : PAKR_ERR_CUDA;
}
