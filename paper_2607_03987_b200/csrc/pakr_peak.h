/* pakr_peak.h -- measurement support, NOT part of the planning library: the microbenchmark behind the ALU / mma.sync
 * roofline denominators of bench.py ("measure a sustained FFMA microbenchmark ... and use that as the
 * denominator next to the nominal one").  Built into libpakr_peak.so, which only bench.py loads. */
#ifndef PAKR_PEAK_H
#define PAKR_PEAK_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

/* Measurement support, not on the planning path: sustained fp32 rates of `cuda_device`, the denominators of the ALU
 * roofline (the measured FFMA rate stands beside the nominal SMs x 128 lanes x clock) and of the
 * tensor-core NN filter's.  Runs five register-only kernels for a few milliseconds each on the default stream and
 * synchronises.  A lane-op is one fp32 add, multiply or fused multiply-add on one lane; a packed f32x2 instruction
 * counts two per lane.  *out is HOST. */
typedef struct {
  double ffma_lane_ops_per_s;     /* scalar fma.rn.f32 (SASS FFMA)                                    */
  double ffma2_lane_ops_per_s;    /* packed fma.rn.f32x2 (SASS FFMA2), the NN scan's arithmetic       */
  double scan_mix_lane_ops_per_s; /* one packed subtract per packed fma: the NN scan's own mix        */
  double sm_clock_mhz;            /* the device's reported peak SM clock                              */
  int32_t sm_count;
  double mma_f16_mac_per_s;         /* mma.sync.m16n8k16 f16 x f16 -> f32 (SASS HMMA.16816.F32), multiply-accumulates/s  */
  double mma_f16_minfold_mac_per_s; /* the same with the NN filter's epilogue: fresh accumulators, 4 FMNMX per mma       */
} pakr_fp32_peak;
/* 0 = ok, 1 = out is NULL, 5 = a CUDA call failed.  The caller's current device is restored. */
int pakr_measure_fp32_peak(int cuda_device, pakr_fp32_peak* out);

#ifdef __cplusplus
}
#endif
#endif /* PAKR_PEAK_H */
