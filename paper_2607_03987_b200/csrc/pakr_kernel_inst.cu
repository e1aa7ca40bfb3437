// pakr_kernel_inst.cu -- instantiates the persistent kernel of pakr_kernel.cuh for every (dynamics, obstacle kind).
// Compiled three times: -DPAKR_STREAM_TIER=0 (tiled NN scan, the normal case), =1 (streaming NN tier for B <= 16)
// and =2 (tiled scan + opt-in NN cell index), so that the sets build in parallel and the rarely used tiers cost
// the common one no registers.
#include "pakr_kernel.cuh"

#ifndef PAKR_STREAM_TIER
#define PAKR_STREAM_TIER 0
#endif

namespace {
template <int DYN, int OBS> const void* kernel_ptr() {
  return (const void*)&pakr::pakr_loop_kernel<DYN, OBS, PAKR_STREAM_TIER>;
}
}  // namespace

#if PAKR_STREAM_TIER == 2
extern "C" const void* pakr_select_kernel_index(int dyn, int obs) {
#elif PAKR_STREAM_TIER == 1
extern "C" const void* pakr_select_kernel_stream(int dyn, int obs) {
#else
extern "C" const void* pakr_select_kernel_tiled(int dyn, int obs) {
#endif
  using namespace pakr;
  switch (dyn * 2 + obs) {
    case DYN_DI2 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DI2, OBS_CIRCLE>();
    case DYN_DI2 * 2 + OBS_BOX: return kernel_ptr<DYN_DI2, OBS_BOX>();
    case DYN_DI3 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DI3, OBS_CIRCLE>();
    case DYN_DI3 * 2 + OBS_BOX: return kernel_ptr<DYN_DI3, OBS_BOX>();
    case DYN_UNI2 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_UNI2, OBS_CIRCLE>();
    case DYN_UNI2 * 2 + OBS_BOX: return kernel_ptr<DYN_UNI2, OBS_BOX>();
#if PAKR_STREAM_TIER != 2  // the opt-in index tier is built for the double integrators and the unicycle only
    case DYN_QUAD * 2 + OBS_CIRCLE: return kernel_ptr<DYN_QUAD, OBS_CIRCLE>();
    case DYN_QUAD * 2 + OBS_BOX: return kernel_ptr<DYN_QUAD, OBS_BOX>();
    case DYN_DA * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DA, OBS_CIRCLE>();
    case DYN_DA * 2 + OBS_BOX: return kernel_ptr<DYN_DA, OBS_BOX>();
    case DYN_UNI1 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_UNI1, OBS_CIRCLE>();
    case DYN_UNI1 * 2 + OBS_BOX: return kernel_ptr<DYN_UNI1, OBS_BOX>();
    case DYN_QUADB * 2 + OBS_CIRCLE: return kernel_ptr<DYN_QUADB, OBS_CIRCLE>();
    case DYN_QUADB * 2 + OBS_BOX: return kernel_ptr<DYN_QUADB, OBS_BOX>();
#endif
  }
  return nullptr;
}
