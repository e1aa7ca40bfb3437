// pakr_kernel_inst.cu -- instantiates the persistent kernel of pakr_kernel.cuh for (dynamics, obstacle kind).
// Compiled once per (tier, part) so that the sets build in parallel and a rarely used tier costs the common one
// no registers:  -DPAKR_STREAM_TIER=0 tiled NN scan (the normal case), =1 streaming NN tier for B <= 16,
// =2 tiled scan + NN index tier, =3 tiled scan + tensor-core coarse filter;
// -DPAKR_PART=0 double integrators, unicycles and the Acrobot, =1 quadrotors and the Dubins airplane.
#include "pakr_kernel.cuh"

#ifndef PAKR_STREAM_TIER
#define PAKR_STREAM_TIER 0
#endif
#ifndef PAKR_PART
#define PAKR_PART 0
#endif

namespace {
template <int DYN, int OBS> const void* kernel_ptr() {
  return (const void*)&pakr::pakr_loop_kernel<DYN, OBS, PAKR_STREAM_TIER>;
}
}  // namespace

#define PAKR_CAT3(a, b, c) a##b##_##c
#define PAKR_SELECT_NAME(tier, part) PAKR_CAT3(pakr_select_kernel_t, tier, part)

// pakr_select_kernel_t<tier>_<part>(dyn, obs): the kernel, or NULL if this unit does not hold it
extern "C" const void* PAKR_SELECT_NAME(PAKR_STREAM_TIER, PAKR_PART)(int dyn, int obs) {
  using namespace pakr;
  switch (dyn * 2 + obs) {
#if PAKR_PART == 0
    case DYN_DI2 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DI2, OBS_CIRCLE>();
    case DYN_DI2 * 2 + OBS_BOX: return kernel_ptr<DYN_DI2, OBS_BOX>();
    case DYN_DI3 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DI3, OBS_CIRCLE>();
    case DYN_DI3 * 2 + OBS_BOX: return kernel_ptr<DYN_DI3, OBS_BOX>();
    case DYN_UNI2 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_UNI2, OBS_CIRCLE>();
    case DYN_UNI2 * 2 + OBS_BOX: return kernel_ptr<DYN_UNI2, OBS_BOX>();
    case DYN_UNI1 * 2 + OBS_CIRCLE: return kernel_ptr<DYN_UNI1, OBS_CIRCLE>();
    case DYN_UNI1 * 2 + OBS_BOX: return kernel_ptr<DYN_UNI1, OBS_BOX>();
    case DYN_ACRO * 2 + OBS_CIRCLE: return kernel_ptr<DYN_ACRO, OBS_CIRCLE>();  // no obstacles: one variant
#else
    case DYN_QUAD * 2 + OBS_CIRCLE: return kernel_ptr<DYN_QUAD, OBS_CIRCLE>();
    case DYN_QUAD * 2 + OBS_BOX: return kernel_ptr<DYN_QUAD, OBS_BOX>();
    case DYN_DA * 2 + OBS_CIRCLE: return kernel_ptr<DYN_DA, OBS_CIRCLE>();
    case DYN_DA * 2 + OBS_BOX: return kernel_ptr<DYN_DA, OBS_BOX>();
    case DYN_QUADB * 2 + OBS_CIRCLE: return kernel_ptr<DYN_QUADB, OBS_CIRCLE>();
    case DYN_QUADB * 2 + OBS_BOX: return kernel_ptr<DYN_QUADB, OBS_BOX>();
#endif
  }
  return nullptr;
}
