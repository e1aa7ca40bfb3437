// pakr_api.cu -- host side of the C ABI declared in include/pakr.h.
// Validates the problem, carves the caller's workspace, launches the persistent cooperative
// kernel of pakr_kernel.cuh and copies the small result block back.  No compute happens here.
#include <algorithm>
#include <cmath>
#include <cstddef>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/pakr.h"
#include "pakr_kernel.cuh"

using namespace pakr;

struct pakr_planner {
  int device = 0;
  int dyn = 0, obs = 0;     // DynKind, ObsKind
  int D = 0, M = 0, PD = 0, DP = 0;
  DevProblem pb{};
  float* d_obstacles = nullptr;
  uint32_t* d_grid_cells = nullptr;
  uint16_t* d_grid_list = nullptr;
  int num_sms = 0, blocks_per_sm = 0;
  bool filter_ok = false; // tensor-core NN filter usable: every feature fits fp16 (pakr_nn_filter.cuh)
  bool index_ok = false;  // NN spatial index usable: finite position box, positive position weights, kernel built
  size_t smem_bytes = 0;
  const void* kernel = nullptr;         // tiled NN scan
  const void* kernel_stream = nullptr;  // streaming NN tier (B <= kStreamB)
  const void* kernel_index = nullptr;   // tiled scan + NN index (only when nn_index != 0)
  const void* kernel_filter = nullptr;  // tiled scan + tensor-core coarse filter
  void* h_pinned = nullptr;  // Ctrl + path staging
  std::string err;
};

static thread_local std::string g_create_err;

// defined in pakr_kernel_inst.cu (one translation unit per NN tier)
extern "C" const void* pakr_select_kernel_t0_0(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t0_1(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t1_0(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t1_1(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t2_0(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t2_1(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t3_0(int dyn, int obs);
extern "C" const void* pakr_select_kernel_t3_1(int dyn, int obs);

static const void* pakr_select_kernel_tiled(int dyn, int obs) {
  const void* k = pakr_select_kernel_t0_0(dyn, obs);
  return k ? k : pakr_select_kernel_t0_1(dyn, obs);
}
static const void* pakr_select_kernel_stream(int dyn, int obs) {
  const void* k = pakr_select_kernel_t1_0(dyn, obs);
  return k ? k : pakr_select_kernel_t1_1(dyn, obs);
}
static const void* pakr_select_kernel_index(int dyn, int obs) {
  const void* k = pakr_select_kernel_t2_0(dyn, obs);
  return k ? k : pakr_select_kernel_t2_1(dyn, obs);
}

static const void* pakr_select_kernel_filter(int dyn, int obs) {
  const void* k = pakr_select_kernel_t3_0(dyn, obs);
  return k ? k : pakr_select_kernel_t3_1(dyn, obs);
}

namespace {

constexpr size_t kAlign = 256;
size_t align_up(size_t v) { return (v + kAlign - 1) / kAlign * kAlign; }

struct Layout {
  size_t states, actions, parents, costs, nn_key, prow, frow, chunkmin, unit_count, scr_state, scr_ctrl, scr_cost, scr_parent,
      scr_flags, idx_keys, idx_ids, idx_hist, idx_ctasum, idx_tile_ids, idx_rows, idx_tlo, idx_thi, idx_slo, idx_shi,
      ctrl, path_rev, path_nodes, path_states, path_controls, total;
};

// nn_mode = kLayoutAllTiers reserves the buffers of every tier the problem admits (pakr_workspace_bytes); a PAKR_NN_*
// value reserves only what that mode can launch (pakr_workspace_bytes_for).  The tree comes first and everything up to
// the path buffers has the same offset whatever the mode, so pakr_get_tree_layout and pakr_read_stats need not know it;
// the tiers' own buffers (all rebuilt inside every launch) follow.
constexpr int kLayoutAllTiers = -1;
constexpr int kAutoMinB = 4096;  // PAKR_NN_AUTO: the spatial index from this many queries up (set_nn_mode)

Layout make_layout(const pakr_planner* pl, int64_t B, int64_t K, int64_t cap, int nn_mode = kLayoutAllTiers) {
  Layout L{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  const size_t BK = (size_t)B * K, U = BK, slots = BK + 32;  // phase-B warp units hold 1..32 children
  L.states = take((size_t)cap * pl->DP * 4);
  L.actions = take((size_t)cap * 16);
  L.parents = take((size_t)cap * 4);
  L.costs = take((size_t)cap * 4);
  L.nn_key = take((size_t)B * 16);  // two iterations in flight
  L.unit_count = take(std::max<size_t>(U, kFuseUnits + 8) * 4);
  L.scr_state = take(slots * pl->DP * 4);
  L.scr_ctrl = take(slots * 16);
  L.scr_cost = take(slots * 4);
  L.scr_parent = take(slots * 4);
  L.scr_flags = take(slots * 4);
  L.ctrl = take(sizeof(Ctrl));
  L.path_rev = take((size_t)kPathMax * 4);
  L.path_nodes = take((size_t)kPathMax * 4);
  L.path_states = take((size_t)kPathMax * kMaxD * 4);
  L.path_controls = take((size_t)kPathMax * kMaxM * 4);
  // per-tier buffers; B <= kStreamB always launches the streaming kernel, which uses neither index nor filter
  const bool stream = B <= kStreamB;
  const bool all = nn_mode == kLayoutAllTiers;
  const size_t want_filter = (!stream && pl->filter_ok && (all || nn_mode == PAKR_NN_FILTER)) ? 1 : 0;
  const size_t want_index = (!stream && pl->index_ok && (all || nn_mode == PAKR_NN_INDEX || (nn_mode == PAKR_NN_AUTO && B >= kAutoMinB))) ? 1 : 0;
  L.prow = take(stream ? ((size_t)cap + 4) * pl->D * 4 : 0);        // streaming tier: packed rows
  L.frow = take(want_filter * ((size_t)cap + 8) * 96);              // filter rows: K <= 48 halves
  L.chunkmin = take(want_filter * (size_t)B * kFilterMaxChunks * 4);
  {  // NN index; nothing when the problem cannot be indexed
    const size_t on = want_index;
    const IdxDims G = idx_dims((int)cap);
    const size_t grid_warps = (size_t)pl->num_sms * kCtasPerSm * kWarps;
    const size_t sort_warps = std::min<size_t>(grid_warps, (size_t)cap / kIdxChunkMin + 1);
    L.idx_keys = take(on * 2 * cap * 4);
    L.idx_ids = take(on * 2 * cap * 4);
    L.idx_hist = take(on * kIdxBins * sort_warps * 4);
    L.idx_ctasum = take(on * pl->num_sms * kCtasPerSm * 4);
    L.idx_tile_ids = take(on * (size_t)G.n_super * 1024 * 4);
    L.idx_rows = take(on * (size_t)G.n_super * 1024 * pl->D * 4);
    L.idx_tlo = take(on * (size_t)G.n_super * pl->D * 32 * 4);
    L.idx_thi = take(on * (size_t)G.n_super * pl->D * 32 * 4);
    L.idx_slo = take(on * (size_t)G.n_groups * pl->D * 32 * 4);
    L.idx_shi = take(on * (size_t)G.n_groups * pl->D * 32 * 4);
  }
  L.total = o;
  return L;
}

bool nn_mode_ok(int nn_mode) {
  return nn_mode == PAKR_NN_AUTO || nn_mode == PAKR_NN_SCAN || nn_mode == PAKR_NN_INDEX || nn_mode == PAKR_NN_FILTER;
}

bool sizes_ok(int64_t B, int64_t K, int64_t cap) {
  return B >= 1 && K >= 1 && K <= 4096 && B * K <= (1ll << 24) && cap >= 2 && cap <= (1ll << 30);
}

size_t tile_floats(int DP) { return (size_t)TileCfg<DYN_DI2>::TILE * 4; }  // every tile buffer is the same size

size_t smem_for(const pakr_planner* pl) {
  const int os = pl->obs == OBS_CIRCLE ? 4 : 8;
  return kWarps * 2 * tile_floats(pl->DP) * 4 + kWarps * 4 * 8 + (kThreads + kWarps + 8) * 4 + kMaxD * 2 * 32 * kQ * 4 + kWarps * 32 * kQ * 8 +
         (size_t)((pl->pb.n_obs * os + 3) & ~3) * 4 + (size_t)pl->pb.g_cells * 4 + (size_t)pl->pb.g_list * 2 + 16;
}

// Obstacle broad phase: a uniform grid over the position box with a CSR list of obstacle ids per cell.
// An obstacle is registered in every cell its bounding box, inflated by a thousandth of a cell, touches,
// using the same clamp(floor((x - org) * inv)) the kernel applies to a position; that function is monotone
// per axis, so a position inside an obstacle always lands in a cell that lists it (exact culling).
struct HostGrid {
  bool on = false;
  int dim[3] = {1, 1, 1};
  float org[3] = {0, 0, 0}, inv[3] = {0, 0, 0};
  std::vector<uint32_t> cells;
  std::vector<uint16_t> list;
};

HostGrid build_grid(const pakr_problem* p, int obs_kind) {
  HostGrid g;
  const int gd = obs_kind == OBS_CIRCLE ? 2 : p->pos_dim;
  if (p->n_obstacles < 4) return g;  // nothing to cull
  for (int a = 0; a < gd; ++a)
    if (!std::isfinite(p->state_lo[a]) || !std::isfinite(p->state_hi[a]) || !(p->state_hi[a] > p->state_lo[a])) return g;
  for (int res = (gd == 2 ? 32 : 16); res >= 4; res /= 2) {
    float cell[3];
    for (int a = 0; a < 3; ++a) g.dim[a] = 1;
    for (int a = 0; a < gd; ++a) {
      g.dim[a] = res;
      g.org[a] = p->state_lo[a];
      cell[a] = (p->state_hi[a] - p->state_lo[a]) / (float)res;
      g.inv[a] = 1.0f / cell[a];
    }
    auto cell_of = [&](float x, int a) {
      const float f = std::floor((x - g.org[a]) * g.inv[a]);
      int c = f >= 2.0e9f ? 2000000000 : f <= -2.0e9f ? -2000000000 : (int)f;
      return std::min(std::max(c, 0), g.dim[a] - 1);
    };
    const int ncells = g.dim[0] * g.dim[1] * g.dim[2];
    std::vector<std::vector<uint16_t>> per(ncells);
    for (int o = 0; o < p->n_obstacles; ++o) {
      int c0[3] = {0, 0, 0}, c1[3] = {0, 0, 0};
      for (int a = 0; a < gd; ++a) {
        float lo, hi;
        if (obs_kind == OBS_CIRCLE) {
          const float* c = p->obstacles + (size_t)o * 3;
          lo = c[a] - std::fabs(c[2]); hi = c[a] + std::fabs(c[2]);
        } else {
          lo = p->obstacles[(size_t)o * 2 * p->pos_dim + a];
          hi = p->obstacles[(size_t)o * 2 * p->pos_dim + p->pos_dim + a];
        }
        const float pad = 1e-3f * cell[a] + 1e-5f * (std::fabs(lo) + std::fabs(hi));
        c0[a] = cell_of(lo - pad, a);
        c1[a] = cell_of(hi + pad, a);
      }
      for (int z = c0[2]; z <= c1[2]; ++z)
        for (int y = c0[1]; y <= c1[1]; ++y)
          for (int x = c0[0]; x <= c1[0]; ++x) per[x + g.dim[0] * (y + g.dim[1] * z)].push_back((uint16_t)o);
    }
    size_t total = 0, worst = 0;
    for (auto& v : per) { total += v.size(); worst = std::max(worst, v.size()); }
    if (worst > 255 || total > 24576) continue;  // coarser grid
    g.cells.resize(ncells);
    g.list.clear();
    for (int c = 0; c < ncells; ++c) {
      const uint32_t cnt = (uint32_t)per[c].size();
      if (cnt <= 2) {  // ids inline (n_obstacles <= 1024 fits 12 bits)
        g.cells[c] = cnt | (cnt > 0 ? (uint32_t)per[c][0] << 8 : 0u) | (cnt > 1 ? (uint32_t)per[c][1] << 20 : 0u);
      } else {
        g.cells[c] = ((uint32_t)g.list.size() << 8) | cnt;
        g.list.insert(g.list.end(), per[c].begin(), per[c].end());
      }
    }
    if (g.list.empty()) g.list.push_back(0);
    g.on = true;
    return g;
  }
  return g;
}

// Morton key layout of the NN index: 30 key bits are dealt out one at a time, always to the dimension whose weighted
// cell (hi - lo) sqrt(w) / 2^bits is widest at that moment -- the split order of a kd-tree over the weighted state
// box.  Keyed: non-angle dimensions with a finite box of positive width and a positive weight.  Returns false if
// no dimension can be keyed (the index tier is then unavailable for the problem).
bool idx_key_layout(DevProblem& pb, int D, unsigned angle_mask) {
  double cell[kMaxD];
  int bits[kMaxD] = {0};
  bool any = false;
  for (int d = 0; d < D; ++d) {
    const bool ok = !((angle_mask >> d) & 1u) && std::isfinite(pb.lo[d]) && std::isfinite(pb.hi[d]) && pb.hi[d] > pb.lo[d] && pb.w[d] > 0.0f;
    cell[d] = ok ? ((double)pb.hi[d] - pb.lo[d]) * std::sqrt((double)pb.w[d]) : 0.0;
    any = any || ok;
  }
  if (!any) return false;
  int order[kIdxDigitBits * kIdxPasses];
  int total = 0;
  for (; total < kIdxDigitBits * kIdxPasses; ++total) {
    int best = -1;
    for (int d = 0; d < D; ++d)
      if (cell[d] > 0.0 && bits[d] < 16 && (best < 0 || cell[d] > cell[best])) best = d;
    if (best < 0) break;
    order[total] = best;
    ++bits[best];
    cell[best] *= 0.5;
  }
  int taken[kMaxD] = {0};
  for (int i = 0; i < total; ++i) {  // i-th dealt bit: key position total-1-i, the dimension's next bit from its top
    const int d = order[i];
    pb.idx_pos[d][bits[d] - 1 - taken[d]] = (uint8_t)(total - 1 - i);
    ++taken[d];
  }
  for (int d = 0; d < D; ++d) {
    pb.idx_bits[d] = (uint8_t)bits[d];
    pb.idx_scale[d] = bits[d] ? (float)((double)(1 << bits[d]) / ((double)pb.hi[d] - pb.lo[d])) : 0.0f;
  }
  return true;
}

pakr_status fail(pakr_planner* pl, pakr_status st, const std::string& msg) {
  if (pl) pl->err = msg;
  else g_create_err = msg;
  return st;
}

// Binds the planner's device for the duration of one ABI call and puts the caller's device back afterwards
// (a host process with several GPUs, e.g. PyTorch, must not find its current device changed).
struct DeviceGuard {
  int prev = -1;
  cudaError_t err;
  explicit DeviceGuard(int dev) {
    if (cudaGetDevice(&prev) != cudaSuccess) prev = -1;
    err = cudaSetDevice(dev);
  }
  ~DeviceGuard() {
    if (prev >= 0) cudaSetDevice(prev);
  }
};

#define CUDA_TRY(pl, expr)                                                                       \
  do {                                                                                           \
    cudaError_t e_ = (expr);                                                                     \
    if (e_ != cudaSuccess)                                                                       \
      return fail(pl, PAKR_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_));        \
  } while (0)

}  // namespace

extern "C" pakr_status pakr_create(const pakr_problem* p, int cuda_device, pakr_planner** out) {
  if (out) *out = nullptr;
  if (!p || !out) return fail(nullptr, PAKR_ERR_INVALID_ARG, "null problem or out pointer");
  if (!p->state_lo || !p->state_hi || !p->dim_kind || !p->nn_weight || !p->control_lo || !p->control_hi ||
      !p->start || !p->goal_center)
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "null array in problem");
  int dyn = -1;
  if (p->dynamics_id == PAKR_DYN_DOUBLE_INTEGRATOR) {
    if (p->pos_dim == 2 && p->state_dim == 4 && p->control_dim == 2) dyn = DYN_DI2;
    else if (p->pos_dim == 3 && p->state_dim == 6 && p->control_dim == 3) dyn = DYN_DI3;
    else return fail(nullptr, PAKR_ERR_INVALID_ARG, "double integrator needs (D,m,pos)=(4,2,2) or (6,3,3)");
  } else if (p->dynamics_id == PAKR_DYN_UNICYCLE2) {
    if (p->pos_dim != 2 || p->state_dim != 5 || p->control_dim != 2)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "unicycle2 needs (D,m,pos)=(5,2,2)");
    dyn = DYN_UNI2;
  } else if (p->dynamics_id == PAKR_DYN_QUADROTOR || p->dynamics_id == PAKR_DYN_QUADROTOR_BODY) {
    if (p->pos_dim != 3 || p->state_dim != 12 || p->control_dim != 4)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "quadrotor needs (D,m,pos)=(12,4,3)");
    if (p->n_dyn_params < 5 || !p->dyn_params)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "quadrotor needs dyn_params m,Ixx,Iyy,Izz,g");
    for (int i = 0; i < 4; ++i)
      if (!(p->dyn_params[i] > 0.0f)) return fail(nullptr, PAKR_ERR_INVALID_ARG, "mass/inertia must be > 0");
    dyn = p->dynamics_id == PAKR_DYN_QUADROTOR ? DYN_QUAD : DYN_QUADB;
  } else if (p->dynamics_id == PAKR_DYN_DUBINS_AIRPLANE) {
    if (p->pos_dim != 3 || p->state_dim != 6 || p->control_dim != 3)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "dubins airplane needs (D,m,pos)=(6,3,3)");
    dyn = DYN_DA;
  } else if (p->dynamics_id == PAKR_DYN_UNICYCLE1) {
    if (p->pos_dim != 2 || p->state_dim != 3 || p->control_dim != 2)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "unicycle1 needs (D,m,pos)=(3,2,2)");
    dyn = DYN_UNI1;
  } else if (p->dynamics_id == PAKR_DYN_ACROBOT) {
    if (p->pos_dim != 2 || p->state_dim != 4 || p->control_dim != 1)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "acrobot needs (D,m,pos)=(4,1,2)");
    if (p->n_dyn_params < 8 || !p->dyn_params)
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "acrobot needs dyn_params m1,m2,l1,lc1,lc2,I1,I2,g");
    for (int i = 0; i < 7; ++i)
      if (!(p->dyn_params[i] > 0.0f) || !std::isfinite(p->dyn_params[i]))
        return fail(nullptr, PAKR_ERR_INVALID_ARG, "acrobot masses, lengths and inertias must be finite and > 0");
    if (!std::isfinite(p->dyn_params[7])) return fail(nullptr, PAKR_ERR_INVALID_ARG, "acrobot g must be finite");
    if (p->n_obstacles > 0)
      return fail(nullptr, PAKR_ERR_UNSUPPORTED, "the acrobot takes no obstacles (its position dims are angles)");
    dyn = DYN_ACRO;
  } else {
    return fail(nullptr, PAKR_ERR_UNSUPPORTED, "unknown dynamics_id");
  }
  if (p->integrator != PAKR_INT_EULER && p->integrator != PAKR_INT_RK4)
    return fail(nullptr, PAKR_ERR_UNSUPPORTED, "unknown integrator");
  if (p->cost_mode != PAKR_COST_DURATION && p->cost_mode != PAKR_COST_PATH_LENGTH)
    return fail(nullptr, PAKR_ERR_UNSUPPORTED, "unknown cost_mode");
  int obs = -1;
  if (p->obstacle_type == PAKR_OBS_CIRCLE2D || p->obstacle_type == PAKR_OBS_ZCYLINDER) obs = OBS_CIRCLE;
  else if (p->obstacle_type == PAKR_OBS_AABB) obs = OBS_BOX;
  else return fail(nullptr, PAKR_ERR_UNSUPPORTED, "unknown obstacle_type");
  if (dyn == DYN_ACRO) obs = OBS_CIRCLE;  // no obstacles: one kernel variant
  if (p->n_obstacles < 0 || p->n_obstacles > 1024 || (p->n_obstacles > 0 && !p->obstacles))
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "n_obstacles must be in [0,1024] with a non-null array");
  const int D = p->state_dim, M = p->control_dim, PD = p->pos_dim;
  {
    const int per = (obs == OBS_CIRCLE) ? 3 : 2 * PD;
    for (int i = 0; i < p->n_obstacles * per; ++i)
      if (!std::isfinite(p->obstacles[i])) return fail(nullptr, PAKR_ERR_INVALID_ARG, "obstacle coordinates must be finite");
  }
  const unsigned angles = dyn == DYN_UNI2 ? DynTraits<DYN_UNI2>::ANGLES : dyn == DYN_QUAD ? DynTraits<DYN_QUAD>::ANGLES
                        : dyn == DYN_DA ? DynTraits<DYN_DA>::ANGLES : dyn == DYN_UNI1 ? DynTraits<DYN_UNI1>::ANGLES
                        : dyn == DYN_QUADB ? DynTraits<DYN_QUADB>::ANGLES : dyn == DYN_ACRO ? DynTraits<DYN_ACRO>::ANGLES : 0u;
  auto angle_dim = [&](int d) { return ((angles >> d) & 1u) != 0; };
  for (int d = 0; d < D; ++d) {
    const bool marked = p->dim_kind[d] == PAKR_DIM_ANGLE;
    if (p->dim_kind[d] > 1 || marked != angle_dim(d))
      return fail(nullptr, PAKR_ERR_UNSUPPORTED, "dim_kind must mark exactly the dynamics' own angle dims");
    if (std::isnan(p->state_lo[d]) || std::isnan(p->state_hi[d]) || std::isnan(p->nn_weight[d]) ||
        std::isnan(p->start[d]))
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "NaN in state bounds, weights or start");
    if (p->state_lo[d] > p->state_hi[d]) return fail(nullptr, PAKR_ERR_INVALID_ARG, "state_lo > state_hi");
    if (p->nn_weight[d] < 0.0f) return fail(nullptr, PAKR_ERR_INVALID_ARG, "nn_weight < 0");
    if (!marked && p->nn_weight[d] > 0.0f && (std::isinf(p->state_lo[d]) || std::isinf(p->state_hi[d])))
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "a sampled dim (weight > 0) needs finite bounds");
  }
  for (int j = 0; j < M; ++j) {
    if (!std::isfinite(p->control_lo[j]) || !std::isfinite(p->control_hi[j]) || p->control_lo[j] > p->control_hi[j])
      return fail(nullptr, PAKR_ERR_INVALID_ARG, "control bounds must be finite with lo <= hi");
  }
  if (!(p->dt > 0.0f) || !std::isfinite(p->dt) || p->steps_per_edge < 1)
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "dt must be > 0 and steps_per_edge >= 1");
  if (!(p->goal_radius >= 0.0f) || !(p->heuristic_speed > 0.0f))
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_radius >= 0 and heuristic_speed > 0 required");
  if (p->goal_angle_dim != -1 && (p->goal_angle_dim < 0 || p->goal_angle_dim >= D || !angle_dim(p->goal_angle_dim)))
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_angle_dim must be -1 or one of the dynamics' angle dims");
  if (p->goal_angle_dim != -1 && (!std::isfinite(p->goal_angle) || !std::isfinite(p->goal_angle_tol) || p->goal_angle_tol < 0.0f))
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_angle must be finite and goal_angle_tol finite and >= 0");
  // goal ball: listed dims, or the position dims
  if (p->goal_n_dims < 0 || p->goal_n_dims > D || (p->goal_n_dims > 0 && !p->goal_dims))
    return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_n_dims must be in [0, state_dim] with a non-null goal_dims");
  const int n_goal = p->goal_n_dims > 0 ? p->goal_n_dims : p->pos_dim;
  int goal_dim[kMaxD];
  for (int i = 0; i < n_goal; ++i) {
    goal_dim[i] = p->goal_n_dims > 0 ? p->goal_dims[i] : i;
    if (goal_dim[i] < 0 || goal_dim[i] >= D) return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_dims entry out of range");
    for (int j = 0; j < i; ++j)
      if (goal_dim[j] == goal_dim[i]) return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_dims entries must be distinct");
    if (!std::isfinite(p->goal_center[i])) return fail(nullptr, PAKR_ERR_INVALID_ARG, "goal_center must be finite");
  }

  auto* pl = new pakr_planner();
  pl->device = cuda_device;
  pl->dyn = dyn; pl->obs = obs; pl->D = D; pl->M = M; pl->PD = PD;
  pl->DP = (D + 3) / 4 * 4;
  DevProblem& pb = pl->pb;
  std::memset(&pb, 0, sizeof(pb));
  bool unit = true;
  for (int d = 0; d < kMaxD; ++d) { pb.lo[d] = -INFINITY; pb.hi[d] = INFINITY; }
  for (int d = 0; d < D; ++d) {
    pb.lo[d] = p->state_lo[d]; pb.hi[d] = p->state_hi[d]; pb.w[d] = p->nn_weight[d]; pb.start[d] = p->start[d];
    if (pb.w[d] != 1.0f) unit = false;
    if (angle_dim(d)) { pb.samp_lo[d] = -kPiF; pb.samp_span[d] = kPiF - (-kPiF); }
    else if (std::isfinite(pb.lo[d]) && std::isfinite(pb.hi[d])) { pb.samp_lo[d] = pb.lo[d]; pb.samp_span[d] = pb.hi[d] - pb.lo[d]; }
    else { pb.samp_lo[d] = 0.0f; pb.samp_span[d] = 0.0f; }
  }
  for (int j = 0; j < M; ++j) { pb.ulo[j] = p->control_lo[j]; pb.uhi[j] = p->control_hi[j]; pb.uspan[j] = pb.uhi[j] - pb.ulo[j]; }
  for (int i = 0; i < n_goal; ++i) { pb.goal_c[goal_dim[i]] = p->goal_center[i]; pb.goal_m[goal_dim[i]] = 1.0f; }
  pb.goal_r = p->goal_radius; pb.goal_angle = p->goal_angle; pb.goal_angle_tol = p->goal_angle_tol;
  pb.goal_angle_dim = p->goal_angle_dim;
  if (dyn == DYN_ACRO) {  // the lumped constants dyn_f<DYN_ACRO> reads (P35)
    const double m1 = p->dyn_params[0], m2 = p->dyn_params[1], l1 = p->dyn_params[2], lc1 = p->dyn_params[3],
                 lc2 = p->dyn_params[4], I1 = p->dyn_params[5], I2 = p->dyn_params[6], g = p->dyn_params[7];
    pb.dyn[0] = (float)(I1 + I2 + m1 * lc1 * lc1 + m2 * (l1 * l1 + lc2 * lc2));
    pb.dyn[1] = (float)(m2 * l1 * lc2);
    pb.dyn[2] = (float)(I2 + m2 * lc2 * lc2);
    pb.dyn[3] = (float)((m1 * lc1 + m2 * l1) * g);
    pb.dyn[4] = (float)(m2 * lc2 * g);
  } else {
    for (int i = 0; i < 5 && i < p->n_dyn_params; ++i) pb.dyn[i] = p->dyn_params[i];
  }
  if (dyn == DYN_QUAD || dyn == DYN_QUADB)
    for (int i = 0; i < 4; ++i) pb.dyn[5 + i] = 1.0f / p->dyn_params[i];
  pb.dt = p->dt; pb.S = p->steps_per_edge; pb.integrator = p->integrator; pb.cost_mode = p->cost_mode;
  pb.inv_hspeed = std::isinf(p->heuristic_speed) ? 0.0f : 1.0f / p->heuristic_speed;
  pb.unit_weights = unit ? 1 : 0;
  pl->index_ok = idx_key_layout(pb, D, angles);
  {
    // tensor-core NN filter: features u_d = sqrt(w_d) (x_d - centre_d) of the real dims, sqrt(w) (cos, sin) of the
    // angle dims, |u_real|^2.  S_max bounds sum_i |c_i u_i| over the state box (c = (-2 v, 1)): |u|^2 <= sum U_d^2,
    // 2 |v.u| <= 2 sum U_d^2, 2 w per angle dim; U_d = sqrt(w_d) (hi_d - lo_d) / 2.
    double sum_u2 = 0.0, w_ang = 0.0;
    bool ok = true;
    for (int d = 0; d < D; ++d) {
      pb.f_scale[d] = std::sqrt(pb.w[d]);
      if (angle_dim(d)) { w_ang += pb.w[d]; pb.f_ctr[d] = 0.0f; continue; }
      if (pb.w[d] > 0.0f) {  // finite box (validated above)
        pb.f_ctr[d] = 0.5f * pb.lo[d] + 0.5f * pb.hi[d];
        const double U = std::sqrt((double)pb.w[d]) * 0.5 * ((double)pb.hi[d] - pb.lo[d]);
        sum_u2 += U * U;
      } else {
        pb.f_ctr[d] = 0.0f;  // weight 0: the feature is 0 whatever the coordinate
      }
    }
    const double s_max = 3.0 * sum_u2 + 2.0 * w_ang;
    if (!(sum_u2 < 3.0e4) || !(s_max > 0.0)) ok = false;  // |u|^2 and every coefficient must fit fp16
    // An angle dim enters through the lower bound w (2 - 2 cos delta) <= w delta^2, loose by up to w (pi^2 - 4): with a
    // heavy angle weight (unicycle heading, Acrobot joints) nearly every chunk stays a candidate, so those problems keep
    // the fp32 scan.  (Exact alternative, not built: two shifted copies of the query per angle dim.)
    if (w_ang > 0.1) ok = false;
    pb.f_qn_ang = (float)(2.0 * w_ang);
    pb.f_eps = (float)(1.0 / 131072.0);
    pl->filter_ok = ok;
  }  // the tier is chosen per call (pakr_plan_opts.nn_mode)
  pb.n_obs = p->n_obstacles;

  // obstacle table in the kernel's shared-memory row format
  const int os = obs == OBS_CIRCLE ? 4 : 8;
  std::vector<float> rows((size_t)std::max(1, p->n_obstacles) * os, 0.0f);
  for (int o = 0; o < p->n_obstacles; ++o) {
    if (obs == OBS_CIRCLE) {
      const float* c = p->obstacles + (size_t)o * 3;
      rows[(size_t)o * 4 + 0] = c[0]; rows[(size_t)o * 4 + 1] = c[1]; rows[(size_t)o * 4 + 2] = c[2] * c[2];
    } else {
      const float* lo = p->obstacles + (size_t)o * 2 * PD;
      const float* hi = lo + PD;
      float* r = &rows[(size_t)o * 8];
      r[0] = lo[0]; r[1] = lo[1]; r[2] = PD == 3 ? lo[2] : -INFINITY; r[3] = 0;
      r[4] = hi[0]; r[5] = hi[1]; r[6] = PD == 3 ? hi[2] : INFINITY; r[7] = 0;
    }
  }
  auto bail = [&](pakr_status st, const std::string& m) { g_create_err = m; pakr_destroy(pl); return st; };
  DeviceGuard guard(cuda_device);
  cudaError_t e = guard.err;
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaSetDevice: ") + cudaGetErrorString(e));
  cudaDeviceProp prop;
  e = cudaGetDeviceProperties(&prop, cuda_device);
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaGetDeviceProperties: ") + cudaGetErrorString(e));
  if (prop.major != 10) return bail(PAKR_ERR_CUDA, "this library is built for sm_100a only");
  if (!prop.cooperativeLaunch) return bail(PAKR_ERR_CUDA, "device lacks cooperative launch");
  pl->num_sms = prop.multiProcessorCount;
  e = cudaMalloc(&pl->d_obstacles, rows.size() * 4);
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaMalloc: ") + cudaGetErrorString(e));
  e = cudaMemcpy(pl->d_obstacles, rows.data(), rows.size() * 4, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaMemcpy: ") + cudaGetErrorString(e));
  pb.obstacles = pl->d_obstacles;
  {
    const HostGrid g = build_grid(p, obs);
    pb.grid_on = g.on ? 1 : 0;
    if (g.on) {
      for (int a = 0; a < 3; ++a) { pb.gdim[a] = g.dim[a]; pb.gorg[a] = g.org[a]; pb.ginv[a] = g.inv[a]; }
      pb.g_cells = (int)g.cells.size();
      pb.g_list = (int)g.list.size();
      e = cudaMalloc(&pl->d_grid_cells, g.cells.size() * 4);
      if (e == cudaSuccess) e = cudaMalloc(&pl->d_grid_list, g.list.size() * 2);
      if (e == cudaSuccess) e = cudaMemcpy(pl->d_grid_cells, g.cells.data(), g.cells.size() * 4, cudaMemcpyHostToDevice);
      if (e == cudaSuccess) e = cudaMemcpy(pl->d_grid_list, g.list.data(), g.list.size() * 2, cudaMemcpyHostToDevice);
      if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("obstacle grid upload: ") + cudaGetErrorString(e));
      pb.grid_cells = pl->d_grid_cells;
      pb.grid_list = pl->d_grid_list;
    }
  }
  pl->kernel = pakr_select_kernel_tiled(dyn, obs);
  pl->kernel_stream = pakr_select_kernel_stream(dyn, obs);
  pl->kernel_index = pakr_select_kernel_index(dyn, obs);
  if (!pl->kernel_index) { pl->kernel_index = pl->kernel; pl->index_ok = false; }  // no index tier for this model
  pl->kernel_filter = pakr_select_kernel_filter(dyn, obs);
  if (!pl->kernel_filter) { pl->kernel_filter = pl->kernel; pl->filter_ok = false; }
  pl->smem_bytes = smem_for(pl);
  e = cudaFuncSetAttribute(pl->kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(pl->kernel_stream, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(pl->kernel_index, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes);
  if (e == cudaSuccess)
    e = cudaFuncSetAttribute(pl->kernel_filter, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)pl->smem_bytes);
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaFuncSetAttribute: ") + cudaGetErrorString(e));
  e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&pl->blocks_per_sm, pl->kernel, kThreads, pl->smem_bytes);
  int occ_stream = 0;
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_stream, pl->kernel_stream, kThreads, pl->smem_bytes);
  int occ_index = 0;
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_index, pl->kernel_index, kThreads, pl->smem_bytes);
  int occ_filter = 0;
  if (e == cudaSuccess) e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_filter, pl->kernel_filter, kThreads, pl->smem_bytes);
  pl->blocks_per_sm = std::min(std::min(pl->blocks_per_sm, occ_filter), std::min(occ_stream, occ_index));  // one grid size for all tiers
  if (e != cudaSuccess || pl->blocks_per_sm < 1)
    return bail(PAKR_ERR_CUDA, "kernel does not fit on an SM (occupancy 0)");
  e = cudaMallocHost(&pl->h_pinned, sizeof(Ctrl) + (size_t)kPathMax * (4 + kMaxD * 4 + kMaxM * 4));
  if (e != cudaSuccess) return bail(PAKR_ERR_CUDA, std::string("cudaMallocHost: ") + cudaGetErrorString(e));
  *out = pl;
  return PAKR_OK;
}

extern "C" void pakr_destroy(pakr_planner* pl) {
  if (!pl) return;
  DeviceGuard guard(pl->device);
  if (pl->d_obstacles) cudaFree(pl->d_obstacles);
  if (pl->d_grid_cells) cudaFree(pl->d_grid_cells);
  if (pl->d_grid_list) cudaFree(pl->d_grid_list);
  if (pl->h_pinned) cudaFreeHost(pl->h_pinned);
  delete pl;
}

extern "C" const char* pakr_last_error(const pakr_planner* pl) { return pl ? pl->err.c_str() : g_create_err.c_str(); }

extern "C" size_t pakr_workspace_bytes(const pakr_planner* pl, int32_t B, int32_t K, int64_t cap) {
  if (!pl || !sizes_ok(B, K, cap)) return 0;
  return make_layout(pl, B, K, cap).total;
}

extern "C" size_t pakr_workspace_bytes_for(const pakr_planner* pl, int32_t B, int32_t K, int64_t cap, int32_t nn_mode) {
  if (!pl || !sizes_ok(B, K, cap) || !nn_mode_ok(nn_mode)) return 0;
  return make_layout(pl, B, K, cap, nn_mode).total;
}

extern "C" pakr_status pakr_get_tree_layout(const pakr_planner* pl, int32_t B, int32_t K, int64_t cap,
                                            pakr_tree_layout* out) {
  if (!pl || !out || !sizes_ok(B, K, cap)) return PAKR_ERR_INVALID_ARG;
  const Layout L = make_layout(pl, B, K, cap);
  out->states_off = L.states; out->actions_off = L.actions; out->parents_off = L.parents; out->costs_off = L.costs;
  out->state_stride = pl->DP; out->action_stride = 4;
  return PAKR_OK;
}

namespace {

void fill_common(const pakr_planner* pl, Params& P, const Layout& L, char* ws, int B, int K, int64_t cap) {
  std::memset(&P, 0, sizeof(P));
  P.pb = pl->pb;
  P.nn_key = reinterpret_cast<unsigned long long*>(ws + L.nn_key);
  P.unit_count = reinterpret_cast<unsigned*>(ws + L.unit_count);
  P.prow = reinterpret_cast<float*>(ws + L.prow);
  P.frow = reinterpret_cast<__half*>(ws + L.frow);
  P.chunkmin = reinterpret_cast<float*>(ws + L.chunkmin);
  P.idx_keys = reinterpret_cast<unsigned*>(ws + L.idx_keys);
  P.idx_ids = reinterpret_cast<int*>(ws + L.idx_ids);
  P.idx_hist = reinterpret_cast<unsigned*>(ws + L.idx_hist);
  P.idx_ctasum = reinterpret_cast<unsigned*>(ws + L.idx_ctasum);
  P.idx_tile_ids = reinterpret_cast<int*>(ws + L.idx_tile_ids);
  P.idx_rows = reinterpret_cast<float*>(ws + L.idx_rows);
  P.idx_tlo = reinterpret_cast<float*>(ws + L.idx_tlo);
  P.idx_thi = reinterpret_cast<float*>(ws + L.idx_thi);
  P.idx_slo = reinterpret_cast<float*>(ws + L.idx_slo);
  P.idx_shi = reinterpret_cast<float*>(ws + L.idx_shi);
  P.scr_state = reinterpret_cast<float*>(ws + L.scr_state);
  P.scr_ctrl = reinterpret_cast<float*>(ws + L.scr_ctrl);
  P.scr_cost = reinterpret_cast<float*>(ws + L.scr_cost);
  P.scr_parent = reinterpret_cast<int*>(ws + L.scr_parent);
  P.scr_flags = reinterpret_cast<int*>(ws + L.scr_flags);
  P.ctrl = reinterpret_cast<Ctrl*>(ws + L.ctrl);
  P.path_nodes_rev = reinterpret_cast<int*>(ws + L.path_rev);
  P.path_nodes = reinterpret_cast<int*>(ws + L.path_nodes);
  P.path_states = reinterpret_cast<float*>(ws + L.path_states);
  P.path_controls = reinterpret_cast<float*>(ws + L.path_controls);
  P.B = B; P.K = K; P.cap = (int)cap;
}

void fill_stats(const Ctrl* hc, int64_t BK, pakr_stats* out) {
  pakr_stats& s = *out;
  std::memset(&s, 0, sizeof(s));
  s.iterations = hc->iterations;
  s.children = hc->iterations * BK;
  s.inserted = hc->inserted;
  s.nn_pairs = hc->nn_pairs;
  s.nn_pairs_evaluated = hc->nn_pairs - hc->nn_idx_covered + (int64_t)hc->nn_scored - hc->nn_filtered + (int64_t)hc->nn_rescored;
  s.nn_pairs_filtered = hc->nn_filtered;
  for (int i = 0; i < 4; ++i) s.phase_ms[i] = (double)hc->phase_ns[i] * 1e-6;
  s.replans_run = hc->replans_run;
  s.replans_solved = hc->replans_solved;
  s.termination = hc->termination;
  s.replan_stats_truncated = hc->replans_run > kStatsMax ? 1 : 0;
  s.path_truncated = hc->path_overflow > 0 ? 1 : 0;
  s.first_solution_ms = hc->replans_solved > 0 ? (double)(hc->t_first_ns - hc->t_start_ns) * 1e-6 : -1.0;
  s.device_ms = (double)(hc->t_end_ns - hc->t_start_ns) * 1e-6;
  for (int i = 0; i < kStatsMax && i < hc->replans_run; ++i) {
    s.replan_cost[i] = hc->replan_cost[i];
    s.replan_nodes[i] = hc->replan_nodes[i];
    s.replan_iters[i] = hc->replan_iters[i];
    s.replan_end_ms[i] = (double)(hc->replan_end_ns[i] - hc->t_start_ns) * 1e-6;
  }
}

// memset of the control words + one cooperative launch; everything on `stream`
// nn_mode (PAKR_NN_*) -> Params::nn_index
bool set_nn_mode(pakr_planner* pl, Params& P, int nn_mode) {
  if (!nn_mode_ok(nn_mode)) return false;
  // PAKR_NN_AUTO (measured on the config 5 sweep and C1-C4): below B = 4096 queries the plain scan
  // kernel -- the trees those batches grow are too small for either accelerator to repay its fixed costs, and both
  // accelerated kernels carry more live state through the 128 registers, so their own scan loop is slower.  From
  // B = 4096 up the spatial index.  The tensor-core filter beats the plain scan from ~10^5 rows up but not the index on
  // the planner's own trees, so it is chosen only explicitly (PAKR_NN_FILTER).
  P.nn_filter = pl->filter_ok && nn_mode == PAKR_NN_FILTER ? 1 : 0;
  P.nn_index = !pl->index_ok ? 0 : nn_mode == PAKR_NN_INDEX ? 2 : (nn_mode == PAKR_NN_AUTO && P.B >= kAutoMinB) ? 1 : 0;
  // The index search addresses its tile rows with 32-bit element offsets (tiles x D x 32 floats).  A capacity whose
  // index would not fit them (~358 M rows at D = 12) keeps the scan tiers: same results, every tier is bit-identical.
  if ((unsigned long long)idx_dims(P.cap).n_super * 1024ull * (unsigned long long)pl->D >= (1ull << 32)) P.nn_index = 0;
  P.filter_min_work = kFilterMinWork;
  P.filter_give_up = kFilterGiveUp;
  P.idx_min_work = kIdxMinWork;
  P.idx_rebuild_work = kIdxRebuildWork;
  return true;
}

pakr_status launch(pakr_planner* pl, Params& P, cudaStream_t stream) {
  CUDA_TRY(pl, cudaMemsetAsync(P.nn_key, 0xFF, (size_t)P.B * 16, stream));
  CUDA_TRY(pl, cudaMemsetAsync(P.ctrl, 0, sizeof(Ctrl), stream));
  static_assert(offsetof(Ctrl, goal_key) == 0, "goal keys first");
  CUDA_TRY(pl, cudaMemsetAsync(P.ctrl, 0xFF, sizeof(unsigned long long) * kSlots, stream));  // goal_key[] = none
  void* args[] = {&P};
  const dim3 grid(pl->num_sms * std::min(pl->blocks_per_sm, kCtasPerSm)), block(kThreads);
  const void* kernel = P.B <= kStreamB ? pl->kernel_stream : P.nn_filter ? pl->kernel_filter : P.nn_index ? pl->kernel_index : pl->kernel;
  CUDA_TRY(pl, cudaLaunchCooperativeKernel(kernel, grid, block, args, pl->smem_bytes, stream));
  return PAKR_OK;
}

}  // namespace

extern "C" pakr_status pakr_plan(pakr_planner* pl, const pakr_plan_opts* o, void* d_ws, size_t ws_bytes,
                                 void* cuda_stream, pakr_result* out) {
  if (!pl) return PAKR_ERR_INVALID_ARG;
  if (!o || !out || !d_ws) return fail(pl, PAKR_ERR_INVALID_ARG, "null opts, result or workspace");
  if (!sizes_ok(o->B, o->K, o->tree_capacity) || o->n_replans < 1 || o->n_replans > 4096 ||
      o->max_iters_per_replan < 0 || o->max_iters_per_replan > (1ll << 30) || out->path_capacity < 0 ||
      std::isnan(o->initial_cost_bound))
    return fail(pl, PAKR_ERR_INVALID_ARG, "B, K, tree_capacity, n_replans or max_iters out of range");
  if (reinterpret_cast<uintptr_t>(d_ws) % kAlign) return fail(pl, PAKR_ERR_INVALID_ARG, "workspace must be 256-byte aligned");
  if (!nn_mode_ok(o->nn_mode)) return fail(pl, PAKR_ERR_INVALID_ARG, "nn_mode must be a PAKR_NN_* value");
  const Layout L = make_layout(pl, o->B, o->K, o->tree_capacity, o->nn_mode);
  if (ws_bytes < L.total) return fail(pl, PAKR_ERR_WORKSPACE_TOO_SMALL, "workspace smaller than pakr_workspace_bytes_for() of this nn_mode");
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  char* ws = static_cast<char*>(d_ws);
  Params P;
  fill_common(pl, P, L, ws, o->B, o->K, o->tree_capacity);
  if (!set_nn_mode(pl, P, o->nn_mode)) return fail(pl, PAKR_ERR_INVALID_ARG, "nn_mode must be a PAKR_NN_* value");
  pl->err.clear();
  DeviceGuard guard(pl->device);
  CUDA_TRY(pl, guard.err);
  P.states = reinterpret_cast<float*>(ws + L.states);
  P.actions = reinterpret_cast<float*>(ws + L.actions);
  P.parents = reinterpret_cast<int*>(ws + L.parents);
  P.costs = reinterpret_cast<float*>(ws + L.costs);
  P.seed = o->seed;
  P.n_replans = o->n_replans;
  const int64_t BK = (int64_t)o->B * o->K;
  int64_t mi = o->max_iters_per_replan > 0 ? o->max_iters_per_replan : std::max<int64_t>(32, o->tree_capacity / BK);
  P.max_iters = (int)mi;
  P.budget_ns = o->time_budget_ms > 0 ? (unsigned long long)(o->time_budget_ms * 1e6) : 0ull;
  P.r0 = 0; P.it0 = 0;
  P.c_best0 = (o->initial_cost_bound > 0.0 && std::isfinite(o->initial_cost_bound)) ? (float)o->initial_cost_bound : INFINITY;
  P.early_exit = 1;
  // Alg. 1 l.4: root node (x_init, no action, parent -1, cost 0); rewritten never, read by every replan
  float root[kMaxD + kMaxM + 2] = {0};
  for (int d = 0; d < pl->D; ++d) root[d] = pl->pb.start[d];
  const int minus1 = -1;
  CUDA_TRY(pl, cudaMemcpyAsync(P.states, root, (size_t)pl->DP * 4, cudaMemcpyHostToDevice, stream));
  CUDA_TRY(pl, cudaMemsetAsync(P.actions, 0, 16, stream));
  CUDA_TRY(pl, cudaMemcpyAsync(P.parents, &minus1, 4, cudaMemcpyHostToDevice, stream));
  CUDA_TRY(pl, cudaMemsetAsync(P.costs, 0, 4, stream));
  pakr_status st = launch(pl, P, stream);
  if (st != PAKR_OK) return st;
  Ctrl* hc = static_cast<Ctrl*>(pl->h_pinned);
  CUDA_TRY(pl, cudaMemcpyAsync(hc, P.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, stream));
  CUDA_TRY(pl, cudaStreamSynchronize(stream));
  // results
  fill_stats(hc, BK, &out->stats);
  out->stats.h2d_bytes = (int64_t)pl->DP * 4 + 4;
  out->stats.d2h_bytes = (int64_t)sizeof(Ctrl);
  out->final_tree_nodes = hc->n_nodes;
  out->outcome = hc->solved ? PAKR_SOLVED : PAKR_NO_SOLUTION;
  out->cost = hc->solved ? (double)hc->best_cost : (double)INFINITY;
  out->path_len = hc->solved ? hc->path_len : 0;
  if (!hc->solved) return PAKR_OK;
  if (hc->path_overflow > 0) {
    // a path of more than PAKR_MAX_PATH_NODES nodes tightened c_best but was not extracted: hand back the last
    // path that fit, with ITS cost; if none did, say how long the buffers would have had to be
    if (hc->path_len == 0) {
      out->path_len = hc->path_overflow;
      return fail(pl, PAKR_ERR_BUFFER_TOO_SMALL, "best path exceeds PAKR_MAX_PATH_NODES nodes");
    }
    out->cost = (double)hc->path_cost;
    pl->err = "a cheaper path exceeded PAKR_MAX_PATH_NODES nodes; the last path that fit is returned (stats.path_truncated)";
  }
  if (hc->path_len > out->path_capacity) {
    if (out->path_nodes || out->path_states || out->path_controls)
      return fail(pl, PAKR_ERR_BUFFER_TOO_SMALL, "path longer than path_capacity");
    return PAKR_OK;
  }
  const int Lp = hc->path_len;
  char* stage = static_cast<char*>(pl->h_pinned) + sizeof(Ctrl);
  int* h_nodes = reinterpret_cast<int*>(stage);
  float* h_states = reinterpret_cast<float*>(stage + (size_t)kPathMax * 4);
  float* h_ctrls = h_states + (size_t)kPathMax * kMaxD;
  if (out->path_nodes) CUDA_TRY(pl, cudaMemcpyAsync(h_nodes, P.path_nodes, (size_t)Lp * 4, cudaMemcpyDeviceToHost, stream));
  if (out->path_states) CUDA_TRY(pl, cudaMemcpyAsync(h_states, P.path_states, (size_t)Lp * pl->D * 4, cudaMemcpyDeviceToHost, stream));
  if (out->path_controls && Lp > 1)
    CUDA_TRY(pl, cudaMemcpyAsync(h_ctrls, P.path_controls, (size_t)(Lp - 1) * pl->M * 4, cudaMemcpyDeviceToHost, stream));
  CUDA_TRY(pl, cudaStreamSynchronize(stream));
  out->stats.d2h_bytes += (out->path_nodes ? (int64_t)Lp * 4 : 0) + (out->path_states ? (int64_t)Lp * pl->D * 4 : 0) +
                          (out->path_controls && Lp > 1 ? (int64_t)(Lp - 1) * pl->M * 4 : 0);
  if (out->path_nodes) std::memcpy(out->path_nodes, h_nodes, (size_t)Lp * 4);
  if (out->path_states) std::memcpy(out->path_states, h_states, (size_t)Lp * pl->D * 4);
  if (out->path_controls && Lp > 1) std::memcpy(out->path_controls, h_ctrls, (size_t)(Lp - 1) * pl->M * 4);
  return PAKR_OK;
}

extern "C" pakr_status pakr_expand_step(pakr_planner* pl, const pakr_step_args* a, void* d_ws, size_t ws_bytes,
                                        void* cuda_stream) {
  if (!pl) return PAKR_ERR_INVALID_ARG;
  if (!a || !d_ws) return fail(pl, PAKR_ERR_INVALID_ARG, "null args or workspace");
  if (!sizes_ok(a->B, a->K, a->tree_capacity)) return fail(pl, PAKR_ERR_INVALID_ARG, "B, K or tree_capacity out of range");
  if (!a->states || !a->actions || !a->parents || !a->costs || !a->n_nodes)
    return fail(pl, PAKR_ERR_INVALID_ARG, "null tree pointer");
  if (std::isnan(a->c_best)) return fail(pl, PAKR_ERR_INVALID_ARG, "c_best is NaN");
  if (reinterpret_cast<uintptr_t>(d_ws) % kAlign || reinterpret_cast<uintptr_t>(a->states) % 16 ||
      reinterpret_cast<uintptr_t>(a->actions) % 16)
    return fail(pl, PAKR_ERR_INVALID_ARG, "workspace must be 256-byte, states/actions 16-byte aligned");
  if (!nn_mode_ok(a->nn_mode)) return fail(pl, PAKR_ERR_INVALID_ARG, "nn_mode must be a PAKR_NN_* value");
  const Layout L = make_layout(pl, a->B, a->K, a->tree_capacity, a->nn_mode);
  if (ws_bytes < L.total) return fail(pl, PAKR_ERR_WORKSPACE_TOO_SMALL, "workspace smaller than pakr_workspace_bytes_for() of this nn_mode");
  Params P;
  fill_common(pl, P, L, static_cast<char*>(d_ws), a->B, a->K, a->tree_capacity);
  if (!set_nn_mode(pl, P, a->nn_mode)) return fail(pl, PAKR_ERR_INVALID_ARG, "nn_mode must be a PAKR_NN_* value");
  DeviceGuard guard(pl->device);
  CUDA_TRY(pl, guard.err);
  P.states = a->states; P.actions = a->actions; P.parents = a->parents; P.costs = a->costs;
  P.seed = a->seed;
  P.n_replans = 1; P.max_iters = 1; P.budget_ns = 0;
  P.r0 = (int)a->replan; P.it0 = (int)a->iteration;
  P.c_best0 = a->c_best;
  P.early_exit = 0;
  P.n_nodes_io = a->n_nodes;
  P.dbg_x_rand = a->x_rand; P.dbg_nn_idx = a->nn_idx; P.dbg_nn_d2 = a->nn_d2;
  P.dbg_child_state = a->child_state; P.dbg_child_ctrl = a->child_ctrl; P.dbg_child_cost = a->child_cost;
  P.dbg_child_flags = a->child_flags; P.dbg_n_inserted = a->n_inserted; P.dbg_goal_node = a->goal_node;
  P.dbg_new_c_best = a->new_c_best;
  return launch(pl, P, reinterpret_cast<cudaStream_t>(cuda_stream));
}

extern "C" pakr_status pakr_read_stats(pakr_planner* pl, int32_t B, int32_t K, int64_t cap, void* d_ws,
                                       size_t ws_bytes, void* cuda_stream, pakr_stats* out) {
  if (!pl) return PAKR_ERR_INVALID_ARG;
  if (!d_ws || !out || !sizes_ok(B, K, cap)) return fail(pl, PAKR_ERR_INVALID_ARG, "null pointer or sizes out of range");
  const Layout L = make_layout(pl, B, K, cap, PAKR_NN_SCAN);  // the control block sits at the same offset in every mode
  if (ws_bytes < L.total) return fail(pl, PAKR_ERR_WORKSPACE_TOO_SMALL, "workspace smaller than pakr_workspace_bytes_for(PAKR_NN_SCAN)");
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  Ctrl* hc = static_cast<Ctrl*>(pl->h_pinned);
  DeviceGuard guard(pl->device);
  CUDA_TRY(pl, guard.err);
  CUDA_TRY(pl, cudaMemcpyAsync(hc, static_cast<char*>(d_ws) + L.ctrl, sizeof(Ctrl), cudaMemcpyDeviceToHost, stream));
  CUDA_TRY(pl, cudaStreamSynchronize(stream));
  fill_stats(hc, (int64_t)B * K, out);
  return PAKR_OK;
}

// ---- pakr_expand_step_static: one iteration with the scratch inside the library image (include/pakr.h) ----------------
//
// For callers that may not allocate device memory once they are running (control loops with deadlines, plug-ins inside a
// host whose pool owns the device).  The scratch below is part of libpakr.so's device image: the driver places one copy
// on every GPU that loads the library and keeps it until the process exits.  Nothing here calls cudaMalloc / cudaFree.
//
// g_static_scratch, as host code sees it, is only a handle for the symbol -- NOT a device address.  Passing
// `g_static_scratch` itself to a kernel would hand it a host pointer (a fault, or on machines where the GPU can reach
// host memory, silent use of the wrong bytes).  The device address is asked for once per device with
// cudaGetSymbolAddress while that device is current, and that is the pointer the kernel parameters are built from.
static __device__ __align__(256) unsigned char g_static_scratch[PAKR_STATIC_SCRATCH_BYTES];

namespace {

constexpr int kStaticMaxDevices = 64;
std::mutex g_static_mu;
void* g_static_ptr[kStaticMaxDevices] = {nullptr};  // device address of g_static_scratch on device i, once known

// Scratch of one tiled-scan iteration, packed from offset 0: what make_layout() reserves minus the tree (the caller's)
// and minus the per-node copies of the streaming / index / filter tiers (never used here).
Layout make_static_layout(const pakr_planner* pl, int64_t B, int64_t K) {
  Layout L{};
  size_t o = 0;
  auto take = [&](size_t bytes) { size_t at = o; o = align_up(o + bytes); return at; };
  const size_t BK = (size_t)B * K, slots = BK + 32;
  L.nn_key = take((size_t)B * 16);
  L.unit_count = take(std::max<size_t>(BK, kFuseUnits + 8) * 4);
  L.scr_state = take(slots * pl->DP * 4);
  L.scr_ctrl = take(slots * 16);
  L.scr_cost = take(slots * 4);
  L.scr_parent = take(slots * 4);
  L.scr_flags = take(slots * 4);
  L.ctrl = take(sizeof(Ctrl));
  L.path_rev = take((size_t)kPathMax * 4);
  L.path_nodes = take((size_t)kPathMax * 4);
  L.path_states = take((size_t)kPathMax * kMaxD * 4);
  L.path_controls = take((size_t)kPathMax * kMaxM * 4);
  L.total = o;
  return L;
}

}  // namespace

extern "C" pakr_status pakr_expand_step_static(pakr_planner* pl, const pakr_step_args* a, void* cuda_stream) {
  if (!pl) return PAKR_ERR_INVALID_ARG;
  if (!a) return fail(pl, PAKR_ERR_INVALID_ARG, "null args");
  if (!sizes_ok(a->B, a->K, a->tree_capacity)) return fail(pl, PAKR_ERR_INVALID_ARG, "B, K or tree_capacity out of range");
  if ((int64_t)a->B * a->K > PAKR_STATIC_MAX_CHILDREN)
    return fail(pl, PAKR_ERR_INVALID_ARG,
                "B*K = " + std::to_string((int64_t)a->B * a->K) + " exceeds the static scratch (PAKR_STATIC_MAX_CHILDREN = " +
                    std::to_string(PAKR_STATIC_MAX_CHILDREN) + "); use pakr_expand_step with a workspace");
  if (a->nn_mode != PAKR_NN_AUTO && a->nn_mode != PAKR_NN_SCAN)
    return fail(pl, PAKR_ERR_UNSUPPORTED, "pakr_expand_step_static runs the tiled fp32 scan only (nn_mode AUTO or SCAN)");
  if (!a->states || !a->actions || !a->parents || !a->costs || !a->n_nodes)
    return fail(pl, PAKR_ERR_INVALID_ARG, "null tree pointer");
  if (std::isnan(a->c_best)) return fail(pl, PAKR_ERR_INVALID_ARG, "c_best is NaN");
  if (reinterpret_cast<uintptr_t>(a->states) % 16 || reinterpret_cast<uintptr_t>(a->actions) % 16)
    return fail(pl, PAKR_ERR_INVALID_ARG, "states/actions must be 16-byte aligned");
  const Layout L = make_static_layout(pl, a->B, a->K);
  if (L.total > (size_t)PAKR_STATIC_SCRATCH_BYTES)  // cannot happen below PAKR_STATIC_MAX_CHILDREN; kept as the real guard
    return fail(pl, PAKR_ERR_INVALID_ARG, "scratch for this (B, K) exceeds PAKR_STATIC_SCRATCH_BYTES");
  if (pl->device < 0 || pl->device >= kStaticMaxDevices)
    return fail(pl, PAKR_ERR_UNSUPPORTED, "static scratch is tracked for device ordinals 0..63 only");
  DeviceGuard guard(pl->device);
  CUDA_TRY(pl, guard.err);
  char* ws = nullptr;
  {
    // set-up, once per device, with that device current: the symbol's address ON THIS DEVICE
    std::lock_guard<std::mutex> lock(g_static_mu);
    if (!g_static_ptr[pl->device]) {
      void* ptr = nullptr;
      CUDA_TRY(pl, cudaGetSymbolAddress(&ptr, g_static_scratch));
      if (!ptr || reinterpret_cast<uintptr_t>(ptr) % kAlign) return fail(pl, PAKR_ERR_CUDA, "static scratch has no usable device address");
      g_static_ptr[pl->device] = ptr;
    }
    ws = static_cast<char*>(g_static_ptr[pl->device]);
  }
  Params P;
  fill_common(pl, P, L, ws, a->B, a->K, a->tree_capacity);
  // tiers that keep per-node copies are off; their pointers must never be followed
  P.prow = nullptr; P.frow = nullptr; P.chunkmin = nullptr;
  P.idx_keys = nullptr; P.idx_ids = nullptr; P.idx_hist = nullptr; P.idx_ctasum = nullptr; P.idx_tile_ids = nullptr;
  P.idx_rows = nullptr; P.idx_tlo = nullptr; P.idx_thi = nullptr; P.idx_slo = nullptr; P.idx_shi = nullptr;
  P.nn_index = 0; P.nn_filter = 0;
  P.filter_min_work = kFilterMinWork; P.filter_give_up = kFilterGiveUp;
  P.idx_min_work = kIdxMinWork; P.idx_rebuild_work = kIdxRebuildWork;
  P.states = a->states; P.actions = a->actions; P.parents = a->parents; P.costs = a->costs;
  P.seed = a->seed;
  P.n_replans = 1; P.max_iters = 1; P.budget_ns = 0;
  P.r0 = (int)a->replan; P.it0 = (int)a->iteration;
  P.c_best0 = a->c_best;
  P.early_exit = 0;
  P.n_nodes_io = a->n_nodes;
  P.dbg_x_rand = a->x_rand; P.dbg_nn_idx = a->nn_idx; P.dbg_nn_d2 = a->nn_d2;
  P.dbg_child_state = a->child_state; P.dbg_child_ctrl = a->child_ctrl; P.dbg_child_cost = a->child_cost;
  P.dbg_child_flags = a->child_flags; P.dbg_n_inserted = a->n_inserted; P.dbg_goal_node = a->goal_node;
  P.dbg_new_c_best = a->new_c_best;
  // The array holds the previous call's bytes.  What the kernel expects to find reset: NN keys = "none" (all ones),
  // control block = 0 with its goal keys = "none".  Everything else in the scratch is written before it is read.
  cudaStream_t stream = reinterpret_cast<cudaStream_t>(cuda_stream);
  CUDA_TRY(pl, cudaMemsetAsync(P.nn_key, 0xFF, (size_t)P.B * 16, stream));
  CUDA_TRY(pl, cudaMemsetAsync(P.ctrl, 0, sizeof(Ctrl), stream));
  CUDA_TRY(pl, cudaMemsetAsync(P.ctrl, 0xFF, sizeof(unsigned long long) * kSlots, stream));
  void* args[] = {&P};
  const dim3 grid(pl->num_sms * std::min(pl->blocks_per_sm, kCtasPerSm)), block(kThreads);
  CUDA_TRY(pl, cudaLaunchCooperativeKernel(pl->kernel, grid, block, args, pl->smem_bytes, stream));  // tiled tier, any B
  return PAKR_OK;
}
