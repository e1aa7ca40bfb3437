// pakr_kernel.cuh -- the persistent cooperative kernel that runs Alg. 1 on device.
//
// One launch = the whole AO-x loop (or one iteration for pakr_expand_step).  Per iteration i, when the children
// are few (the usual case):
//   phase X, one grid barrier at its end
//     propagate CTAs: propagate(i)  (Alg. 1 l.8-12)  one lane per child, state in registers, obstacles and
//                                     their broad-phase grid in shared memory, ballot compaction to scratch
//                     barrier among themselves, then
//                     insert(i)     (Alg. 1 l.13-15) ordered prefix of survivor counts, append at the tree
//                                     tail, goal winner by atomicMin
//                     tail of NN(i+1) over the rows just appended (TMA gather from the scratch rows)
//     scan CTAs:      NN(i+1) over the frozen snapshot [0, n_i)  (Alg. 1 l.6-7): warps own 32*Q queries in
//                                     registers, tree tiles stream into shared memory by TMA bulk copies
//                                     (speculative: dropped when iteration i ends the replan)
// NN(i+1) = min(scan of [0, n_i), scan of [n_i, n_{i+1})): the snapshot a batch sees is exactly the tree after
// the previous batch's inserts.  Large batches of new rows get a tail-scan phase of their own
// ("A'"), and with many children every warp propagates, then scans, and the insert is a phase of its own.
// Loop state (n, c_best, replan, iteration) is replicated in registers of every thread and
// recomputed from the same global values, so no broadcast step is needed.
#pragma once
#include <cooperative_groups.h>

#include <cuda_fp16.h>

#include "pakr_device.cuh"

namespace pakr {
namespace cg = cooperative_groups;

constexpr int kThreads = 256;    // 256 x 2 CTAs per SM measured 1.4x faster in the NN scan than 512 x 1
constexpr int kCtasPerSm = 2;
constexpr int kWarps = kThreads / 32;
constexpr int kQ = 4;            // queries per lane in the NN scan
constexpr int kIdxMinRows = 4096;    // NN index: smaller trees are scanned
constexpr long long kIdxMinWork = 2400000000ll;  // ... and so are iterations whose scan (B*n*D) takes less than ~250 us:
                                                 // measured crossover of scan vs rebuilds + search on config 5's trees
constexpr long long kIdxRebuildWork = 400000000ll;  // rebuild once scanning the rows added since the last rebuild costs
                                                    // about as much as rebuilding: B * rows * D lane-ops (~50 us)
constexpr int kPathMax = 8192;   // longest path the device buffers hold
constexpr int kStatsMax = 64;
constexpr unsigned long long kKeyNone = ~0ull;

// Per-iteration words the whole grid reads right after the barrier that ends iteration i live in slot i % 3:
// slot (i+1) % 3 is re-armed during iteration i, and its last readers (iteration i-2's) all passed the barrier of
// iteration i-1 before that, so no read can ever see a later iteration's value.
constexpr int kSlots = 3;

struct Ctrl {  // device control block (in the workspace)
  unsigned long long goal_key[kSlots];  // min (cost bits, node) over the goal children inserted in the iteration
  unsigned long long t_start_ns, t_first_ns, t_end_ns;
  long long iterations, inserted, nn_pairs;
  unsigned long long nn_scored;  // (query, row) pairs the NN index tier scored, summed over its warps
  long long nn_idx_covered;      // sum over iterations of B * (rows the index answered for): pairs NOT scanned
  long long nn_filtered;         // (query, row) pairs the tensor-core filter answered approximately
  unsigned long long nn_rescored;         // ... and the rows its second phase rescored exactly, summed over the launch
  unsigned long long f_rescored[kSlots];  // the same per iteration (slot rotation as goal_key)
  unsigned long long phase_ns[4];  // leader's time in NN / propagate / insert (incl. the grid sync after each) / index rebuilds
  int n_nodes;
  int stop[kSlots];        // 1: the time budget ran out during the iteration (written by the leader every iteration)
  unsigned pbar;           // arrival counter of the barrier among the propagate CTAs (insert inside phase X)
  unsigned sbar;           // ... and of the one among the scan CTAs (between the two phases of the tensor-core NN filter)
  int iter_total[kSlots];  // survivors of the iteration, published by CTA 0 when the insert ran inside phase X
  int idx_query[2][kSlots];// NN index tier: next query to hand out ([0] whole-tree NN of the iteration, [1] look-ahead)
  int path_len, solved;
  int path_overflow;       // a solved replan's path was longer than kPathMax and was not extracted
  float path_cost;         // cost of the path held in the path buffers
  float best_cost;
  int replans_run, replans_solved, termination;
  float replan_cost[kStatsMax];
  int replan_nodes[kStatsMax];
  int replan_iters[kStatsMax];
  unsigned long long replan_end_ns[kStatsMax];
};

struct Params {
  DevProblem pb;
  // tree
  float* states; float* actions; int* parents; float* costs;
  // per-iteration work buffers
  unsigned long long* nn_key;  // [2][B] (d2 bits << 32) | node, combined with atomicMin; two iterations in flight
  // NN cell index (exact spatial pruning): tree rows [0, n_sorted) bucketed by position cell
  int nn_index;                // 0: scan tiers only; 1: index when B*n is large; 2: index whenever n >= 256 (tests)
  long long idx_min_work, idx_rebuild_work;  // thresholds of nn_index == 1 (kIdxMinWork, kIdxRebuildWork)
  long long filter_min_work; int filter_give_up;  // kFilterMinWork, kFilterGiveUp
  unsigned* idx_keys;          // [2][cap] Morton keys (radix-sort ping-pong)
  int* idx_ids;                // [2][cap] row ids, sorted together with the keys
  unsigned* idx_hist;          // [kIdxBins][sorting warps] digit histogram / scatter offsets
  unsigned* idx_ctasum;        // [CTAs] partial sums of the histogram scan
  int* idx_tile_ids;           // [tiles][32] row id of every tile slot (-1: padding)
  float* idx_rows;             // [tiles][D][32] the sorted rows, dimension-major inside a tile
  float* idx_tlo; float* idx_thi;  // [super-tiles][D][32] boxes of the tiles
  float* idx_slo; float* idx_shi;  // [groups][D][32] boxes of the super-tiles
  float* prow;                 // streaming tier: [cap + 4][D] the tree rows packed without pad lanes
  // tensor-core NN filter (pakr_nn_filter.cuh)
  int nn_filter;               // host: 1 = launch the filter tier's kernel
  __half* frow;                // [cap + 8][K halves] filter rows of the tree
  float* chunkmin;             // [B][kFilterMaxChunks] minimum approximate key per (query, row range)
  unsigned* unit_count;        // [ceil(B*K/32)] survivors per warp unit
  float* scr_state; float* scr_ctrl; float* scr_cost; int* scr_parent; int* scr_flags;
  Ctrl* ctrl;
  int* path_nodes_rev; int* path_nodes; float* path_states; float* path_controls;
  // loop
  unsigned long long seed;
  int B, K;
  int cap;
  int n_replans;
  int max_iters;
  unsigned long long budget_ns;  // 0 = none
  int r0, it0;
  float c_best0;
  int early_exit;
  int* n_nodes_io;               // expand_step: tree size in/out (else NULL: start from the root)
  // expand_step debug outputs (NULL in pakr_plan)
  float* dbg_x_rand; int* dbg_nn_idx; float* dbg_nn_d2; float* dbg_child_state; float* dbg_child_ctrl;
  float* dbg_child_cost; int* dbg_child_flags; int* dbg_n_inserted; int* dbg_goal_node;
  float* dbg_new_c_best;
};

__device__ __forceinline__ unsigned long long globaltimer_ns() {
  unsigned long long t;
  asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
  return t;
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return (uint32_t)__cvta_generic_to_shared(p);
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, int count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity)
      : "memory");
}
// TMA 1-D bulk copy global -> shared, completion counted on an mbarrier (SASS: UBLKCP).
__device__ __forceinline__ void tma_load_1d(void* dst, const void* src, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
          smem_u32(dst)),
      "l"(src), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async;" ::: "memory"); }

// Barrier among a subset of the (co-resident, cooperative-launch) CTAs: monotonic counter, `target` = number
// of participants x generation.  Same release / acquire pattern as the cooperative-groups grid barrier.
__device__ __forceinline__ void cta_group_barrier(unsigned* ctr, unsigned target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(ctr, 1u);
    while ((int)(*reinterpret_cast<volatile unsigned*>(ctr) - target) < 0) {}  // wrap-safe
    __threadfence();
  }
  __syncthreads();
}

constexpr int kTileBufFloats = 1024;  // every TMA tile buffer is 4 KB (two per warp)
template <int DYN> struct TileCfg {  // nodes per TMA tile: <= 4 KB per buffer
  static constexpr int DP = DynTraits<DYN>::DP;
  static constexpr int TILE = ((DP == 4) ? 256 : (DP == 8) ? 128 : 64) ; 
  static constexpr int TILE_FLOATS = TILE * DP;
};

// squared weighted distance between a query (registers) and a node (shared memory row p)
template <int DYN, bool UNIT_W>
__device__ __forceinline__ float dist2(const DevProblem& pb, const float (&q)[DynTraits<DYN>::D],
                                       const float (&p)[DynTraits<DYN>::DP]) {
  constexpr int D = DynTraits<DYN>::D;
  float acc = 0.0f;
#pragma unroll
  for (int d = 0; d < D; ++d) {
    const float delta = is_angle<DYN>(d) ? angle_absdiff(q[d], p[d]) : (q[d] - p[d]);
    if (UNIT_W) acc = fmaf(delta, delta, acc);
    else acc = fmaf(delta * pb.w[d], delta, acc);
  }
  return acc;
}

// Packed pairs of fp32 (Blackwell f32x2 instructions, SASS FADD2 / FFMA2): one issue slot does the arithmetic
// of two queries; every component is rounded exactly like the scalar instruction, so results are bit-identical.
typedef unsigned long long f32x2;
__device__ __forceinline__ f32x2 pack2(float lo, float hi) {
  f32x2 r;
  asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
  return r;
}
__device__ __forceinline__ void unpack2(f32x2 v, float& lo, float& hi) {
  asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v));
}
__device__ __forceinline__ f32x2 sub2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 mul2(f32x2 a, f32x2 b) {
  f32x2 r;
  asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
  return r;
}
__device__ __forceinline__ f32x2 fma2(f32x2 a, f32x2 b, f32x2 c) {
  f32x2 r;
  asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
  return r;
}

// squared weighted distances of two queries (packed) to one node; same operations per component as dist2()
template <int DYN, bool UNIT_W>
__device__ __forceinline__ void dist2x2(const DevProblem& pb, const f32x2 (&q2)[DynTraits<DYN>::D],
                                        const float (&p)[DynTraits<DYN>::DP], float& d_lo, float& d_hi) {
  constexpr int D = DynTraits<DYN>::D;
  f32x2 acc = pack2(0.0f, 0.0f);
#pragma unroll
  for (int d = 0; d < D; ++d) {
    f32x2 delta;
    if (is_angle<DYN>(d)) {
      float qa, qb;
      unpack2(q2[d], qa, qb);
      delta = pack2(angle_absdiff(qa, p[d]), angle_absdiff(qb, p[d]));
    } else {
      delta = sub2(q2[d], pack2(p[d], p[d]));
    }
    if (UNIT_W) acc = fma2(delta, delta, acc);
    else acc = fma2(mul2(delta, pack2(pb.w[d], pb.w[d])), delta, acc);
  }
  unpack2(acc, d_lo, d_hi);
}

// Scores `cnt` rows of a shared-memory tile (node ids base, base+1, ...) against the lane's kQ queries.
template <int DYN, bool UNIT_W>
__device__ __forceinline__ void scan_rows(const DevProblem& pb, const float4* __restrict__ tp, int cnt, int base,
                                          const f32x2 (&q2)[kQ / 2][DynTraits<DYN>::D], float (&best)[kQ],
                                          int (&bidx)[kQ]) {
  constexpr int DP = DynTraits<DYN>::DP;
  float4 nx[DP / 4];  // row i+1 is fetched while row i is scored (hides the shared-memory latency)
#pragma unroll
  for (int v = 0; v < DP / 4; ++v) nx[v] = tp[v];
#pragma unroll 2
  for (int i = 0; i < cnt; ++i) {
    float p[DP];
#pragma unroll
    for (int v = 0; v < DP / 4; ++v) {
      p[4 * v] = nx[v].x; p[4 * v + 1] = nx[v].y; p[4 * v + 2] = nx[v].z; p[4 * v + 3] = nx[v].w;
    }
    const int in = min(i + 1, cnt - 1);
#pragma unroll
    for (int v = 0; v < DP / 4; ++v) nx[v] = tp[in * (DP / 4) + v];  // warp-uniform address: broadcast
#pragma unroll
    for (int h = 0; h < kQ / 2; ++h) {
      float da, db;
      dist2x2<DYN, UNIT_W>(pb, q2[h], p, da, db);
      if (da < best[2 * h]) { best[2 * h] = da; bidx[2 * h] = base + i; }  // strict <: lowest index wins
      if (db < best[2 * h + 1]) { best[2 * h + 1] = db; bidx[2 * h + 1] = base + i; }
    }
  }
}

// ---- streaming tier of the NN scan: few queries (B <= kStreamB) -------------------------------------
// With only a handful of queries sharing one pass over the tree the scan is HBM-bound, not ALU-bound
// (DESIGN.md "Kernels"): here every LANE owns tree rows (each warp streams one contiguous chunk of the
// tree through its double-buffered TMA tiles) and the queries sit in registers; a warp-level min per query
// and one atomicMin per (warp, query) finish it.  Same per-pair arithmetic (dist2x2) and the same
// (d2, index) ordering as the tiled tier, so both tiers return identical results.
constexpr int kStreamB = 16;

template <int DYN, bool UNIT_W, int QS>  // QS: query slots held in registers per pass over the rows
__device__ __forceinline__ void nn_stream(const Params& P, int nbeg, int nend, uint32_t r, uint32_t it,
                                       unsigned long long* key, int vb, int vbcount, float* sm_q,
                                          float* sm_tile, uint64_t* sm_bar, uint32_t& par0, uint32_t& par1, uint32_t& parx) {
  constexpr int D = DynTraits<DYN>::D, DP = DynTraits<DYN>::DP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  __syncthreads();  // earlier readers of sm_q are done
  for (int t = threadIdx.x; t < P.B; t += kThreads) {
    float x[D];
    sample_state<D>(P.pb, P.seed, r, it, (uint32_t)t, x);
#pragma unroll
    for (int d = 0; d < D; ++d) sm_q[t * D + d] = x[d];
    if (vb == 0) {
#pragma unroll
      for (int d = 0; d < DP; ++d) {
        if (P.dbg_x_rand && nbeg == 0) P.dbg_x_rand[(size_t)t * DP + d] = d < D ? x[d] : 0.0f;
      }
    }
  }
  __syncthreads();
  // The rows come from the PACKED copy of the tree (D floats per row, no pad lanes): every byte that crosses HBM is a
  // coordinate, 4 D n per pass -- the algorithmic figure of SURVEY.md 8(d).  Tiles are whole rows; a tile starts at a
  // multiple of 4 rows and carries a multiple of 4 rows so that every bulk copy is 16-byte aligned and sized.
  // A CTA streams ONE contiguous chunk of rows; its warps take the chunk's tiles round robin (warp w: tiles w, w + 8,
  // ...), so the eight bulk copies a CTA has in flight cover one contiguous 24-32 KB stretch of HBM instead of eight
  // separate streams.  Tiles hold a multiple of 32 rows (every lane of the row loop busy), at most 4 KB, two buffers
  // per warp.  Inside a tile lane l scores rows l, l+32, ...: ascending per lane over the whole call.
  constexpr int NS = 2, BUF = kTileBufFloats;
  constexpr int TILE = ((BUF / D) & ~31), TF = TILE * D;
  const int base = nbeg & ~3;
  const int span = nend - base;
  const int cchunk = ((span + vbcount - 1) / vbcount + TILE - 1) / TILE * TILE;  // rows per CTA: whole tiles
  const int cb = base + min(span, vb * cchunk), ce = base + min(span, (vb + 1) * cchunk);
  const int ctiles = (ce - cb + TILE - 1) / TILE;
  const int ntiles = ctiles > warp ? (ctiles - warp + kWarps - 1) / kWarps : 0;  // this warp's tiles
  const float* src = P.prow + (size_t)cb * D;
  auto issue = [&](int t) {  // lane 0: bulk copy of this warp's t-th tile into stage t % NS
    const int st = t % NS, T = t * kWarps + warp;
    const uint32_t bytes = (uint32_t)((min(TILE, ce - cb - T * TILE) + 3) & ~3) * D * 4;
    mbar_expect_tx(&sm_bar[st], bytes);
    tma_load_1d(sm_tile + st * BUF, src + (size_t)T * TF, bytes, &sm_bar[st]);
  };
  for (int q0 = 0; q0 < P.B; q0 += QS) {
    f32x2 q2[QS / 2][D];
    float best[QS];
    int bidx[QS];
#pragma unroll
    for (int h = 0; h < QS / 2; ++h) {
      const int sa = min(q0 + 2 * h, P.B - 1), sb = min(q0 + 2 * h + 1, P.B - 1);
#pragma unroll
      for (int d = 0; d < D; ++d) q2[h][d] = pack2(sm_q[sa * D + d], sm_q[sb * D + d]);
    }
#pragma unroll
    for (int j = 0; j < QS; ++j) { best[j] = __int_as_float(0x7f800000); bidx[j] = 0x7fffffff; }
    if (lane == 0)
      for (int t = 0; t < min(NS - 1, ntiles); ++t) issue(t);
    for (int t = 0; t < ntiles; ++t) {
      const int T = t * kWarps + warp;
      const int cnt = min(TILE, ce - cb - T * TILE);
      if (t + NS - 1 < ntiles && lane == 0) issue(t + NS - 1);  // into the stage tile t-1 left (syncwarp below)
      const int st = t % NS;
      if (st == 0) { mbar_wait(&sm_bar[0], par0); par0 ^= 1; }
      else { mbar_wait(&sm_bar[1], par1); par1 ^= 1; }
      const float* tp = sm_tile + st * BUF;
#pragma unroll 2
      for (int i = lane; i < cnt; i += 32) {
        float p[DP];
        if constexpr (D % 2 == 0) {  // 8-byte aligned rows: LDS.64, conflict-free per half-warp (row stride D words)
          const float2* rp = reinterpret_cast<const float2*>(tp + i * D);
#pragma unroll
          for (int v = 0; v < D / 2; ++v) { const float2 a = rp[v]; p[2 * v] = a.x; p[2 * v + 1] = a.y; }
        } else {                      // odd row stride: scalar loads are conflict-free
#pragma unroll
          for (int d = 0; d < D; ++d) p[d] = tp[i * D + d];
        }
#pragma unroll
        for (int d = D; d < DP; ++d) p[d] = 0.0f;
        const int row = cb + T * TILE + i;
        if (row < nbeg) continue;  // the first tile starts at the aligned row below nbeg
#pragma unroll
        for (int h = 0; h < QS / 2; ++h) {
          float da, db;
          dist2x2<DYN, UNIT_W>(P.pb, q2[h], p, da, db);
          if (da < best[2 * h]) { best[2 * h] = da; bidx[2 * h] = row; }  // ascending rows per lane, strict <
          if (db < best[2 * h + 1]) { best[2 * h + 1] = db; bidx[2 * h + 1] = row; }
        }
      }
      __syncwarp();  // every lane is done with this stage before lane 0 refills it
    }
#pragma unroll
    for (int j = 0; j < QS; ++j) {
      unsigned long long kv = ((unsigned long long)__float_as_uint(best[j]) << 32) | (unsigned)bidx[j];
      if (bidx[j] == 0x7fffffff) kv = kKeyNone;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) kv = min(kv, __shfl_xor_sync(0xffffffffu, kv, o));
      if (lane == 0 && q0 + j < P.B && kv != kKeyNone) atomicMin(&key[q0 + j], kv);
    }
  }
}

// ---- NN index tier: exact nearest neighbour with spatial pruning ----------
// RRT trees are strongly clustered, so the structure is BALANCED: tree rows [0, n_sorted) are sorted by a Morton
// key over the weighted state box (the host decides how many bits every dimension gets: always the dimension whose
// weighted cell is widest next, DevProblem::idx_*) and cut into tiles of 32 consecutive rows; a tile knows the
// bounding box of its rows over every non-angle dimension, 32 tiles form a super-tile with the box of their union.
// Dense regions get many small boxes, empty space gets none.
//   rebuild  keys -> LSD radix sort (3 passes of 10 bits: per-warp histograms, grid-wide exclusive scan, stable
//            per-warp scatter) -> tiles: rows copied as [tile][dim][32] so that a lane reads its row with
//            coalesced loads -> tile boxes -> super-tile boxes.  Runs when scanning the rows added since the
//            last rebuild would cost about as much as rebuilding (kIdxRebuildWork).
//   search   one warp per query.  A lower bound of the weighted squared distance from the query to a box is
//            sum_d w_d max(0, lo_d - q_d, q_d - hi_d)^2.  Pass A walks the super-tile boxes (one per lane), descends
//            into the nearest one and scores its nearest tile: the exact distance of a real row, an upper bound ub.
//            Pass B walks the super-tile boxes again and opens only boxes whose bound (shrunk by 1e-5 against
//            fp32 rounding) does not exceed ub; every scored tile tightens ub.  A row is skipped only if its box
//            bound is strictly above the final minimum, so the result -- min over (d2 bits, row id) with the same
//            dist2() arithmetic as the scan tiers -- is bit-identical to the brute-force scan, ties included.
// Rows appended since the last rebuild are scanned by the tiled tier; atomicMin merges the two partial results.
constexpr int kIdxDigitBits = 10, kIdxBins = 1 << kIdxDigitBits, kIdxPasses = 3;  // 30-bit keys
constexpr int kIdxChunkMin = 512;    // rows per sorting warp at least (keeps the histogram table <= 2n entries)
constexpr float kIdxShrink = 1.0f - 1e-5f;

struct IdxDims {  // sizes of the index over n rows
  int n_tiles, n_super, n_groups;
};
__host__ __device__ __forceinline__ IdxDims idx_dims(int n) {
  IdxDims d;
  d.n_tiles = (n + 31) / 32;
  d.n_super = (d.n_tiles + 31) / 32;
  d.n_groups = (d.n_super + 31) / 32;
  return d;
}

__device__ __forceinline__ unsigned long long warp_min_key(unsigned long long m) {
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) m = min(m, __shfl_xor_sync(0xffffffffu, m, o));
  return m;
}

// Morton key of a row: per keyed dimension a quantised coordinate, its bits dealt to the key positions the host chose.
template <int DYN>
__device__ __forceinline__ unsigned idx_key(const DevProblem& pb, const float (&x)[DynTraits<DYN>::DP]) {
  unsigned key = 0;
#pragma unroll
  for (int d = 0; d < DynTraits<DYN>::D; ++d) {
    const int nb = pb.idx_bits[d];
    if (nb == 0) continue;
    int q = __float2int_rd((x[d] - pb.lo[d]) * pb.idx_scale[d]);
    q = min(max(q, 0), (1 << nb) - 1);
    for (int b = 0; b < nb; ++b) key |= (unsigned)((q >> b) & 1) << pb.idx_pos[d][b];
  }
  return key;
}

// Grid-wide rebuild over rows [0, n).  sm_hist: kWarps * kIdxBins words (the TMA tile buffers, idle here);
// sm_scan: kThreads + kWarps + 8 words.
template <int DYN>
__device__ __forceinline__ void idx_rebuild(const Params& P, int n, cg::grid_group& grid, unsigned* sm_hist, int* sm_scan) {
  using T = DynTraits<DYN>;
  constexpr int D = T::D, DP = T::DP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int NB = gridDim.x, W = NB * kWarps;
  // sorting warps: warp 0 of every CTA first, then the warps 1, ... (spread over the SMs when few take part)
  const int pj = warp * NB + (int)blockIdx.x;
  int chunk = ((n + W - 1) / W + 31) & ~31;
  if (chunk < kIdxChunkMin) chunk = kIdxChunkMin;
  const int Wp = (n + chunk - 1) / chunk;
  const int cb = min(n, pj * chunk), ce = min(n, cb + chunk);
  unsigned* h = sm_hist + warp * kIdxBins;
  // keys of the chunk (buffer 0): the same lanes read them back below, no barrier needed
  for (int i = cb + lane; i < ce; i += 32) {
    float x[DP];
    const float4* sp = reinterpret_cast<const float4*>(P.states + (size_t)i * DP);
#pragma unroll
    for (int v = 0; v < DP / 4; ++v) {
      const float4 a = __ldcg(sp + v);
      x[4 * v] = a.x; x[4 * v + 1] = a.y; x[4 * v + 2] = a.z; x[4 * v + 3] = a.w;
    }
    P.idx_keys[i] = idx_key<DYN>(P.pb, x);
    P.idx_ids[i] = i;
  }
  const int E = kIdxBins * Wp;                                      // histogram table [bin][sorting warp]
  const int per = (E + NB * kThreads - 1) / (NB * kThreads);        // entries per thread in the scan
  for (int pass = 0; pass < kIdxPasses; ++pass) {
    const unsigned* ksrc = P.idx_keys + (size_t)(pass & 1) * P.cap;
    const int* isrc = P.idx_ids + (size_t)(pass & 1) * P.cap;
    unsigned* kdst = P.idx_keys + (size_t)((pass & 1) ^ 1) * P.cap;
    int* idst = P.idx_ids + (size_t)((pass & 1) ^ 1) * P.cap;
    const int shift = pass * kIdxDigitBits;
    // 1. per-warp digit histogram
    if (pj < Wp) {
      for (int b = lane; b < kIdxBins; b += 32) h[b] = 0;
      __syncwarp();
      for (int i = cb + lane; i < ce; i += 32) atomicAdd(&h[(__ldcg(&ksrc[i]) >> shift) & (kIdxBins - 1)], 1u);
      __syncwarp();
      for (int b = lane; b < kIdxBins; b += 32) P.idx_hist[(size_t)b * Wp + pj] = h[b];
    }
    __threadfence();
    grid.sync();
    // 2. exclusive scan of the table: thread sums -> CTA totals -> (barrier) -> offsets written in place
    const int e0 = min(E, ((int)blockIdx.x * kThreads + (int)threadIdx.x) * per), e1 = min(E, e0 + per);
    unsigned mine = 0;
    for (int e = e0; e < e1; ++e) mine += __ldcg(&P.idx_hist[e]);
    unsigned incl = mine;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const unsigned t = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= o) incl += t;
    }
    __syncthreads();
    if (lane == 31) sm_scan[kThreads + warp] = (int)incl;
    __syncthreads();
    unsigned wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) {
      const unsigned t = (unsigned)sm_scan[kThreads + w];
      if (w < warp) wbase += t;
      total += t;
    }
    if (threadIdx.x == 0) P.idx_ctasum[blockIdx.x] = total;
    __threadfence();
    grid.sync();
    unsigned before = 0;  // sum of the totals of the CTAs before this one
    for (int c = (int)threadIdx.x; c < (int)blockIdx.x; c += kThreads) before += __ldcg(&P.idx_ctasum[c]);
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) before += __shfl_xor_sync(0xffffffffu, before, o);
    __syncthreads();
    if (lane == 0) sm_scan[kThreads + warp] = (int)before;
    __syncthreads();
    unsigned cta_before = 0;
#pragma unroll
    for (int w = 0; w < kWarps; ++w) cta_before += (unsigned)sm_scan[kThreads + w];
    unsigned run = cta_before + wbase + incl - mine;
    for (int e = e0; e < e1; ++e) {
      const unsigned v = __ldcg(&P.idx_hist[e]);
      P.idx_hist[e] = run;
      run += v;
    }
    __threadfence();
    grid.sync();
    // 3. stable scatter: the warp walks its chunk in order, 32 keys at a time
    if (pj < Wp) {
      for (int b = lane; b < kIdxBins; b += 32) h[b] = __ldcg(&P.idx_hist[(size_t)b * Wp + pj]);
      __syncwarp();
      for (int i0 = cb; i0 < ce; i0 += 32) {
        const int i = i0 + lane;
        const bool on = i < ce;
        const unsigned act = __ballot_sync(0xffffffffu, on);
        if (on) {
          const unsigned key = __ldcg(&ksrc[i]);
          const int id = __ldcg(&isrc[i]);
          const unsigned dg = (key >> shift) & (kIdxBins - 1);
          const unsigned m = __match_any_sync(act, dg);
          const unsigned base = h[dg];
          const unsigned pos = base + __popc(m & ((1u << lane) - 1u));
          __syncwarp(act);
          if ((m >> lane) == 1u) h[dg] = base + __popc(m);  // highest lane of the group
          kdst[pos] = key;
          idst[pos] = id;
        }
        __syncwarp();
      }
    }
    __threadfence();
    grid.sync();
  }
  // sorted ids are in buffer (kIdxPasses & 1).  Tiles: rows as [tile][dim][32], ids padded with -1, boxes.
  const int* sorted = P.idx_ids + (size_t)(kIdxPasses & 1) * P.cap;
  const IdxDims G = idx_dims(n);
  const int gw = (int)blockIdx.x * kWarps + warp;
  const float inf = __int_as_float(0x7f800000);
  for (int t = gw; t < G.n_super * 32; t += W) {
    const int pos = t * 32 + lane;
    const int id = pos < n ? __ldcg(&sorted[pos]) : -1;
    float x[DP];
    const float4* sp = reinterpret_cast<const float4*>(P.states + (size_t)max(id, 0) * DP);
#pragma unroll
    for (int v = 0; v < DP / 4; ++v) {
      const float4 a = __ldcg(sp + v);
      x[4 * v] = a.x; x[4 * v + 1] = a.y; x[4 * v + 2] = a.z; x[4 * v + 3] = a.w;
    }
    P.idx_tile_ids[pos] = id;
    float mylo = inf, myhi = -inf;
#pragma unroll
    for (int d = 0; d < D; ++d) {
      P.idx_rows[((size_t)t * D + d) * 32 + lane] = id >= 0 ? x[d] : 0.0f;
      float lo = id >= 0 ? x[d] : inf, hi = id >= 0 ? x[d] : -inf;
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
      }
      if (lane == d) { mylo = lo; myhi = hi; }
    }
    if (lane < D) {
      const size_t at = ((size_t)(t >> 5) * D + lane) * 32 + (t & 31);
      P.idx_tlo[at] = mylo;
      P.idx_thi[at] = myhi;
    }
  }
  __threadfence();
  grid.sync();
  for (int s = gw; s < G.n_groups * 32; s += W) {
    float mylo = inf, myhi = -inf;
#pragma unroll
    for (int d = 0; d < D; ++d) {
      float lo = inf, hi = -inf;
      if (s < G.n_super) {
        lo = __ldcg(&P.idx_tlo[((size_t)s * D + d) * 32 + lane]);
        hi = __ldcg(&P.idx_thi[((size_t)s * D + d) * 32 + lane]);
      }
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) {
        lo = fminf(lo, __shfl_xor_sync(0xffffffffu, lo, o));
        hi = fmaxf(hi, __shfl_xor_sync(0xffffffffu, hi, o));
      }
      if (lane == d) { mylo = lo; myhi = hi; }
    }
    if (lane < D) {
      const size_t at = ((size_t)(s >> 5) * D + lane) * 32 + (s & 31);
      P.idx_slo[at] = mylo;
      P.idx_shi[at] = myhi;
    }
  }
  __threadfence();
  __syncthreads();
  fence_proxy_async();  // the histogram words live in the TMA tile buffers: order them before the next bulk copy
  grid.sync();
}

// lower bound of the weighted squared distance from q to box `j` of a [group][dim][32] box table (lane-private j)
template <int DYN>
__device__ __forceinline__ float idx_box_bound(const DevProblem& pb, const float* __restrict__ lo,
                                               const float* __restrict__ hi, size_t group, int j,
                                               const float (&q)[DynTraits<DYN>::D]) {
  constexpr int D = DynTraits<DYN>::D;
  float acc = 0.0f;
#pragma unroll
  for (int d = 0; d < D; ++d) {
    if (is_angle<DYN>(d)) continue;  // wrapped dims take no part in the bound (they add >= 0)
    const float l = __ldcg(&lo[(group * D + d) * 32 + j]), h = __ldcg(&hi[(group * D + d) * 32 + j]);
    const float e = fmaxf(fmaxf(l - q[d], q[d] - h), 0.0f);
    acc = fmaf(e * pb.w[d], e, acc);
  }
  return acc * kIdxShrink;
}

// Scores the first `cnt` (1..NT, warp-uniform) of the tiles t[] (32 rows each, one per lane) against q and returns the
// tightened upper bound.  The distance is accumulated dimension by dimension over all NT tiles at once -- NT
// independent coalesced loads per dimension, so a warp keeps NT..2NT cache lines in flight instead of one tile's --
// with the operations and the order of dist2(), hence bit-identical keys.  Slots past cnt re-read tile t[0].
template <int DYN, bool UNIT_W, int NT>
__device__ __forceinline__ float idx_score_tiles(const Params& P, const int (&t)[NT], int cnt,
                                                 const float (&q)[DynTraits<DYN>::D], unsigned long long& best, float ub) {
  constexpr int D = DynTraits<DYN>::D;
  const int lane = threadIdx.x & 31;
  int id[NT];
  unsigned off[NT];
  float acc[NT];
#pragma unroll
  for (int a = 0; a < NT; ++a) {
    const int ta = a < cnt ? t[a] : t[0];
    id[a] = __ldcg(&P.idx_tile_ids[(size_t)ta * 32 + lane]);
    off[a] = (unsigned)ta * (D * 32) + lane;  // < 2^32: the host keeps larger trees off the index (set_nn_mode)
    acc[a] = 0.0f;
  }
#pragma unroll
  for (int d = 0; d < D; ++d) {
    float v[NT];
#pragma unroll
    for (int a = 0; a < NT; ++a) v[a] = __ldcg(&P.idx_rows[(size_t)off[a] + d * 32]);
#pragma unroll
    for (int a = 0; a < NT; ++a) {
      const float delta = is_angle<DYN>(d) ? angle_absdiff(q[d], v[a]) : (q[d] - v[a]);
      if (UNIT_W) acc[a] = fmaf(delta, delta, acc[a]);
      else acc[a] = fmaf(delta * P.pb.w[d], delta, acc[a]);
    }
  }
  unsigned bits = 0x7f800000u;
#pragma unroll
  for (int a = 0; a < NT; ++a) {
    if (a < cnt && id[a] >= 0) {
      const unsigned b = __float_as_uint(acc[a]);  // d2 >= 0: uint order == float order
      best = min(best, ((unsigned long long)b << 32) | (unsigned)id[a]);
      bits = min(bits, b);
    }
  }
  return fminf(ub, __uint_as_float(__reduce_min_sync(0xffffffffu, bits)));
}

// Pops the candidate with the smallest bound out of the lane mask `cand` (lane j holds bound `lb`): returns its lane,
// or -1 -- and empties the mask -- once the smallest remaining bound is above ub.
__device__ __forceinline__ int idx_pop_nearest(unsigned& cand, float lb, float ub) {
  const int lane = threadIdx.x & 31;
  const unsigned mine = ((cand >> lane) & 1u) ? __float_as_uint(lb) : 0xffffffffu;  // lb >= 0
  const unsigned mb = __reduce_min_sync(0xffffffffu, mine);
  if (!(__uint_as_float(mb) <= ub)) { cand = 0; return -1; }  // also taken when cand was already empty (mb all ones = NaN)
  const int j = __ffs(__ballot_sync(0xffffffffu, mine == mb)) - 1;
  cand &= ~(1u << j);
  return j;
}

// One warp, one query (all lanes hold the same q): exact NN over the indexed rows [0, n_sorted).
// Super-tile boxes are opened nearest-first, so ub tightens early and most boxes are never opened.  Inside a
// super-tile the nearest tile goes first and the others follow in key order; tiles wait in a small warp-uniform
// queue that is scored NT at a time (across super-tiles), and what is left of a super-tile is re-filtered against
// the tightened ub after every batch.  Scoring a tile the final ub would have excluded costs time, never exactness.
template <int DYN, bool UNIT_W>
__device__ __forceinline__ unsigned long long idx_search(const Params& P, const IdxDims& G,
                                                         const float (&q)[DynTraits<DYN>::D], long long& scored,
                                                         int part, int nparts, const unsigned long long* shared_key) {
  constexpr int NT = 8;  // tiles scored together
  const int lane = threadIdx.x & 31;
  const float inf = __int_as_float(0x7f800000);
  unsigned long long best = kKeyNone;
  float ub = inf;
  int s_near = -1, t_near = -1;
  bool have_bound = false;
  if (part > 0) {  // a later part: what the earlier parts of this query left in key[s] is a real row's distance already
    const unsigned long long kv = __ldcg(shared_key);
    if (kv != kKeyNone) { ub = __uint_as_float((unsigned)(kv >> 32)); have_bound = true; }
  }
  if (G.n_super > 32 && !have_bound) {
    // pass A (several groups of super-tiles): the globally nearest super-tile box, its nearest tile box, that
    // tile's rows -> the exact distance of a real row
    unsigned long long near = kKeyNone;
    for (int s0 = 0; s0 < G.n_super; s0 += 32) {
      const int s = s0 + lane;
      const float lb = s < G.n_super ? idx_box_bound<DYN>(P.pb, P.idx_slo, P.idx_shi, (size_t)(s0 >> 5), lane, q) : inf;
      near = min(near, ((unsigned long long)__float_as_uint(lb) << 32) | (unsigned)s);
    }
    s_near = (int)(unsigned)(warp_min_key(near) & 0xffffffffu);
    const int t = s_near * 32 + lane;
    const float lb = t < G.n_tiles ? idx_box_bound<DYN>(P.pb, P.idx_tlo, P.idx_thi, (size_t)s_near, lane, q) : inf;
    t_near = (int)(unsigned)(warp_min_key(((unsigned long long)__float_as_uint(lb) << 32) | (unsigned)t) & 0xffffffffu);
    const int one[1] = {t_near};
    unsigned long long near_best = kKeyNone;
    ub = idx_score_tiles<DYN, UNIT_W, 1>(P, one, 1, q, near_best, ub);
    scored += 32;
    if (part == 0) best = near_best;  // every part scores this tile for its bound; part 0 reports it
  }
  int pend[NT];  // warp-uniform queue of tiles waiting to be scored
  int np = 0;
#pragma unroll
  for (int a = 0; a < NT; ++a) pend[a] = 0;
  // pass B: every box that can still hold a row at distance <= ub
  for (int s0 = 0; s0 < G.n_super; s0 += 32) {
    const int s_mine = s0 + lane;
    const float lb = s_mine < G.n_super ? idx_box_bound<DYN>(P.pb, P.idx_slo, P.idx_shi, (size_t)(s0 >> 5), lane, q) : inf;
    // this part's super-tiles: every nparts-th one (spatially spread, so the parts cost about the same)
    unsigned cand = __ballot_sync(0xffffffffu, s_mine < G.n_super && s_mine % nparts == part && lb <= ub);
    for (;;) {
      if (nparts > 1) {  // what the other parts of this query have found so far tightens the bound
        const unsigned long long kv = __ldcg(shared_key);
        if (kv != kKeyNone) ub = fminf(ub, __uint_as_float((unsigned)(kv >> 32)));
      }
      const int j = idx_pop_nearest(cand, lb, ub);
      if (j < 0) break;
      const int s = s0 + j;
      const int t_mine = s * 32 + lane;
      const float lbt = t_mine < G.n_tiles ? idx_box_bound<DYN>(P.pb, P.idx_tlo, P.idx_thi, (size_t)s, lane, q) : inf;
      unsigned tc = __ballot_sync(0xffffffffu, t_mine < G.n_tiles && lbt <= ub);
      if (s == s_near) tc &= ~(1u << (t_near & 31));  // scored in pass A
      bool first = true;
      while (tc) {
        int k;
        if (first) {  // nearest tile of the super-tile first
          k = idx_pop_nearest(tc, lbt, ub);
          first = false;
          if (k < 0) break;
        } else {
          k = __ffs(tc) - 1;
          tc &= tc - 1;
        }
#pragma unroll
        for (int a = 0; a < NT; ++a)
          if (a == np) pend[a] = s * 32 + k;
        if (++np == NT) {
          ub = idx_score_tiles<DYN, UNIT_W, NT>(P, pend, NT, q, best, ub);
          scored += 32 * NT;
          np = 0;
          tc &= __ballot_sync(0xffffffffu, lbt <= ub);  // the rest of this super-tile against the tightened bound
        }
      }
      if (np > 0 && ub == inf) {  // no real row scored yet (small index, no pass A): get a bound before opening more
        ub = idx_score_tiles<DYN, UNIT_W, NT>(P, pend, np, q, best, ub);
        scored += 32 * np;
        np = 0;
      }
    }
  }
  if (np > 0) {
    ub = idx_score_tiles<DYN, UNIT_W, NT>(P, pend, np, q, best, ub);
    scored += 32 * np;
  }
  return warp_min_key(best);
}

// All indexed rows against every query of iteration `it` (Alg. 1 l.6-7).  The warps of the CTAs vb = 0..vbcount-1
// take work off a shared counter (far queries open many more boxes than near ones: static shares would leave most
// warps waiting for the unlucky ones).  A unit is (query, part): the super-tiles of a query are dealt to kIdxParts
// units, handed out part by part, so that one expensive query is four medium units instead of one long tail, and the
// later parts start from the bound the earlier ones left in key[s] -- but only while queries are scarce (fewer than ~8
// per warp): with many queries the balance is there already and the repeated first pass would only cost.
// Each unit draws its query itself.
constexpr int kIdxParts = 4;

template <int DYN, bool UNIT_W>
__device__ __forceinline__ void idx_phase(const Params& P, int n_sorted, uint32_t r, uint32_t it,
                                          unsigned long long* key, int vb, int vbcount, int* counter, long long& scored) {
  constexpr int D = DynTraits<DYN>::D, DP = DynTraits<DYN>::DP;
  if (vb < 0) return;
  const int lane = threadIdx.x & 31;
  const IdxDims G = idx_dims(n_sorted);
  const int want = 8 * vbcount * kWarps / P.B;  // parts that bring the units to ~8 per warp (8 parts measured slower)
  const int nparts = G.n_super < 4 * kIdxParts ? 1 : want >= 4 ? kIdxParts : want >= 2 ? 2 : 1;
  const int units = P.B * nparts;
  for (;;) {
    int u = 0;
    if (lane == 0) u = atomicAdd(counter, 1);
    u = __shfl_sync(0xffffffffu, u, 0);
    if (u >= units) break;
    const int part = u / P.B, s = u - part * P.B;
    float q[D];
    sample_state<D>(P.pb, P.seed, r, it, (uint32_t)s, q);
    if (lane == 0 && part == 0) {
#pragma unroll
      for (int d = 0; d < DP; ++d) {
        if (P.dbg_x_rand) P.dbg_x_rand[(size_t)s * DP + d] = d < D ? q[d] : 0.0f;
      }
    }
    const unsigned long long kv = idx_search<DYN, UNIT_W>(P, G, q, scored, part, nparts, &key[s]);
    if (lane == 0 && kv != kKeyNone) atomicMin(&key[s], kv);
  }
}

}  // namespace pakr
#include "pakr_nn_filter.cuh"
namespace pakr {

// ---- NN scan of tree rows [nbeg, nend) for the queries of iteration `it` (Alg. 1 l.6-7) ----
// CTAs vb = 0..vbcount-1 take part (vb < 0: this CTA sits out; the call is CTA-uniform).  Work units are
// (query group of 128, node range); a CTA takes kWarps consecutive units per round, one per warp.  The
// sampled states of the (at most two) query groups a CTA touches in a round are drawn once by the CTA into
// shared memory (Alg. 1 l.6) instead of once per warp.  Partial minima are merged into key[s] with a 64-bit
// atomicMin, so any split of the rows over warps / phases gives the same result.
template <int DYN, bool UNIT_W, bool STREAM, bool FILTER>
__device__ __forceinline__ void nn_phase(const Params& P, int nbeg, int nend, uint32_t r, uint32_t it,
                                         unsigned long long* key, int vb, int vbcount, float* sm_tile,
                                         uint64_t* sm_bar, float* sm_q, unsigned long long* sm_keys, uint32_t& par0,
                                         uint32_t& par1, cg::grid_group& grid, unsigned& sgen,
                                         bool filter_live, unsigned long long* f_slot, long long& filtered,
                                         unsigned long long& ph_outer, unsigned long long& ph_refine, unsigned long long& tp, uint32_t& parx) {
  constexpr int D = DynTraits<DYN>::D, DP = DynTraits<DYN>::DP;
  constexpr int TILE = TileCfg<DYN>::TILE, TF = TileCfg<DYN>::TILE_FLOATS;
  constexpr int QG = 32 * kQ;  // queries per group
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int n = nend - nbeg;
  if (vb < 0 || n <= 0) return;
  if constexpr (STREAM) {  // few queries (B <= kStreamB, chosen by the host): HBM-bound streaming tier
    // 8 query slots when the rows are short (D <= 8) and there are more than 4 queries, else 4: with few queries the
    // arithmetic per byte stays under the machine balance and the pass is HBM-bound
    if (D <= 8 && P.B > 4) nn_stream<DYN, UNIT_W, 8>(P, nbeg, nend, r, it, key, vb, vbcount, sm_q, sm_tile, sm_bar, par0, par1, parx);
    else nn_stream<DYN, UNIT_W, 4>(P, nbeg, nend, r, it, key, vb, vbcount, sm_q, sm_tile, sm_bar, par0, par1, parx);
    return;
  } else if constexpr (FILTER) {
   if (filter_live && n >= kFilterMinRows && (long long)P.B * n * D >= P.filter_min_work) {
    // long row ranges: tensor-core coarse filter, then exact rescoring of the few candidate chunks (same result)
    const FilterPlan fp = filter_plan<DYN>(P.B, n, vbcount * kWarps);
    nn_filter_scan<DYN>(P, nbeg, nend, r, it, vb, vbcount, fp, sm_tile, sm_bar, reinterpret_cast<__half*>(sm_q),
                        reinterpret_cast<float*>(sm_keys), par0, par1);
    if (vbcount == (int)gridDim.x) {
      __threadfence();
      grid.sync();
    } else {
      ++sgen;
      cta_group_barrier(&P.ctrl->sbar, (unsigned)vbcount * sgen);
    }
    const bool timer = blockIdx.x == (unsigned)(gridDim.x - vbcount) && threadIdx.x == 0;  // first participating CTA
    if (timer && blockIdx.x == 0) { const unsigned long long t = globaltimer_ns(); ph_outer += t - tp; tp = t; }
    nn_filter_refine<DYN, UNIT_W>(P, nbeg, nend, r, it, key, vb, vbcount, fp, f_slot, reinterpret_cast<int*>(sm_tile - (threadIdx.x >> 5) * 2 * kTileBufFloats));
    fence_proxy_async();  // the candidate lists were written into the TMA tile buffers with ordinary stores; the next
                          // bulk copy into them belongs to the async proxy (same reuse as after idx_rebuild)
    if (timer && blockIdx.x == 0) { const unsigned long long t = globaltimer_ns(); ph_refine += t - tp; tp = t; }
    filtered += (long long)P.B * n;
    return;
   }
  }
  const int W = vbcount * kWarps;
  const int G = (P.B + QG - 1) / QG;  // query groups
  int R = W / G;                      // node ranges per group
  if (R < 1) R = 1;
  int len = (n + R - 1) / R;
  if (len < 32) len = 32;
  const int Reff = (n + len - 1) / len;
  const int U = G * Reff;
  for (int ub = vb * kWarps; ub < U; ub += W) {
    const int u = ub + warp;
    const bool has = u < U;
    const int g_lo = ub / Reff, g_hi = min(U - 1, ub + kWarps - 1) / Reff;
    const int g = has ? u / Reff : g_lo, rr = has ? u - g * Reff : 0;  // idle warps still read group g_lo's queries
    const int beg = nbeg + rr * len;
    const int end = min(nend, beg + len);
    const bool shared_q = (g_hi - g_lo) <= 1;  // CTA-uniform
    const float* src = P.states + (size_t)beg * DP;
    if (has && lane == 0) {  // the first tile is on its way while the queries are drawn
      const uint32_t bytes = (uint32_t)min(TILE, end - beg) * DP * 4;
      mbar_expect_tx(&sm_bar[0], bytes);
      tma_load_1d(sm_tile, src, bytes, &sm_bar[0]);
    }
    f32x2 q2[kQ / 2][D];  // queries 2h and 2h+1 of this lane, packed per dimension
    float best[kQ];
    int bidx[kQ];
    if (shared_q) {
      if (ub != vb * kWarps) __syncthreads();  // previous round's readers are done with sm_q
      const int ng = (g_hi - g_lo + 1) * QG;
      for (int t = threadIdx.x; t < ng; t += kThreads) {
        float x[D];
        sample_state<D>(P.pb, P.seed, r, it, (uint32_t)(g_lo * QG + t), x);
#pragma unroll
        for (int d = 0; d < D; ++d) sm_q[d * (2 * QG) + t] = x[d];
      }
      __syncthreads();
    }
#pragma unroll
    for (int h = 0; h < kQ / 2; ++h) {
      float qa[D], qb[D];
      const int sa = g * QG + (2 * h) * 32 + lane, sb = sa + 32;
      if (shared_q) {
#pragma unroll
        for (int d = 0; d < D; ++d) {
          qa[d] = sm_q[d * (2 * QG) + (g - g_lo) * QG + (2 * h) * 32 + lane];
          qb[d] = sm_q[d * (2 * QG) + (g - g_lo) * QG + (2 * h + 1) * 32 + lane];
        }
      } else {
        sample_state<D>(P.pb, P.seed, r, it, (uint32_t)sa, qa);
        sample_state<D>(P.pb, P.seed, r, it, (uint32_t)sb, qb);
      }
#pragma unroll
      for (int d = 0; d < D; ++d) q2[h][d] = pack2(qa[d], qb[d]);
      if (P.dbg_x_rand && has && rr == 0 && nbeg == 0) {
#pragma unroll
        for (int d = 0; d < DP; ++d) {
          if (sa < P.B) P.dbg_x_rand[(size_t)sa * DP + d] = d < D ? qa[d] : 0.0f;
          if (sb < P.B) P.dbg_x_rand[(size_t)sb * DP + d] = d < D ? qb[d] : 0.0f;
        }
      }
    }
#pragma unroll
    for (int j = 0; j < kQ; ++j) {
      best[j] = __int_as_float(0x7f800000);
      bidx[j] = 0x7fffffff;
    }
    if (has) {
    const int ntiles = (end - beg + TILE - 1) / TILE;
    for (int t = 0; t < ntiles; ++t) {
      const int cnt = min(TILE, end - beg - t * TILE);
      if (t + 1 < ntiles && lane == 0) {  // prefetch the next tile into the other buffer
        const int b = (t + 1) & 1;
        const uint32_t bytes = (uint32_t)min(TILE, end - beg - (t + 1) * TILE) * DP * 4;
        mbar_expect_tx(&sm_bar[b], bytes);
        tma_load_1d(sm_tile + b * TF, src + (size_t)(t + 1) * TF, bytes, &sm_bar[b]);
      }
      if (t & 1) { mbar_wait(&sm_bar[1], par1); par1 ^= 1; }
      else { mbar_wait(&sm_bar[0], par0); par0 ^= 1; }
      const float4* tp = reinterpret_cast<const float4*>(sm_tile + (t & 1) * TF);
      const int base = beg + t * TILE;
      scan_rows<DYN, UNIT_W>(P.pb, tp, cnt, base, q2, best, bidx);
      __syncwarp();  // every lane is done with this buffer before lane 0 refills it
    }
    }  // has
    if (shared_q) {
      // CTA-level merge: one global atomicMin per (CTA, query) instead of one per (warp, query)
#pragma unroll
      for (int j = 0; j < kQ; ++j)
        sm_keys[warp * QG + j * 32 + lane] =
            (has && bidx[j] != 0x7fffffff) ? (((unsigned long long)__float_as_uint(best[j]) << 32) | (unsigned)bidx[j]) : kKeyNone;
      __syncthreads();
      const int ngroups = g_hi - g_lo + 1;
      for (int t = threadIdx.x; t < ngroups * QG; t += kThreads) {
        const int gi = g_lo + t / QG, qi = t % QG;
        // warps of this round whose unit belongs to group gi: units [max(ub, gi*Reff), min(ub+kWarps, (gi+1)*Reff, U))
        const int w0 = max(ub, gi * Reff) - ub, w1 = min(min(ub + kWarps, (gi + 1) * Reff), U) - ub;
        unsigned long long m = kKeyNone;
        for (int w = w0; w < w1; ++w) m = min(m, sm_keys[w * QG + qi]);
        const int s = gi * QG + qi;
        if (s < P.B && m != kKeyNone) atomicMin(&key[s], m);  // d2 >= 0: uint order == float order; ties -> lowest node
      }
    } else if (has) {
#pragma unroll
      for (int j = 0; j < kQ; ++j) {
        const int s = g * QG + j * 32 + lane;
        if (s < P.B && bidx[j] != 0x7fffffff) {
          const unsigned long long kv =
              ((unsigned long long)__float_as_uint(best[j]) << 32) | (unsigned)bidx[j];
          atomicMin(&key[s], kv);
        }
      }
    }
  }
}

// ---- propagate: controls, RK4 edge, validity, prune, goal flag, per-warp compaction (Alg. 1 l.8-12) ----
// One lane per child, state in registers for the whole edge.  Warp unit u = children [32u, 32u+32) is taken
// by the warp with index pw == u (mod W) among the W warps that propagate (pw < 0: not one of them).
// Survivors go to the scratch rows of the unit, packed by ballot rank.
template <int DYN, int OBS>
__device__ __forceinline__ void prop_phase(const Params& P, uint32_t r, uint32_t it, float c_best,
                                           const unsigned long long* key, bool root_only, int pw, int W,
                                           const float* sm_obs, const uint32_t* sm_cells,
                                           const uint16_t* sm_list) {
  using T = DynTraits<DYN>;
  constexpr int D = T::D, M = T::M, DP = T::DP, PD = T::PD;
  const DevProblem& pb = P.pb;
  const int lane = threadIdx.x & 31;
  const int BK = P.B * P.K;
  const int U = (BK + 31) / 32;
  if (pw < 0) return;
  for (int u = pw; u < U; u += W) {
    const int c = u * 32 + lane;
    const bool active = c < BK;
    const int s = active ? c / P.K : 0;
    const int k = active ? c - s * P.K : 0;
    int parent = 0;
    if (!root_only) {
      const unsigned long long kv = __ldcg(&key[s]);
      parent = (int)(unsigned)(kv & 0xffffffffu);
      if (active && k == 0) {
        if (P.dbg_nn_idx) P.dbg_nn_idx[s] = parent;
        if (P.dbg_nn_d2) P.dbg_nn_d2[s] = __uint_as_float((unsigned)(kv >> 32));
      }
    }
    float x[D], ctl[M];
    {
      const float4* sp = reinterpret_cast<const float4*>(P.states + (size_t)parent * DP);
      float tmp[DP];
#pragma unroll
      for (int v = 0; v < DP / 4; ++v) {
        const float4 a = __ldcg(sp + v);
        tmp[4 * v] = a.x; tmp[4 * v + 1] = a.y; tmp[4 * v + 2] = a.z; tmp[4 * v + 3] = a.w;
      }
#pragma unroll
      for (int d = 0; d < D; ++d) x[d] = tmp[d];
    }
    const float parent_cost = __ldcg(&P.costs[parent]);
    sample_control<M>(pb, P.seed, r, it, (uint32_t)s, (uint32_t)k, ctl);
    // margins: bm >= 0 / om > 0 mean still valid.  Inactive lanes start dead.
    float bm = active ? __int_as_float(0x7f800000) : -1.0f;
    float om = bm;
    float length = 0.0f;
    // Steps are taken in chunks of kChunk: the integration chain runs ahead and the obstacle tests of the
    // chunk's step-end positions (dependent shared-memory lookups) are issued together.
    constexpr int kChunk = 4;
    for (int j0 = 0; j0 < pb.S; j0 += kChunk) {
      float pos[kChunk][PD];
#pragma unroll
      for (int cj = 0; cj < kChunk; ++cj) {
        if (j0 + cj < pb.S) {
          float px[PD];
#pragma unroll
          for (int a = 0; a < PD; ++a) px[a] = x[a];
          dyn_step<DYN>(pb, x, ctl);
          if (pb.cost_mode == 1) {
            float seg = 0.0f;
#pragma unroll
            for (int a = 0; a < PD; ++a) seg = fmaf(x[a] - px[a], x[a] - px[a], seg);
            length += sqrtf(seg);
          }
          bm = fminf(bm, bounds_margin<DYN>(pb, x));
        }
#pragma unroll
        for (int a = 0; a < PD; ++a) pos[cj][a] = x[a];  // past the last step: a repeat of it (harmless)
      }
      if (pb.grid_on) {
        uint32_t hdr[kChunk];
#pragma unroll
        for (int cj = 0; cj < kChunk; ++cj) hdr[cj] = sm_cells[grid_cell<OBS, PD>(pb, pos[cj])];
#pragma unroll
        for (int cj = 0; cj < kChunk; ++cj) om = fminf(om, cell_margin<OBS, PD>(hdr[cj], sm_list, sm_obs, pos[cj]));
      } else {
#pragma unroll
        for (int cj = 0; cj < kChunk; ++cj) om = fminf(om, obstacle_margin<OBS, PD>(sm_obs, pb.n_obs, pos[cj], 0, 1));
      }
      if (P.early_exit && __all_sync(0xffffffffu, !(bm >= 0.0f) || !(om > 0.0f))) break;  // whole warp dead
    }
    bool finite = true;
#pragma unroll
    for (int d = 0; d < D; ++d) finite = finite & (fabsf(x[d]) <= 3.4e38f);
    const bool inb = (bm >= 0.0f) & finite;  // closed box (P12); a non-finite state is out of bounds
    const bool cf = om > 0.0f;               // closed obstacles (P11)
#pragma unroll
    for (int d = 0; d < D; ++d)
      if (is_angle<DYN>(d)) x[d] = wrap_pi(x[d]);
    const float edge = (pb.cost_mode == 1) ? length : (float)pb.S * pb.dt;
    const float c_new = parent_cost + edge;
    const float gd = goal_dist<DYN>(pb, x);
    const float h = fmaxf(0.0f, gd - pb.goal_r) * pb.inv_hspeed;
    const bool notpruned = (c_new + h) < c_best;
    bool ing = gd <= pb.goal_r;
#pragma unroll
    for (int d = 0; d < D; ++d)  // optional heading tolerance on one of the angle dims
      if (is_angle<DYN>(d) && d == pb.goal_angle_dim) ing = ing && (fabsf(wrap_pi(x[d] - pb.goal_angle)) <= pb.goal_angle_tol);
    const bool valid = inb && cf;
    const bool keep = valid && notpruned;
    const int flags = (valid ? 1 : 0) | (inb ? 2 : 0) | (cf ? 4 : 0) | (notpruned ? 8 : 0) | ((keep && ing) ? 16 : 0);
    const unsigned bal = __ballot_sync(0xffffffffu, keep);
    const int rank = __popc(bal & ((1u << lane) - 1u));
    if (lane == 0) P.unit_count[u] = __popc(bal);
    float4 cv;
    {
      float t4[4] = {0.f, 0.f, 0.f, 0.f};
#pragma unroll
      for (int j = 0; j < M; ++j) t4[j] = ctl[j];
      cv = make_float4(t4[0], t4[1], t4[2], t4[3]);
    }
    float xs[DP];
#pragma unroll
    for (int d = 0; d < DP; ++d) xs[d] = d < D ? x[d] : 0.0f;
    if (keep) {
      const size_t slot = (size_t)u * 32 + rank;
      float4* dst = reinterpret_cast<float4*>(P.scr_state + slot * DP);
#pragma unroll
      for (int v = 0; v < DP / 4; ++v) __stcg(dst + v, make_float4(xs[4 * v], xs[4 * v + 1], xs[4 * v + 2], xs[4 * v + 3]));
      __stcg(reinterpret_cast<float4*>(P.scr_ctrl) + slot, cv);
      __stcg(&P.scr_cost[slot], c_new);
      __stcg(&P.scr_parent[slot], parent);
      __stcg(&P.scr_flags[slot], flags | (lane << 8));
    }
    if (active && P.dbg_child_flags) {
      P.dbg_child_flags[c] = flags;
      if (P.dbg_child_cost) P.dbg_child_cost[c] = c_new;
      if (P.dbg_child_ctrl) reinterpret_cast<float4*>(P.dbg_child_ctrl)[c] = cv;
      if (P.dbg_child_state) {
#pragma unroll
        for (int d = 0; d < DP; ++d) P.dbg_child_state[(size_t)c * DP + d] = xs[d];
      }
    }
  }
}

// ---- phase C: ordered insert at the tree tail, goal winner (Alg. 1 l.13-15; P19, P20) ----
// Returns the number of survivors of this iteration (identical in every thread of the grid).
//
// Fused tail scan: when the survivors are few, the NN of the NEXT iteration is completed here as well, straight
// from the scratch rows (their node ids n + rank are known from the prefix), so that no separate scan phase and
// barrier is needed before the next propagate.  `fused` tells the caller (grid-uniform).
constexpr int kFuseUnits = 2048;  // per-unit prefix kept in shared memory up to this many warp units
constexpr int kXTailRows = 1024;  // larger batches of new rows get a scan phase of their own on all CTAs

// One tail-scan item: the survivors of warp units [rg*RU, rg*RU+RU) (gathered by TMA into one tile buffer, in
// node order) against the 128 queries of group g held in q2.
template <int DYN, bool UNIT_W>
__device__ __forceinline__ void tail_item(const Params& P, int n, int g, int rg, int U, const int* sm_upre,
                                          unsigned long long* key_next,
                                          const f32x2 (&q2)[kQ / 2][DynTraits<DYN>::D], float* sm_tile,
                                          uint64_t* sm_bar, uint32_t& par0) {
  constexpr int DP = DynTraits<DYN>::DP, QG = 32 * kQ;
  constexpr int RU = TileCfg<DYN>::TILE / 32;  // units per item: their survivors always fit one tile buffer
  const int lane = threadIdx.x & 31;
  const int ua = rg * RU, ub = min(U, ua + RU);
  const int rows = sm_upre[ub] - sm_upre[ua];
  if (rows == 0) return;
  if (lane == 0) mbar_expect_tx(&sm_bar[0], (uint32_t)rows * DP * 4);
  __syncwarp();
  if (lane < ub - ua) {
    const int u = ua + lane;
    const int cnt = sm_upre[u + 1] - sm_upre[u];
    if (cnt > 0)
      tma_load_1d(sm_tile + (size_t)(sm_upre[u] - sm_upre[ua]) * DP, P.scr_state + (size_t)u * 32 * DP,
                  (uint32_t)cnt * DP * 4, &sm_bar[0]);
  }
  float best[kQ];
  int bidx[kQ];
#pragma unroll
  for (int j = 0; j < kQ; ++j) { best[j] = __int_as_float(0x7f800000); bidx[j] = 0x7fffffff; }
  mbar_wait(&sm_bar[0], par0);
  par0 ^= 1;
  scan_rows<DYN, UNIT_W>(P.pb, reinterpret_cast<const float4*>(sm_tile), rows, n + sm_upre[ua], q2, best, bidx);
#pragma unroll
  for (int j = 0; j < kQ; ++j) {
    const int s = g * QG + j * 32 + lane;
    if (s < P.B && bidx[j] != 0x7fffffff)
      atomicMin(&key_next[s], ((unsigned long long)__float_as_uint(best[j]) << 32) | (unsigned)bidx[j]);
  }
  __syncwarp();  // every lane is done with the tile before it is refilled
}

// Only the propagate CTAs take part (insert inside phase X): CTA-sized chunks of items that share one query
// group; the CTA draws that group's 128 sampled states of iteration it_next itself (Alg. 1 l.6) into sm_qt.
template <int DYN, bool UNIT_W>
__device__ __forceinline__ void tail_scan_rounds(const Params& P, int n, int U, const int* sm_upre,
                                                 unsigned long long* key_next, uint32_t r, uint32_t it_next, int pcta,
                                                 int npcta, float* sm_qt, float* sm_tile, uint64_t* sm_bar,
                                                 uint32_t& par0) {
  using T = DynTraits<DYN>;
  constexpr int D = T::D, QG = 32 * kQ;
  constexpr int RU = TileCfg<DYN>::TILE / 32;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int G = (P.B + QG - 1) / QG;
  const int NR = (U + RU - 1) / RU;
  const int NRp = (NR + kWarps - 1) / kWarps * kWarps;  // items per group, padded to whole CTA chunks
  const int chunks = G * (NRp / kWarps);
  for (int ch = pcta; ch < chunks; ch += npcta) {  // CTA-uniform trip count
    const int g = ch / (NRp / kWarps);
    const int rg = (ch - g * (NRp / kWarps)) * kWarps + warp;
    __syncthreads();  // the previous chunk's readers are done with sm_qt
    for (int t = threadIdx.x; t < QG; t += kThreads) {
      float x[D];
      sample_state<D>(P.pb, P.seed, r, it_next, (uint32_t)min(g * QG + t, P.B - 1), x);
#pragma unroll
      for (int d = 0; d < D; ++d) sm_qt[d * QG + t] = x[d];
    }
    __syncthreads();
    if (rg < NR) {
      f32x2 q2[kQ / 2][D];
#pragma unroll
      for (int h = 0; h < kQ / 2; ++h) {
#pragma unroll
        for (int d = 0; d < D; ++d)
          q2[h][d] = pack2(sm_qt[d * QG + (2 * h) * 32 + lane], sm_qt[d * QG + (2 * h + 1) * 32 + lane]);
      }
      tail_item<DYN, UNIT_W>(P, n, g, rg, U, sm_upre, key_next, q2, sm_tile, sm_bar, par0);
    }
  }
}

// The first `npcta` CTAs take part (all of them when the insert is a phase of its own; only the propagate CTAs
// when it runs inside phase X).  tail_mode: 0 none, 2 CTA rounds (r, it_next) when the insert runs inside phase X.
template <int DYN, bool FILTER, bool STREAM>
__device__ __forceinline__ int insert_phase(const Params& P, int n, int gslot, unsigned long long* key_done,
                                            int tail_mode, unsigned long long* key_next, uint32_t r, uint32_t it_next,
                                            int npcta, int* sm_pref, int* sm_upre, float* sm_qt, float* sm_tile,
                                            uint64_t* sm_bar, uint32_t& par0, bool& fused) {
  using T = DynTraits<DYN>;
  constexpr int DP = T::DP;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int W = npcta * kWarps;
  const int gw = blockIdx.x * kWarps + warp;
  const int BK = P.B * P.K;
  constexpr int cpw = 32;
  const int U = (BK + cpw - 1) / cpw;  // warp units of the propagate phase (32 children each)
  const bool small = U <= kFuseUnits;  // per-unit prefix in shared memory, else per thread-chunk
  constexpr int UPT = kFuseUnits / kThreads;
  const int cpt = small ? UPT : (U + kThreads - 1) / kThreads;  // units per thread-chunk
  int mine = 0;
  int c[UPT];
  if (small) {
#pragma unroll
    for (int k = 0; k < UPT; ++k) {
      const int v = threadIdx.x * UPT + k;
      c[k] = v < U ? (int)__ldcg(&P.unit_count[v]) : 0;
    }
#pragma unroll
    for (int k = 0; k < UPT; ++k) mine += c[k];
  } else {
    for (int v = threadIdx.x * cpt; v < min(U, (threadIdx.x + 1) * cpt); ++v) mine += (int)__ldcg(&P.unit_count[v]);
  }
  int incl = mine;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) {
    const int t = __shfl_up_sync(0xffffffffu, incl, o);
    if (lane >= o) incl += t;
  }
  __syncthreads();  // shared-memory reuse across iterations
  if (lane == 31) sm_pref[kThreads + warp] = incl;
  __syncthreads();
  int wbase = 0, total = 0;
#pragma unroll
  for (int w = 0; w < kWarps; ++w) {
    const int t = sm_pref[kThreads + w];
    if (w < warp) wbase += t;
    total += t;
  }
  sm_pref[threadIdx.x] = wbase + incl - mine;
  if (small) {
    int run = wbase + incl - mine;
#pragma unroll
    for (int k = 0; k < UPT; ++k) {
      sm_upre[threadIdx.x * UPT + k] = run;
      run += c[k];
    }
    if (threadIdx.x == kThreads - 1) sm_upre[kFuseUnits] = run;  // == total
  }
  __syncthreads();
  const int room = P.cap - n;
  for (int u = gw; u < U; u += W) {
    int off, cnt;
    if (small) {
      off = sm_upre[u];
      cnt = sm_upre[u + 1] - off;
    } else {
      const int ch = u / cpt;
      int part = 0;
      for (int v = ch * cpt + lane; v < u; v += 32) part += (int)__ldcg(&P.unit_count[v]);
#pragma unroll
      for (int o = 16; o > 0; o >>= 1) part += __shfl_xor_sync(0xffffffffu, part, o);
      off = sm_pref[ch] + part;
      cnt = (int)__ldcg(&P.unit_count[u]);
    }
    const int pos = off + lane;
    if (lane < cnt && pos < room) {
      const size_t slot = (size_t)u * cpw + lane;
      const int node = n + pos;
      const float4* src = reinterpret_cast<const float4*>(P.scr_state + slot * DP);
      float4* dst = reinterpret_cast<float4*>(P.states + (size_t)node * DP);
      float xr[DP];
#pragma unroll
      for (int v = 0; v < DP / 4; ++v) {
        const float4 a = __ldcg(src + v);
        dst[v] = a;
        xr[4 * v] = a.x; xr[4 * v + 1] = a.y; xr[4 * v + 2] = a.z; xr[4 * v + 3] = a.w;
      }
      if constexpr (STREAM) {
#pragma unroll
        for (int d = 0; d < T::D; ++d) P.prow[(size_t)node * T::D + d] = xr[d];
      }
      if constexpr (FILTER) {
        float xd[T::D];
#pragma unroll
        for (int d = 0; d < T::D; ++d) xd[d] = xr[d];
        filter_write_row<DYN>(P.pb, P.frow, (size_t)node, xd);
      }
      reinterpret_cast<float4*>(P.actions)[node] = __ldcg(reinterpret_cast<const float4*>(P.scr_ctrl) + slot);
      const float cost = __ldcg(&P.scr_cost[slot]);
      P.costs[node] = cost;
      P.parents[node] = __ldcg(&P.scr_parent[slot]);
      const int fl = __ldcg(&P.scr_flags[slot]);
      if (fl & 16)  // goal child: min cost, ties -> lowest node id == lowest child index
        atomicMin(&P.ctrl->goal_key[gslot], ((unsigned long long)__float_as_uint(cost) << 32) | (unsigned)node);
      if (P.dbg_child_flags) P.dbg_child_flags[u * cpw + (fl >> 8)] |= 32;
    }
  }
  if constexpr (FILTER) if (blockIdx.x == 0 && threadIdx.x < 8) {  // filter rows up to the next multiple of 8: far away
    const int n_new = n + min(total, room), row = n_new + (int)threadIdx.x;
    if (row < ((n_new + 7) & ~7)) filter_write_sentinel<DYN>(P.frow, (size_t)row);
  }
  // fused tail scan of the next iteration's NN (every survivor inserted)
  {
    fused = tail_mode == 2 && small && total <= room && total <= kXTailRows;
    if (fused && total > 0) {
      if (P.pb.unit_weights) tail_scan_rounds<DYN, true>(P, n, U, sm_upre, key_next, r, it_next, (int)blockIdx.x, npcta, sm_qt, sm_tile, sm_bar, par0);
      else tail_scan_rounds<DYN, false>(P, n, U, sm_upre, key_next, r, it_next, (int)blockIdx.x, npcta, sm_qt, sm_tile, sm_bar, par0);
    }
  }
  // the NN keys this iteration consumed are free again: reset them for iteration i+2
  for (int s = blockIdx.x * kThreads + threadIdx.x; s < P.B; s += npcta * kThreads) key_done[s] = kKeyNone;
  return total;
}

// Alg. 1 l.16 ExtractPath: warp 0 of block 0 walks parents, then copies in parallel.
// A path of more than kPathMax nodes is not extracted: the buffers keep the last path that fit (with its cost).
template <int DYN>
__device__ __forceinline__ void extract_path(const Params& P, int goal_node, float cost) {
  using T = DynTraits<DYN>;
  const int lane = threadIdx.x & 31;
  int len = 0;
  if (lane == 0) {
    for (int i = goal_node; i >= 0; i = __ldcg(&P.parents[i])) ++len;
    if (len <= kPathMax) {
      int at = kPathMax;
      for (int i = goal_node; i >= 0; i = __ldcg(&P.parents[i])) P.path_nodes_rev[--at] = i;
      P.ctrl->path_len = len;
      P.ctrl->path_cost = cost;
    } else {
      P.ctrl->path_overflow = len;
    }
  }
  len = __shfl_sync(0xffffffffu, len, 0);
  if (len > kPathMax) return;
  __syncwarp();
  for (int i = lane; i < len; i += 32) {
    const int node = P.path_nodes_rev[kPathMax - len + i];
    P.path_nodes[i] = node;
    for (int d = 0; d < T::D; ++d) P.path_states[(size_t)i * T::D + d] = __ldcg(&P.states[(size_t)node * T::DP + d]);
    if (i > 0)
      for (int j = 0; j < T::M; ++j) P.path_controls[(size_t)(i - 1) * T::M + j] = __ldcg(&P.actions[(size_t)node * 4 + j]);
  }
}

// TIER: 0 tiled NN scan, 1 streaming NN scan (B <= kStreamB), 2 tiled scan + NN index, 3 tiled scan + tensor-core filter
template <int DYN, int OBS, int TIER>
__global__ void __launch_bounds__(kThreads, kCtasPerSm) pakr_loop_kernel(const __grid_constant__ Params P) {
  constexpr bool STREAM = TIER == 1, INDEX = TIER == 2, FILTER = TIER == 3;
  using T = DynTraits<DYN>;
  constexpr int OS = (OBS == OBS_CIRCLE) ? 4 : 8;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // [tiles: kWarps * 2 * kTileBufFloats][bars: kWarps * 4][pref: kThreads + kWarps + 8][queries: kMaxD * 256]
  // [merge keys: kWarps * 128 x u64]
  // [obstacles][grid cells][grid lists]
  float* sm_tiles = reinterpret_cast<float*>(smem_raw);
  uint64_t* sm_bars = reinterpret_cast<uint64_t*>(sm_tiles + kWarps * 2 * kTileBufFloats);
  int* sm_pref = reinterpret_cast<int*>(sm_bars + kWarps * 4);
  float* sm_q = reinterpret_cast<float*>(sm_pref + kThreads + kWarps + 8);
  unsigned long long* sm_keys = reinterpret_cast<unsigned long long*>(sm_q + kMaxD * 2 * 32 * kQ);
  float* sm_obs = reinterpret_cast<float*>(sm_keys + kWarps * 32 * kQ);
  uint32_t* sm_cells = reinterpret_cast<uint32_t*>(sm_obs + ((P.pb.n_obs * OS + 3) & ~3));
  uint16_t* sm_list = reinterpret_cast<uint16_t*>(sm_cells + P.pb.g_cells);
  cg::grid_group grid = cg::this_grid();
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  const bool leader = (blockIdx.x == 0 && threadIdx.x == 0);

  for (int i = threadIdx.x; i < P.pb.n_obs * OS; i += kThreads) sm_obs[i] = P.pb.obstacles[i];
  if (P.pb.grid_on) {
    for (int i = threadIdx.x; i < P.pb.g_cells; i += kThreads) sm_cells[i] = P.pb.grid_cells[i];
    for (int i = threadIdx.x; i < P.pb.g_list; i += kThreads) sm_list[i] = P.pb.grid_list[i];
  }
  if (lane == 0) {
#pragma unroll
    for (int b = 0; b < 4; ++b) mbar_init(&sm_bars[warp * 4 + b], 1);  // [2], [3]: the streaming tier's extra stages
  }
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  fence_proxy_async();
  __syncthreads();
  float* my_tile = sm_tiles + warp * 2 * kTileBufFloats;
  uint64_t* my_bar = sm_bars + warp * 4;
  uint32_t par0 = 0, par1 = 0, parx = 0;

  // Roles in phase X.  When the children fill at most a quarter of the SMs, the first NPB CTAs only
  // propagate (latency-bound dependent chains, kept away from the issue-bound scan warps) and the other
  // CTAs run the look-ahead NN scan meanwhile; otherwise every warp does both, one after the other.
  const int NB = gridDim.x;
  const int W = NB * kWarps;
  const int gw = blockIdx.x * kWarps + warp;
  const int U_prop = (P.B * P.K + 31) / 32;
  const int NPB1 = (U_prop + kWarps - 1) / kWarps;  // propagate CTAs at one warp unit (32 children) per warp
  const bool split = NPB1 * 4 <= NB;
  // insert inside phase X by the propagate CTAs (one grid barrier per iteration) when the children are few
  const bool xins = split && U_prop <= kFuseUnits;
  // Rough per-unit cost of an edge and per-pair cost of the scan (ns / ps, from profiles/r02_phases.jsonl): when the
  // look-ahead scan of an iteration takes much longer than the edges, the propagate warps take 2 or 4 units each and
  // the CTAs that frees join the scan.
  const float unit_ns = 3000.0f + (float)P.pb.S * (P.pb.integrator ? 4.0f : 1.0f) *
                                      ((DYN == DYN_DI2 || DYN == DYN_DI3) ? 150.0f : (DYN == DYN_QUAD || DYN == DYN_QUADB) ? 460.0f : 360.0f);
  const float pair_ps = (P.pb.unit_weights ? 0.08f : 0.11f) * (float)T::D;
  unsigned ptarget = 0, sgen = 0;
  unsigned long long* const key0 = P.nn_key;
  unsigned long long* const key1 = P.nn_key + P.B;

  if constexpr (STREAM) {
    // packed rows of what is already in the tree: the root (pakr_plan) or a caller's whole tree (pakr_expand_step)
    const int n0 = P.n_nodes_io ? __ldcg(P.n_nodes_io) : 1;
    for (int i = blockIdx.x * kThreads + threadIdx.x; i < n0; i += gridDim.x * kThreads) {
#pragma unroll
      for (int d = 0; d < T::D; ++d) P.prow[(size_t)i * T::D + d] = __ldcg(&P.states[(size_t)i * T::DP + d]);
    }
    __threadfence();
    fence_proxy_async();
    grid.sync();
  }
  if constexpr (FILTER) {
    // filter rows of what is already in the tree: the root (pakr_plan) or a caller's whole tree (pakr_expand_step),
    // plus far-away rows up to the next multiple of 8.  A hand-over cost, taken before the clock starts.
    const int n0 = P.n_nodes_io ? __ldcg(P.n_nodes_io) : 1;
    for (int i = blockIdx.x * kThreads + threadIdx.x; i < ((n0 + 7) & ~7); i += gridDim.x * kThreads) {
      if (i < n0) {
        float xd[T::D];
#pragma unroll
        for (int d = 0; d < T::D; ++d) xd[d] = __ldcg(&P.states[(size_t)i * T::DP + d]);
        filter_write_row<DYN>(P.pb, P.frow, (size_t)i, xd);
      } else {
        filter_write_sentinel<DYN>(P.frow, (size_t)i);
      }
    }
    __threadfence();
    fence_proxy_async();
    grid.sync();
  }
  unsigned long long t_start = 0;
  if (leader) { t_start = globaltimer_ns(); P.ctrl->t_start_ns = t_start; }

  float c_best = P.c_best0;
  int n = P.n_nodes_io ? __ldcg(P.n_nodes_io) : 1;
  int solved_any = 0, replans_solved = 0, replans_run = 0, termination = 0;
  long long iterations = 0, inserted = 0, nn_pairs = 0;
  long long nn_scored = 0;       // per warp: pairs the index tier scored (lane 0 reports at the end)
  long long nn_idx_covered = 0;  // uniform: pairs of the NN definition the index answered without a scan
  long long nn_filtered = 0;
  unsigned long long nn_rescored = 0;  // uniform (read back from the per-iteration slots)
  unsigned long long ph0 = 0, ph1 = 0, ph2 = 0, ph3 = 0, tp = t_start;
  bool stop = false;
  int cur = 0;  // key buffer of the current iteration

  for (int r = P.r0; r < P.r0 + P.n_replans && !stop; ++r) {
    if (!P.n_nodes_io) n = 1;  // Alg. 1 l.4: node 0 = (x_init, 0, -1, 0) is written once by the host
    int it = P.it0;
    int iters = 0;
    int goal_node = -1;
    int n_scanned = 0;  // NN(it) already covers tree rows [0, n_scanned)
    int n_sorted = 0;   // rows [0, n_sorted) are in the NN index
    int cov_cur = 0, cov_next = 0;  // rows of NN(it) / NN(it+1) the index answered for
    bool filter_live = FILTER;            // tensor-core NN filter in use (per replan)
    long long filt_ahead = 0;             // pairs it took on for the NEXT iteration's NN (credited when that NN is used)
    for (;;) {
      unsigned long long* const kcur = cur ? key1 : key0;
      unsigned long long* const knext = cur ? key0 : key1;
      // per-iteration control words live in slots that rotate over the whole launch (not per replan); see kSlots
      const int slot = (int)(iterations % kSlots);
      const int slot_next = (slot + 1) % kSlots;
      long long filt_head = 0, filt_x = 0;  // pairs the tensor-core filter took on for NN(it) now / for NN(it+1) (uniform)
      // a fresh tree is the root alone: every query's nearest node is node 0, no scan needed
      const bool root_only = (n == 1) && !P.n_nodes_io;
      // NN index tier: used once B*n is large; rebuilt when scanning the rows added since the last rebuild would
      // cost about as much as rebuilding.  When every warp both propagates and searches (no split of the CTAs) the
      // whole NN of the iteration runs at its head, right after the rebuild, instead of one iteration ahead: the
      // rows of the previous batch are then inside the index and need no brute-force pass of their own.
      bool idx_use = false;
      if constexpr (INDEX) idx_use = P.nn_index == 2 ? n >= 256 : (n >= kIdxMinRows && (long long)P.B * n * T::D >= P.idx_min_work);
      if (!idx_use) n_sorted = 0;
      const bool idx_head = idx_use && !split;
      if constexpr (INDEX) {
        const bool grown = P.nn_index == 2 ? n - n_sorted > 64
                                           : (long long)P.B * (n - n_sorted) * T::D >= P.idx_rebuild_work;
        if (idx_use && (n_sorted == 0 || grown) && (n_scanned == 0 || !idx_head)) {
          idx_rebuild<DYN>(P, n, grid, reinterpret_cast<unsigned*>(sm_tiles), sm_pref);
          n_sorted = n;
          if (leader) { const unsigned long long t = globaltimer_ns(); ph3 += t - tp; tp = t; }
        }
      }
      // phase A': rows appended since the look-ahead scan
      if (!root_only && n_scanned < n) {
        int a_beg = n_scanned;
        if (idx_use && n_sorted > 0 && n_scanned == 0) {  // whole-tree NN (first call on a given tree): index + rest
          int* qc = &P.ctrl->idx_query[0][iterations % kSlots];
          if (P.pb.unit_weights) idx_phase<DYN, true>(P, n_sorted, (uint32_t)r, (uint32_t)it, kcur, (int)blockIdx.x, NB, qc, nn_scored);
          else idx_phase<DYN, false>(P, n_sorted, (uint32_t)r, (uint32_t)it, kcur, (int)blockIdx.x, NB, qc, nn_scored);
          a_beg = n_sorted;
          cov_cur = n_sorted;
        }
        if (P.pb.unit_weights) nn_phase<DYN, true, STREAM, FILTER>(P, a_beg, n, (uint32_t)r, (uint32_t)it, kcur, (int)blockIdx.x, NB, my_tile, my_bar, sm_q, sm_keys, par0, par1, grid, sgen, filter_live, &P.ctrl->f_rescored[slot], filt_head, ph0, ph3, tp, parx);
        else nn_phase<DYN, false, STREAM, FILTER>(P, a_beg, n, (uint32_t)r, (uint32_t)it, kcur, (int)blockIdx.x, NB, my_tile, my_bar, sm_q, sm_keys, par0, par1, grid, sgen, filter_live, &P.ctrl->f_rescored[slot], filt_head, ph0, ph3, tp, parx);
        grid.sync();
      }
      if (leader) { const unsigned long long t = globaltimer_ns(); ph0 += t - tp; tp = t; }
      // phase X: propagate(it) and, meanwhile, NN(it+1) over the frozen snapshot [0, n)
      const bool ahead = (iters + 1 < P.max_iters) && !idx_head;
      // roles of this iteration (uniform: every thread derives them from the same n)
      int upw = 1;  // warp units per propagate warp
      if (split && !FILTER && ahead) {
        const float scan_ns = (float)P.B * (float)n * pair_ps * 1e-3f;
        upw = 4.0f * unit_ns <= 0.8f * scan_ns ? 4 : 2.0f * unit_ns <= 0.8f * scan_ns ? 2 : 1;
      }
      const int NPB = (U_prop + kWarps * upw - 1) / (kWarps * upw);
      const int x_pw = split ? ((int)blockIdx.x < NPB ? gw : -1) : gw;  // propagate warp index, count
      const int x_pcnt = split ? NPB * kWarps : W;
      const int x_vb = split ? (int)blockIdx.x - NPB : (int)blockIdx.x;  // scan CTA index (< 0: none), count
      const int x_vbcnt = split ? NB - NPB : NB;
      ptarget += (unsigned)NPB;
      prop_phase<DYN, OBS>(P, (uint32_t)r, (uint32_t)it, c_best, kcur, root_only, x_pw, x_pcnt, sm_obs, sm_cells, sm_list);
      bool fused = false;
      int total = 0;
      if (xins) {
        // The propagate CTAs finish the iteration among themselves while the scan CTAs are still busy:
        // barrier of their own, ordered insert, tail of NN(it+1) over the new rows.
        if ((int)blockIdx.x < NPB) {
          fence_proxy_async();  // scratch rows written with st.global are gathered by TMA below
          cta_group_barrier(&P.ctrl->pbar, ptarget);  // running count of arrivals: NPB may change between iterations
          fence_proxy_async();
          total = insert_phase<DYN, FILTER, STREAM>(P, n, slot, kcur, ahead ? 2 : 0, knext, (uint32_t)r, (uint32_t)(it + 1), NPB, sm_pref,
                                    reinterpret_cast<int*>(sm_q), reinterpret_cast<float*>(sm_keys), my_tile, my_bar, par0,
                                    fused);
          if (leader) P.ctrl->iter_total[slot] = total;
          __threadfence();
          fence_proxy_async();  // tree rows written with st.global are read next by TMA (async proxy)
        }
      }
      if (ahead) {
        int x_beg = 0;
        if (idx_use && n_sorted > 0) {
          int* qc = &P.ctrl->idx_query[1][slot];
          if (P.pb.unit_weights) idx_phase<DYN, true>(P, n_sorted, (uint32_t)r, (uint32_t)(it + 1), knext, x_vb, x_vbcnt, qc, nn_scored);
          else idx_phase<DYN, false>(P, n_sorted, (uint32_t)r, (uint32_t)(it + 1), knext, x_vb, x_vbcnt, qc, nn_scored);
          x_beg = n_sorted;
          cov_next = n_sorted;
        }
        if (P.pb.unit_weights) nn_phase<DYN, true, STREAM, FILTER>(P, x_beg, n, (uint32_t)r, (uint32_t)(it + 1), knext, x_vb, x_vbcnt, my_tile, my_bar, sm_q, sm_keys, par0, par1, grid, sgen, filter_live, &P.ctrl->f_rescored[slot], filt_x, ph1, ph3, tp, parx);
        else nn_phase<DYN, false, STREAM, FILTER>(P, x_beg, n, (uint32_t)r, (uint32_t)(it + 1), knext, x_vb, x_vbcnt, my_tile, my_bar, sm_q, sm_keys, par0, par1, grid, sgen, filter_live, &P.ctrl->f_rescored[slot], filt_x, ph1, ph3, tp, parx);
      }
      if (leader) {
        P.ctrl->goal_key[slot_next] = kKeyNone;
        P.ctrl->f_rescored[slot_next] = 0ull;
        P.ctrl->idx_query[0][slot_next] = 0;
        P.ctrl->idx_query[1][slot_next] = 0;
        if (xins) P.ctrl->stop[slot] = (P.budget_ns && globaltimer_ns() - t_start >= P.budget_ns) ? 1 : 0;
      }
      fence_proxy_async();  // scratch rows written with st.global may be read by TMA in the insert phase
      grid.sync();
      fence_proxy_async();
      if (leader) { const unsigned long long t = globaltimer_ns(); ph1 += t - tp; tp = t; }
      if (xins) {
        total = __ldcg(&P.ctrl->iter_total[slot]);
        fused = ahead && total <= P.cap - n && total <= kXTailRows;
      } else {
        // phase C: insert as a phase of its own (every CTA takes part)
        total = insert_phase<DYN, FILTER, STREAM>(P, n, slot, kcur, 0, knext, (uint32_t)r, (uint32_t)(it + 1), NB, sm_pref,
                                  reinterpret_cast<int*>(sm_q), reinterpret_cast<float*>(sm_keys), my_tile, my_bar, par0,
                                  fused);
        if (leader) P.ctrl->stop[slot] = (P.budget_ns && globaltimer_ns() - t_start >= P.budget_ns) ? 1 : 0;
        __threadfence();
        fence_proxy_async();  // tree rows written with st.global are read next by TMA (async proxy)
        grid.sync();
        if (leader) { const unsigned long long t = globaltimer_ns(); ph2 += t - tp; tp = t; }
        fence_proxy_async();
      }
      const int added = min(total, P.cap - n);
      nn_pairs += (long long)P.B * n;  // (query, node) pairs of this iteration's NN
      nn_idx_covered += (long long)P.B * cov_cur;
      cov_cur = cov_next;
      cov_next = 0;
      n_scanned = ahead ? (fused ? n + added : n) : 0;  // fused: NN(it+1) already covers the new rows
      n += added;
      inserted += added;
      ++iterations;
      ++iters;
      cur ^= 1;
      nn_filtered += filt_ahead + filt_head;  // what NN(it) got from the filter (its look-ahead ran one iteration ago)
      filt_ahead = filt_x;
      const long long filt_iter = filt_head + filt_x;  // the filter's work inside this iteration
      if (filt_iter > 0) {
        // The filter pays only while its second phase rescans few rows: dense, clustered trees put many rows within the
        // rounding band of the nearest one.  Once it does not, the rest of the replan uses the exact scan (the tree only
        // gets denser).  Every thread reads the same counter after the same barrier: the decision is grid-uniform.
        const unsigned long long rsc = __ldcg(&P.ctrl->f_rescored[slot]);
        nn_rescored += rsc;
        if ((long long)rsc * P.filter_give_up > filt_iter) filter_live = false;
      }
      const unsigned long long gk = __ldcg(&P.ctrl->goal_key[slot]);
      stop = __ldcg(&P.ctrl->stop[slot]) != 0;
      ++it;
      if (gk != kKeyNone) {  // Alg. 1 l.14-17
        c_best = __uint_as_float((unsigned)(gk >> 32));
        goal_node = (int)(unsigned)(gk & 0xffffffffu);
        break;
      }
      if (n >= P.cap || iters >= P.max_iters || stop) break;
    }
    ++replans_run;
    if (goal_node >= 0) {
      ++replans_solved;
      solved_any = 1;
      if (blockIdx.x == 0 && warp == 0) extract_path<DYN>(P, goal_node, c_best);
    }
    if (leader) {
      const unsigned long long now = globaltimer_ns();
      if (goal_node >= 0 && replans_solved == 1) P.ctrl->t_first_ns = now;
      const int ri = r - P.r0;
      if (ri < kStatsMax) {
        P.ctrl->replan_cost[ri] = c_best;
        P.ctrl->replan_nodes[ri] = n;
        P.ctrl->replan_iters[ri] = iters;
        P.ctrl->replan_end_ns[ri] = now;
      }
      if (P.dbg_goal_node) *P.dbg_goal_node = goal_node;
    }
    if (stop) termination = 1;
  }
  if (lane == 0 && nn_scored) atomicAdd(&P.ctrl->nn_scored, (unsigned long long)nn_scored);
  if (leader) {
    Ctrl* c = P.ctrl;
    c->t_end_ns = globaltimer_ns();
    c->iterations = iterations;
    c->inserted = inserted;
    c->nn_pairs = nn_pairs;
    c->nn_idx_covered = nn_idx_covered;
    c->nn_filtered = nn_filtered;
    c->nn_rescored = nn_rescored;
    c->phase_ns[0] = ph0; c->phase_ns[1] = ph1; c->phase_ns[2] = ph2; c->phase_ns[3] = ph3;
    c->n_nodes = n;
    c->solved = solved_any;
    c->best_cost = c_best;
    c->replans_run = replans_run;
    c->replans_solved = replans_solved;
    c->termination = termination;
    if (P.n_nodes_io) *P.n_nodes_io = n;
    if (P.dbg_n_inserted) *P.dbg_n_inserted = (int)inserted;
    if (P.dbg_new_c_best) *P.dbg_new_c_best = c_best;
  }
}

}  // namespace pakr
