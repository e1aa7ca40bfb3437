/*
 * pakr.h -- C ABI of the B200-native (sm_100a) PAKR hot path.
 *
 * One thing lives behind this header: the batched tree-expansion iteration of PAKR
 * (Alg. 1 lines 5-17; implementation notes PAPER.md:136-144) run in a
 * device-resident loop inside AO-x cost-bounded replanning (Alg. 1 lines 1-4, 18).
 * Every step (sampling, nearest neighbour, propagation, validity, prune, insert, goal, path
 * extraction, the replan loop) runs in CUDA kernels; there is no CPU fallback.
 *
 * Conventions
 *   - "HOST" / "DEVICE" says where a pointer must point.  The library never frees or keeps a
 *     caller pointer beyond the call, except the planner object it returns.
 *   - All bulk device memory is the caller's workspace (DEVICE, 256-byte aligned, at least
 *     pakr_workspace_bytes()).  The library owns only the small planner object.
 *   - Calls on one planner must not overlap (one stream at a time).  pakr_plan and
 *     pakr_expand_step enqueue on `cuda_stream` (a cudaStream_t passed as void*); pakr_plan
 *     synchronises that stream before filling HOST outputs, pakr_expand_step does not.
 *   - No call throws; every failure is a pakr_status and pakr_last_error() text.
 *   - Notation follows BASELINE.json: B sampled states per iteration, K controls per sampled
 *     state, B*K children per iteration (the paper's "batch B", "B/A samples", "A controls",
 *     PAPER.md:95-106,:142).
 *
 * Device tree layout ("four contiguous buffers" + a scalar count), fp32, node-major:
 *   states [cap][Dp]  Dp = state_dim rounded up to a multiple of 4 (pad lanes are 0)
 *   actions[cap][4]   control that produced node i from parents[i] (pad lanes 0); node 0: zeros
 *   parents[cap]      int32, parents[0] = -1, parents[i] < i
 *   costs  [cap]      cost-to-come
 */
#ifndef PAKR_H
#define PAKR_H
#include <stddef.h>
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

typedef struct pakr_planner pakr_planner; /* opaque, owned by the library */

typedef enum {
  PAKR_OK = 0,
  PAKR_ERR_INVALID_ARG = 1,
  PAKR_ERR_UNSUPPORTED = 2,
  PAKR_ERR_WORKSPACE_TOO_SMALL = 3,
  PAKR_ERR_BUFFER_TOO_SMALL = 4,
  PAKR_ERR_CUDA = 5
} pakr_status;

enum { PAKR_DYN_DOUBLE_INTEGRATOR = 0, PAKR_DYN_UNICYCLE2 = 1, PAKR_DYN_QUADROTOR = 2,
       PAKR_DYN_DUBINS_AIRPLANE = 3, PAKR_DYN_UNICYCLE1 = 4, PAKR_DYN_QUADROTOR_BODY = 5, PAKR_DYN_ACROBOT = 6 };
enum { PAKR_INT_EULER = 0, PAKR_INT_RK4 = 1 };
enum { PAKR_OBS_CIRCLE2D = 0, PAKR_OBS_AABB = 1, PAKR_OBS_ZCYLINDER = 2 };
enum { PAKR_COST_DURATION = 0, PAKR_COST_PATH_LENGTH = 1 };
enum { PAKR_DIM_REAL = 0, PAKR_DIM_ANGLE = 1 };
enum { PAKR_NO_SOLUTION = 0, PAKR_SOLVED = 1 }; /* "no solution" is not an error */
/* nearest-neighbour tier (pakr_plan_opts.nn_mode, pakr_step_args.nn_mode) */
enum { PAKR_NN_AUTO = 0,  /* the library picks: the brute-force fp32 scan below B = 4096 queries, the spatial index (once
                             the tree is large enough to pay for building it) from there up */
       PAKR_NN_SCAN = 1,  /* brute-force fp32 scan tiers only (tiled; streaming when B <= 16) */
       PAKR_NN_INDEX = 2, /* spatial index on every tree of >= 256 nodes (tests).  Not with B <= 16 (see below), not for
                             problems without a finite, positively weighted real dim, and not for capacities whose
                             index rows would pass 2^32 floats (~358 M nodes at state_dim 12): those keep the scan */
       PAKR_NN_FILTER = 3 /* tensor-core coarse filter (fp16 hi/lo mma.sync, fp32 accumulate) on every scan of >= 4096
                             rows that is long enough to pay, exact fp32 rescoring of its candidates; problems whose
                             angle dims weigh more than 0.1 in total keep the fp32 scan */ };
/* B <= 16 queries always run the streaming scan tier, whatever nn_mode says: with so few queries the scan is bound by
 * reading the tree once, which neither the index nor the filter can beat. */

/* child flag bits written by pakr_expand_step (Alg. 1 l.10-14) */
enum {
  PAKR_F_VALID = 1,     /* in bounds and collision free at every step-end state */
  PAKR_F_INBOUNDS = 2,  /* every step-end state inside the state box                           */
  PAKR_F_COLLFREE = 4,  /* every step-end position outside every obstacle                      */
  PAKR_F_NOTPRUNED = 8, /* c_new + h(x_new) < c_best (Alg. 1 l.11)                             */
  PAKR_F_GOAL = 16,     /* kept and x_new in X_goal (Alg. 1 l.14)                              */
  PAKR_F_INSERTED = 32  /* appended to the tree (Alg. 1 l.13)                                  */
};

/* Problem statement (dynamics f, x_init, X_goal, U, cost J) plus the propagation
 * settings of PAPER.md:144 (fixed dt, T steps per edge).  All arrays HOST, copied at create. */
typedef struct {
  int32_t dynamics_id; /* PAKR_DYN_*: double integrator [p, pdot], second-order
                          unicycle [x,y,theta,v,omega], quadrotor [p, v, (phi,theta,
                          psi) ZYX, (p,q,r)] with control (T, tau) (BASELINE.json config 4), Dubins airplane
                          [x,y,z,yaw,pitch,v] with control (yaw rate, pitch rate, acceleration),
                          first-order unicycle [x,y,theta] with control (v, omega), quadcopter with
                          body-frame velocities [p, (phi,theta,psi), (u,v,w) body, (p,q,r)] exactly as PAPER.md:174,
                          Acrobot [theta1, theta2, theta1_dot, theta2_dot] with the elbow torque as control
                          (theta1 from the downward vertical, theta2 relative to link 1) */
  int32_t integrator;  /* PAKR_INT_*: forward Euler or classical RK4 */
  int32_t state_dim, control_dim, pos_dim; /* must match dynamics_id: DI (2*pos_dim, pos_dim,
                          2|3), unicycle2 (5,2,2), both quadrotors (12,4,3), Dubins airplane (6,3,3), unicycle1 (3,2,2),
                          Acrobot (4,1,2: its "position" dims are the two joint angles) */
  const float* dyn_params; int32_t n_dyn_params; /* quadrotors: m, Ixx, Iyy, Izz, g; Acrobot: m1, m2, l1, lc1, lc2, I1,
                          I2, g (link masses, length of link 1, distances joint -> centre of mass, inertias about the
                          centres of mass); else 0 */
  const float* state_lo; const float* state_hi;  /* [D]; +-INF = unbounded; box-tested every step */
  const uint8_t* dim_kind; /* [D] PAKR_DIM_*; angle dims (unicycle theta, quadrotor psi, airplane yaw, both Acrobot
                          joint angles) are wrapped to [-pi,pi) and never bounds-tested; must match the dynamics */
  const float* nn_weight;  /* [D] >= 0, d^2 = sum_d w_d delta_d^2; 0 drops a dim */
  const float* control_lo; const float* control_hi; /* [m] */
  int32_t obstacle_type;   /* PAKR_OBS_*: circle/cylinder rows (cx, cy, r); box rows (lo[pos_dim],
                          hi[pos_dim]).  Closed sets, point robot. */
  const float* obstacles; int32_t n_obstacles;   /* n_obstacles <= 1024; the Acrobot takes none (its position dims are
                          angles: UNSUPPORTED with n_obstacles > 0) */
  const float* start;       /* [D] x_init */
  const float* goal_center; /* [pos_dim], or [goal_n_dims] when goal_dims is given */
  float goal_radius;        /* X_goal = closed ball over the goal dims (default: the position dims) ... */
  int32_t goal_angle_dim; float goal_angle, goal_angle_tol; /* ... and |wrap(x[dim]-angle)| <= tol; -1 = none */
  float dt; int32_t steps_per_edge; /* every edge is exactly steps_per_edge steps of dt */
  int32_t cost_mode;      /* PAKR_COST_DURATION (J = T) or PAKR_COST_PATH_LENGTH */
  float heuristic_speed;  /* h(x) = max(0, |p - goal| - r) / heuristic_speed; +INF => h = 0 */
  /* Goal region over listed state dims (PAPER.md:67 X_goal; the Acrobot's swing-up goal lives in angle space,
   * PAPER.md:209,:212): X_goal = { x : sqrt(sum_i delta_i^2) <= goal_radius }, delta_i = x[goal_dims[i]] -
   * goal_center[i], wrapped to [-pi,pi) on angle dims.  goal_n_dims = 0 / goal_dims = NULL: the first pos_dim dims.
   * The heuristic uses the same distance; it stays admissible only if heuristic_speed bounds the rate of change of that
   * distance (with velocity dims in the ball, pass +INF). */
  int32_t goal_n_dims; const int32_t* goal_dims; /* [goal_n_dims] distinct state indices, HOST */
} pakr_problem;

/* Validates and copies the problem; selects the compiled kernel variant; binds `cuda_device` (the caller's current
 * device is restored before returning, here and in every other call).
 * INVALID_ARG: NULL, dims that do not match the dynamics, lo > hi, NaN, weight < 0, a sampled
 * real dim (weight > 0) with an infinite bound, dt <= 0, steps < 1, goal_dims out of range or repeated.
 * UNSUPPORTED: unknown ids, dim_kind not the dynamics' own, obstacles with the Acrobot.  CUDA: device not usable (no sm_100 device). */
pakr_status pakr_create(const pakr_problem* problem, int cuda_device, pakr_planner** out);
void pakr_destroy(pakr_planner* planner);
/* Text of the last failure on this planner ("" if none); valid until the next call on it.
 * pakr_last_error(NULL) returns the text of the last failed pakr_create in this thread. */
const char* pakr_last_error(const pakr_planner* planner);

/* Bytes of DEVICE workspace pakr_plan / pakr_expand_step need for (B, K, tree_capacity), whichever nn_mode is used later:
 * tree 4*(Dp+6) bytes per node, ~(Dp+7)*4 bytes per child, the control block and path buffers (0.6 MB), plus the buffers
 * of EVERY tier the problem admits: packed rows when B <= 16; else index arrays ~(4 D + 20) bytes per node, filter rows
 * 96 bytes per node and B * 16 KB of chunk minima.  0 if an argument is invalid (B < 1, K < 1, K > 4096, B*K > 2^24,
 * capacity < 2 or > 2^30). */
size_t pakr_workspace_bytes(const pakr_planner* planner, int32_t B, int32_t K, int64_t tree_capacity);
/* The same for a caller that knows the nn_mode it will pass: only that mode's tier buffers are counted (AUTO: the index
 * arrays from B = 4096 up, never the filter's; SCAN: none).  A workspace of this size is accepted by pakr_plan /
 * pakr_expand_step calls with this nn_mode (and by pakr_read_stats, pakr_get_tree_layout: the tree, the control block and
 * the path buffers have the same offsets in every mode).  Always <= pakr_workspace_bytes().  0 on invalid arguments. */
size_t pakr_workspace_bytes_for(const pakr_planner* planner, int32_t B, int32_t K, int64_t tree_capacity, int32_t nn_mode);

/* Where pakr_plan keeps its tree inside the workspace (byte offsets), so a caller can read the
 * tree of the last replan after pakr_plan returns (tests check the tree invariants on it). */
typedef struct {
  size_t states_off, actions_off, parents_off, costs_off; /* layouts as in the header comment */
  int32_t state_stride, action_stride;                    /* Dp, 4 */
} pakr_tree_layout;
pakr_status pakr_get_tree_layout(const pakr_planner* planner, int32_t B, int32_t K,
                                 int64_t tree_capacity, pakr_tree_layout* out);

typedef struct {
  uint64_t seed;          /* Philox key; draws are keyed by (seed, replan, iteration, sample, branch) */
  int32_t B, K;
  int64_t tree_capacity;  /* nodes */
  int32_t n_replans;      /* AO-x restarts (Alg. 1 l.3); 1 = plain parallel RRT; <= 4096 */
  double time_budget_ms;  /* > 0: stop at the first iteration boundary past the budget (device
                             %globaltimer; non-deterministic); <= 0: none (deterministic) */
  int64_t max_iters_per_replan; /* 0 = default max(32, capacity / (B*K)) */
  double initial_cost_bound;    /* c_best before the first replan (Alg. 1 l.1); <= 0 or +INF = none.  A finite bound
                                   (e.g. the best cost another replica found) prunes from the start;
                                   the result reports only what THIS call found (NO_SOLUTION if nothing cheaper) */
  int32_t nn_mode;              /* PAKR_NN_*: which nearest-neighbour tier answers Alg. 1 l.7.  Every tier returns the
                                   same (d^2, lowest index) result bit for bit (PAPER.md:142 tiers have no semantics) */
} pakr_plan_opts;

#define PAKR_MAX_REPLAN_STATS 64
#define PAKR_MAX_PATH_NODES 8192 /* longest path (nodes) the device-side extraction holds */
typedef struct {
  int64_t iterations;      /* inner-loop trips over all replans */
  int64_t children;        /* = iterations * B * K propagated and checked ("expanded nodes") */
  int64_t inserted;        /* nodes appended over all replans */
  int64_t nn_pairs;        /* sum over iterations of B * n: the (query, node) pairs of the NN definition */
  int64_t nn_pairs_evaluated; /* fp32 distances actually evaluated: = nn_pairs under the plain scan tiers; fewer when the
                              NN index answered (it scores only rows whose bounding box can beat the running best) or
                              the tensor-core filter did (only the rows of its candidate ranges are rescored exactly) */
  int64_t nn_pairs_filtered;  /* pairs answered by the tensor-core coarse filter (fp16 hi/lo mma, fp32 accumulate) */
  int64_t h2d_bytes, d2h_bytes; /* bytes pakr_plan copied host->device (root node) and device->host (control
                                   block, path) in this call; kernel parameters (~1.3 KB) not counted */
  int32_t replans_run, replans_solved;
  int32_t termination;     /* 0 all replans run, 1 time budget */
  int32_t replan_stats_truncated; /* 1 if replans_run > PAKR_MAX_REPLAN_STATS: the per-replan arrays hold the first 64 */
  int32_t path_truncated;  /* 1 if a solved replan's path had more than PAKR_MAX_PATH_NODES nodes: it tightened c_best
                              but could not be extracted; pakr_result then holds the last path that fit and ITS cost */
  double first_solution_ms;/* device time from kernel start to the end of the first solved replan; -1 if none */
  double device_ms;        /* device time of the whole loop (%globaltimer) */
  double phase_ms[4];      /* CTA 0's time in: NN phases of their own (whole-tree NN at the head of an iteration, scans
                              of rows added since the look-ahead) / the propagate phase (with the next iteration's NN
                              look-ahead beside it and, when children are few, the insert inside it) / insert phases
                              of their own / rebuilds of the NN index (index tier) or the exact rescoring phase of the
                              tensor-core filter when every CTA takes part in it (filter tier; the filter's first phase
                              is counted with the phase it runs in); each incl. its grid barriers */
  /* first PAKR_MAX_REPLAN_STATS replans: */
  float replan_cost[PAKR_MAX_REPLAN_STATS];   /* c_best after the replan (+INF before any solution) */
  int32_t replan_nodes[PAKR_MAX_REPLAN_STATS];/* tree size at its end */
  int32_t replan_iters[PAKR_MAX_REPLAN_STATS];
  double replan_end_ms[PAKR_MAX_REPLAN_STATS];/* device time at its end */
} pakr_stats;

typedef struct {
  /* caller-allocated HOST buffers; any may be NULL if not wanted */
  int32_t* path_nodes;    /* [path_capacity] node ids root -> goal (ids in the solving replan's tree) */
  float* path_states;     /* [path_capacity][state_dim] */
  float* path_controls;   /* [path_capacity-1][control_dim]; control i is held for steps_per_edge*dt */
  int32_t path_capacity;  /* in  */
  int32_t path_len;       /* out: nodes on the best path (L+1), 0 if none */
  double cost;            /* out: cost of the returned path = c_best (see stats.path_truncated), +INF if none */
  int32_t outcome;        /* out: PAKR_SOLVED / PAKR_NO_SOLUTION */
  int32_t final_tree_nodes; /* out: size of the tree left in the workspace (the last replan's) */
  pakr_stats stats;       /* out */
} pakr_result;

/* Alg. 1 whole: AO-x loop around the batched expansion, one persistent cooperative kernel, no
 * host round trip per iteration.  Returns the best path found (sigma*, Alg. 1 l.18).
 * BUFFER_TOO_SMALL: path longer than path_capacity (path_len = needed length, cost/outcome
 * still set), or no solved replan's path fit PAKR_MAX_PATH_NODES.  WORKSPACE_TOO_SMALL / INVALID_ARG: nothing
 * launched.  The caller's current CUDA device is left as it was. */
pakr_status pakr_plan(pakr_planner* planner, const pakr_plan_opts* opts, void* d_workspace,
                      size_t workspace_bytes, void* cuda_stream, pakr_result* out);

/* One trip of Alg. 1 l.6-17 on caller-visible DEVICE buffers (test hook; same kernels).  The streaming, index and
 * filter tiers first build their own copy of the caller's tree rows inside the workspace (a hand-over pass before the
 * kernel's clock starts).  PAKR_NN_FILTER assumes every row lies inside the state box on the weighted dims (rows the
 * planner inserted always do): its rounding band is derived from the box. */
typedef struct {
  uint64_t seed; uint32_t replan, iteration;
  int32_t B, K; int64_t tree_capacity;
  float c_best;                 /* +INF = no bound yet */
  int32_t nn_mode;              /* PAKR_NN_* */
  /* tree, DEVICE, layouts as in the header comment; in/out */
  float* states; float* actions; int32_t* parents; float* costs;
  int32_t* n_nodes;             /* DEVICE scalar, in/out */
  /* optional DEVICE debug outputs, each may be NULL */
  float* x_rand;                /* [B][Dp] */
  int32_t* nn_idx;              /* [B] */
  float* nn_d2;                 /* [B] */
  float* child_state;           /* [B*K][Dp]; angle dims wrapped */
  float* child_ctrl;            /* [B*K][4] */
  float* child_cost;            /* [B*K] */
  int32_t* child_flags;         /* [B*K] PAKR_F_* */
  int32_t* n_inserted;          /* scalar */
  int32_t* goal_node;           /* scalar, -1 if no goal child was inserted */
  float* new_c_best;            /* scalar */
} pakr_step_args;

pakr_status pakr_expand_step(pakr_planner* planner, const pakr_step_args* args, void* d_workspace,
                             size_t workspace_bytes, void* cuda_stream);

/* pakr_expand_step for callers that have no device memory to hand over as a workspace and are not allowed to get any.
 *
 * Who that is: a planner embedded in a control loop usually reserves all its memory while the robot boots and is
 * forbidden to allocate afterwards -- cudaMalloc / cudaFree may stall the whole device for an unbounded time, which a
 * loop with a deadline cannot accept -- and a plug-in inside a host program whose own pool owns the device memory has
 * nobody to ask for 2 MB more.  Such a caller already holds its tree buffers (inputs and outputs); what it lacks is
 * the scratch one iteration of Alg. 1 l.6-17 needs on top of them: the NN keys of the B queries, the children
 * between propagation and the ordered insert (Alg. 1 l.8-13), the control block and the path buffers.
 *
 * Here that scratch is a fixed array of PAKR_STATIC_SCRATCH_BYTES that is part of the library image itself (a
 * file-scope __device__ array): every GPU that loads libpakr.so carries it from then until the process exits,
 * whether or not this call is ever made.  The call itself performs no cudaMalloc, cudaMallocHost, cudaFree or any other
 * allocating routine, on the first call or later; it enqueues three small memsets of its own scratch and one
 * cooperative kernel launch on `cuda_stream` and returns without synchronising.  `planner` comes from pakr_create,
 * which does allocate a few KB (obstacle tables, a pinned staging block) and therefore belongs to start-up.
 *
 * Same arguments, outputs and bit-for-bit results as pakr_expand_step with nn_mode = PAKR_NN_SCAN, except:
 *   - limit: B * K <= PAKR_STATIC_MAX_CHILDREN.  More is PAKR_ERR_INVALID_ARG ("... exceeds the static scratch ...");
 *     nothing is launched.  tree_capacity is not limited by the scratch (the tree is the caller's), only by 2^30.
 *   - args->nn_mode must be PAKR_NN_AUTO or PAKR_NN_SCAN (else PAKR_ERR_UNSUPPORTED): the NN is always the tiled fp32
 *     scan, also for B <= 16; the streaming, index and filter tiers keep per-node copies that do not fit a fixed array.
 *   - pakr_read_stats has nothing to read afterwards (it looks inside a caller workspace).
 * First call on each device: the library looks up that device's address of the array (cudaGetSymbolAddress, with the
 * planner's device current) and remembers it.  Make one call per device during start-up, before any stream capture
 * begins; later calls skip the look-up.
 * Sharing: there is ONE array per device, used by every planner and every thread of the process.  Two calls whose
 * kernels can run at the same time on one device (different streams, or different host threads) corrupt each other's
 * results: issue them on one stream, or order them with events.  The array keeps whatever the previous call left;
 * the words that must start from a known value (NN keys, control block) are reset on `cuda_stream` by each call. */
#define PAKR_STATIC_MAX_CHILDREN 16384
#define PAKR_STATIC_SCRATCH_BYTES (2304u * 1024u) /* 2.25 MiB per device */
pakr_status pakr_expand_step_static(pakr_planner* planner, const pakr_step_args* args, void* cuda_stream);

/* Statistics of the last pakr_plan / pakr_expand_step launch that used this workspace with the same
 * (B, K, tree_capacity): synchronises `cuda_stream`, then copies the device control block into *out (HOST).
 * After pakr_expand_step: iterations = 1, phase_ms[0] = the NN scan of the whole tree, [1] = propagate (+ insert
 * when the children are few), [2] = insert as a phase of its own, each including its grid barrier. */
pakr_status pakr_read_stats(pakr_planner* planner, int32_t B, int32_t K, int64_t tree_capacity,
                            void* d_workspace, size_t workspace_bytes, void* cuda_stream, pakr_stats* out);

#ifdef __cplusplus
}
#endif
#endif /* PAKR_H */
