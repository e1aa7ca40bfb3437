/*
 * pakr_oracle.h -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, single-threaded fp64 CPU restatement of the PAKR batched tree-expansion
 * iteration (Alg. 1, Sec. IV-A) under the readings P1-P30
 * of SURVEY.md Sec. 8(c) / DESIGN.md "Readings of the paper".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg may
 * load this library.  It shares no code, header, table or helper with the CUDA path under
 * paper_2607_03987_b200/csrc/ and include/pakr.h; the numeric values of the enums below are
 * restated there (they are ABI constants documented in DESIGN.md, not shared code).
 *
 * Parity pins (tests/test_oracle_*.py): Philox against the Random123 known-answer vectors and
 * cuRAND's host generator; NN against hand cases; integrators against closed forms (incl. the
 * sign of w x Iw: axisymmetric precession); PATH_LENGTH edge cost against chord-sum closed forms;
 * collision and state-box closedness against analytic rim cases through orc_propagate's flags;
 * prune strictness at c_new + h == c_best and the GOAL flag of a pruned child; insert order
 * against a Python copy_if; tree invariants; how orc_plan ends a replan (goal, tree full,
 * default iteration cap) and the initial cost bound against hand counts; plan re-propagation.
 * Every pin was mutation-checked.  Whole-method trajectory of the randomised
 * planner: "parity unpinned" by the paper (it prints no worked example) -- see DESIGN.md.
 */
#ifndef PAKR_ORACLE_H
#define PAKR_ORACLE_H
#include <stdint.h>
#ifdef __cplusplus
extern "C" {
#endif

enum { ORC_DYN_DOUBLE_INTEGRATOR = 0, ORC_DYN_UNICYCLE2 = 1, ORC_DYN_QUADROTOR = 2,
       ORC_DYN_DUBINS_AIRPLANE = 3, ORC_DYN_UNICYCLE1 = 4, ORC_DYN_QUADROTOR_BODY = 5, ORC_DYN_ACROBOT = 6 };
enum { ORC_INT_EULER = 0, ORC_INT_RK4 = 1 };
enum { ORC_OBS_CIRCLE2D = 0, ORC_OBS_AABB = 1, ORC_OBS_ZCYLINDER = 2 };
enum { ORC_COST_DURATION = 0, ORC_COST_PATH_LENGTH = 1 };
enum { ORC_DIM_REAL = 0, ORC_DIM_ANGLE = 1 };

/* child flag bits (one iteration, Alg. 1 l.10-14) */
enum {
  ORC_F_VALID = 1,     /* in bounds and collision free at every step-end state */
  ORC_F_INBOUNDS = 2,  /* every step-end state inside the state box                           */
  ORC_F_COLLFREE = 4,  /* every step-end position outside every obstacle                      */
  ORC_F_NOTPRUNED = 8, /* c_new + h(x_new) < c_best  (Alg. 1 l.11)                            */
  ORC_F_GOAL = 16,     /* kept and x_new in X_goal    (Alg. 1 l.14)                            */
  ORC_F_INSERTED = 32  /* appended to the tree        (Alg. 1 l.13)                            */
};

/* Problem statement of PAPER.md:59-69 plus the propagation settings of PAPER.md:144.
 * All arrays are caller-owned, fp64 (fp32 inputs widened by the caller). */
typedef struct {
  int32_t dynamics_id, integrator, state_dim, control_dim, pos_dim;
  const double* dyn_params; int32_t n_dyn_params;    /* quadrotor: m, Ixx, Iyy, Izz, g; acrobot: m1, m2, l1, lc1,
                                                        lc2, I1, I2, g (I about each link's centre of mass) */
  const double* state_lo; const double* state_hi;    /* [D]; +-inf = unbounded          */
  const uint8_t* dim_kind;                           /* [D] ORC_DIM_*                   */
  const double* nn_weight;                           /* [D] >= 0                        */
  const double* control_lo; const double* control_hi;/* [m]                             */
  int32_t obstacle_type; const double* obstacles; int32_t n_obstacles;
  const double* start;                               /* [D]                             */
  const double* goal_center; double goal_radius;     /* ball over the goal dims (below) */
  int32_t goal_angle_dim; double goal_angle, goal_angle_tol; /* -1 = no heading test    */
  double dt; int32_t steps_per_edge;
  int32_t cost_mode; double heuristic_speed;         /* h = max(0,|p-g|-r)/speed        */
  /* X_goal = { x : sqrt(sum_{i} delta_i^2) <= goal_radius }, delta_i = x[goal_dims[i]] - goal_center[i], wrapped to
   * [-pi, pi) when that dim is an angle dim.  goal_n_dims = 0: the first pos_dim dims (goal_center[pos_dim]). */
  int32_t goal_n_dims; const int32_t* goal_dims;     /* [goal_n_dims] state indices     */
} orc_problem;

/* Tree of PAPER.md:140: four buffers + a scalar count.  Node-major (states[i*D+d]). */
typedef struct {
  double* states; double* actions; int32_t* parents; double* costs;
  int64_t capacity; int64_t n;
} orc_tree;

/* ---- Philox4x32-10 sampler (reading P4) ---- */
void orc_philox4x32_10(const uint32_t ctr[4], const uint32_t key[2], uint32_t out[4]);
/* u = (word>>8)*2^-24, then fmaf(u, hi-lo, lo) evaluated in fp32 (single IEEE rounding each) */
float orc_uniform_f32(uint32_t word, float lo, float hi);
/* draw j of the stream (seed; it, r, s, kind, k): word j&3 of block j>>2 */
uint32_t orc_draw_word(uint64_t seed, uint32_t it, uint32_t r, uint32_t s, uint32_t kind,
                       uint32_t k, uint32_t j);
void orc_sample_state(const orc_problem* P, uint64_t seed, uint32_t r, uint32_t it, uint32_t s,
                      double* x /*[D]*/);                         /* Alg. 1 l.6 */
void orc_sample_control(const orc_problem* P, uint64_t seed, uint32_t r, uint32_t it, uint32_t s,
                        uint32_t k, double* u /*[m]*/);           /* Alg. 1 l.8 */

/* ---- geometry / dynamics building blocks ---- */
double orc_wrap_pi(double a);                                      /* -> [-pi, pi)          */
double orc_dist2(const orc_problem* P, const double* a, const double* b);   /* reading P5 */
int64_t orc_nearest(const orc_problem* P, const double* states, int64_t n, const double* q,
                    double* d2_out);                               /* Alg. 1 l.7, P6       */
void orc_f(const orc_problem* P, const double* x, const double* u, double* xdot); /* Eq.(1) */
void orc_step(const orc_problem* P, const double* x, const double* u, double* x_next); /* one dt */
/* signed distance-like margin of a position to the obstacle set: >0 free, <=0 in collision */
double orc_obstacle_margin(const orc_problem* P, const double* x);
double orc_bounds_margin(const orc_problem* P, const double* x);   /* >=0 inside (closed)   */
/* S steps with the control held; returns flags VALID|INBOUNDS|COLLFREE,
 * first_bad_step = 1-based index of the first invalid step-end state or 0,
 * min_margin = min over steps of min(|bounds margin|, |obstacle margin|).  x_new has angle
 * dims wrapped (P13). */
int32_t orc_propagate(const orc_problem* P, const double* x0, const double* u, double* x_new,
                      int32_t* first_bad_step, double* min_margin, double* edge_cost);
/* edge cost (P14): DURATION S*dt; PATH_LENGTH sum_j |p_j - p_{j-1}| over step-end positions
 * (PAPER.md:65).  orc_propagate returns it through edge_cost. */
double orc_heuristic(const orc_problem* P, const double* x);       /* P15                  */
int32_t orc_in_goal(const orc_problem* P, const double* x, double* margin); /* P18         */

/* ---- one iteration of the inner loop (Alg. 1 l.6-17) on a caller-visible tree ---- */
typedef struct {
  double* x_rand;       /* [B][D]   or NULL */
  int32_t* nn_idx;      /* [B]      or NULL */
  double* nn_d2;        /* [B]      or NULL */
  double* child_state;  /* [B*K][D] or NULL */
  double* child_ctrl;   /* [B*K][m] or NULL */
  double* child_cost;   /* [B*K]    or NULL */
  int32_t* child_flags; /* [B*K]    or NULL */
  double* child_margin; /* [B*K] min |margin| to a validity boundary, or NULL */
  double* prune_margin; /* [B*K] |c_new+h-c_best|, or NULL */
  double* goal_margin;  /* [B*K] distance of the goal test to its boundary, or NULL */
  int64_t n_inserted;   /* out */
  int64_t goal_node;    /* out: node id of the winner or -1 */
  double new_c_best;    /* out: c_best after the iteration */
  double phase_ms[3];   /* out: wall time of this trip spent in l.6-7 (sample + nearest neighbour), l.8-12 (controls,
                           propagate, validity, prune, goal test), l.13-15 (insert, goal winner); timing only */
} orc_iter_debug;

void orc_tree_reset(const orc_problem* P, orc_tree* T);            /* Alg. 1 l.4 */
/* returns 1 if a goal child was inserted (replan ends), else 0 */
int32_t orc_expand_iteration(const orc_problem* P, orc_tree* T, uint64_t seed, uint32_t r,
                             uint32_t it, int32_t B, int32_t K, double c_best,
                             orc_iter_debug* dbg);

/* ---- AO-x outer loop (Alg. 1 l.1-3,18) ---- */
typedef struct {
  uint64_t seed; int32_t B, K; int64_t tree_capacity; int32_t n_replans;
  double time_budget_ms;          /* <=0: none */
  int64_t max_iters_per_replan;   /* 0: default max(32, cap/(B*K)) (P21) */
  double initial_cost_bound;      /* c_best of Alg. 1 l.1; <= 0 or inf: +inf (the paper's value) */
} orc_plan_opts;

typedef struct {
  int32_t* path_nodes; double* path_states; double* path_controls;
  int32_t path_capacity, path_len;  /* path_len = number of nodes on the path (L+1) */
  double cost; int32_t outcome;     /* 1 solved, 0 no solution */
  int64_t iterations, children, inserted; int32_t replans_run, replans_solved;
  double first_solution_ms, total_ms;
  double* replan_cost;  /* [n_replans] c_best after each replan (inf if none) or NULL */
  int64_t* replan_nodes;/* [n_replans] tree size at the end of each replan or NULL    */
  int64_t* replan_iters;/* [n_replans] or NULL */
  double phase_ms[3];   /* sums of orc_iter_debug.phase_ms over every iteration of the call */
} orc_plan_result;

int32_t orc_plan(const orc_problem* P, const orc_plan_opts* O, orc_tree* T, orc_plan_result* R);

/* Re-propagate a plan from P->start (north_star "every returned plan is re-propagated by the
 * oracle"): returns 0 if every step-end state is valid and the last state is in X_goal, else a
 * positive code (1 collision/bounds, 2 not in goal, 3 control out of bounds);
 * per_edge = 0: one continuous roll-out from P->start; 1: every edge restarts from the stored
 * path state (the tree invariant state[i] = Propagate(state[parent[i]], action[i]));
 * cost_out = sum of edge costs; max_state_err = max abs difference to the given path_states. */
int32_t orc_validate_plan(const orc_problem* P, const double* path_states,
                          const double* path_controls, int32_t path_len, int32_t per_edge,
                          double* cost_out, double* max_state_err);
#ifdef __cplusplus
}
#endif
#endif
