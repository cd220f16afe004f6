/*
 * wm.h — C-ABI of the B200-native Waymax closed-loop step (arXiv 2310.08710).
 *
 * One thing is exported: the data-parallel hot path of the simulator — the batched
 * closed-loop environment step over B scenarios x A agents — as hand-written sm_100a CUDA
 * kernels.  Citations are PAPER.md line numbers (+ section / equation); "Dnn" are the
 * readings listed in DESIGN.md where the paper is silent or ambiguous.
 *
 * Conventions
 *  - Every function returns int: WM_OK (0) or a negative wm_status.  Nothing throws, aborts
 *    or prints.  After WM_ERR_CUDA, wm_last_cuda_error() returns the cudaError_t.
 *  - Unless a function says HOST, every data pointer is a DEVICE pointer owned by the
 *    caller; the library owns only what hangs off wm_handle (prepared road-edge segments and
 *    search grids, bucketed roadgraph points, scratch, the instantiated CUDA graph, staging buffers).
 *  - Work is enqueued on the caller's stream (`void* stream` = cudaStream_t; NULL = the
 *    legacy default stream) and NOT synchronised, unless a function says it synchronises.
 *  - Functions are pure in the paper's sense (L120): outputs depend only on the arguments,
 *    repeated calls are bit-identical.
 *  - Arrays are struct-of-arrays, innermost dimension contiguous, 16-byte aligned:
 *      trajectories  [B][T][A]  (time-major rows of A agents; paper state L82, L322)
 *      roadgraph     [B][R]
 *      actions       [B][C][A]  (one step) or [B][n_steps][C][A] (rollout)
 *  - Invalid slots (valid == 0) may hold anything, NaN included; they are never read for
 *    arithmetic that reaches an output (D10).  Outputs for invalid agents are 0 / flag 0 /
 *    index -1.
 *  - Limits: 1 <= A <= 1024, 1 <= B, T >= 1, R >= 1, topk <= R, history <= T.
 */
#ifndef WM_H_
#define WM_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef enum {
  WM_OK = 0,
  WM_ERR_ARG = -1,          /* null / misaligned pointer, bad shape, t out of range */
  WM_ERR_CUDA = -2,         /* a CUDA call failed; see wm_last_cuda_error() */
  WM_ERR_UNSUPPORTED = -3,  /* e.g. A > 1024, B > 65535 scenarios per call, topk > R, more than 131 072 road-edge segments in a scenario */
  WM_ERR_STATE = -4,        /* e.g. metrics_offroad before wm_prepare */
  WM_ERR_TOO_LARGE = -5     /* the problem does not fit the fixed, built-in scratch of a no-allocation entry point
                               (wm_observe_topk_static): use the regular entry point, which allocates what it needs */
} wm_status;

enum { WM_DYN_INVERTIBLE_BICYCLE = 0, WM_DYN_DELTA_LOCAL = 1, WM_DYN_DELTA_GLOBAL = 2 };   /* DELTA_GLOBAL: Eq. 1 literally (world-frame delta) */
enum { WM_TYPE_LANE = 1, WM_TYPE_ROAD_EDGE = 2 };

/* Dynamic state, PAPER.md L82 / L322: s = (x, y, yaw, v_x, v_y) + box dims + validity,
 * per agent and timestep.  Each pointer addresses [B][T][A]. */
typedef struct {
  int32_t B, A, T;
  float *x, *y, *yaw, *vel_x, *vel_y, *length, *width;
  uint8_t* valid;
} wm_traj;

/* Static roadgraph, PAPER.md L82 / L100: oriented points; z ignored (D27). [B][R] each. */
typedef struct {
  int32_t B, R;
  float *x, *y, *dir_x, *dir_y;
  int32_t *type, *id;
  uint8_t* valid;
} wm_roadgraph;

typedef struct {
  int32_t dynamics;     /* WM_DYN_* */
  float dt;             /* 0.1 s (D1) */
  float max_accel;      /* 6.0 m/s^2, L104; <= 0 disables clipping (D7) */
  float max_curvature;  /* 0.3 1/m,  L104; <= 0 disables clipping (D7) */
  int32_t history;      /* 11 steps: the first second of the log (L78) */
  int32_t topk;         /* 1000 nearest roadgraph points per ego (D23) */
  int32_t offroad_mode; /* WM_OFFROAD_*: how wm_metrics_offroad / wm_rollout search the segments */
  int32_t rollout_mode; /* WM_ROLLOUT_*: how wm_rollout runs the n_steps */
  int32_t topk_order;   /* WM_TOPK_*: order of the k selected roadgraph points in wm_observe's outputs */
} wm_config;

/* Both modes find the nearest segment exactly and use the same per-pair arithmetic; they return the
 * same bits whenever they pick the same segment (at a polyline vertex the two neighbours' float32
 * distances can differ by an ulp).
 * CULLED (default): wm_prepare lays nested grids over the segments (2 m cells near the map, 8 m cells in the
 *   wide margin around it); every cell lists, as runs of consecutive segments, the only segments that can
 *   be nearest to a point inside it; a query walks the list of its corner's cell (about 8 segments).  Crowded cells and points outside the grids
 *   fall back to a bounding-box search over all segments, exact as well.
 * BRUTE_FORCE: every corner-segment pair is evaluated (the FP32-roofline reference kernel). */
enum { WM_OFFROAD_CULLED = 0, WM_OFFROAD_BRUTE_FORCE = 1 };

/* Both modes return bit-identical rows (same device arithmetic), both replayed as one CUDA graph (L200).
 * FUSED (default): TWO kernel launches for all n_steps: k_rollout_dyn_bulk (k_rollout_dyn when A is not a multiple
 *   of 16) lays down the whole trajectory with its log divergence and ADE, one CTA per scenario; k_rollout_metrics
 *   then computes overlap and offroad of every row, one CTA per (scenario, block of 8 steps) with those rows in
 *   shared memory; needs WM_OFFROAD_CULLED (with BRUTE_FORCE the stepwise graph is used).
 * STEPWISE: n_steps x {k_step, k_overlap, k_offroad} + k_aggregate, the kernels of the single-step
 *   entry points. */
enum { WM_ROLLOUT_FUSED = 0, WM_ROLLOUT_STEPWISE = 1 };

/* Order of the top-k outputs of wm_observe (the selected SET is the same).  BY_INDEX (default, D24): ascending
 * roadgraph index.  BY_DISTANCE (D44): ascending distance to the ego centre (the float32 selection key),
 * ties -> lower index: "sub-samples the roadgraph via distance" (L82) as a nearest-first list. */
enum { WM_TOPK_BY_INDEX = 0, WM_TOPK_BY_DISTANCE = 1 };

typedef struct wm_handle wm_handle; /* opaque */

/* Per-step metric rows [B][n_steps][A] and aggregates [B][A] of a rollout. Any pointer may be
 * NULL (that output is skipped). ade = sum of valid log divergences / count (D21). */
typedef struct {
  uint8_t *overlap, *offroad;
  float *offroad_dist, *log_div;
  uint8_t *any_overlap, *any_offroad;
  float* ade;
} wm_rollout_out;

/* Create / destroy a handle. `cfg` is copied. HOST pointers. wm_destroy synchronises. */
int wm_create(wm_handle** out, const wm_config* cfg);
int wm_destroy(wm_handle* h);
int wm_last_cuda_error(void);
/* Human-readable build tag, e.g. "wm_b200 sm_100a". HOST. */
const char* wm_version(void);

/*
 * Static precompute at reset time (the roadgraph does not change during an episode, L82):
 *  - road-edge segments for the offroad metric (L100; D14-D17): consecutive entries
 *    (i, i+1) with both valid, both WM_TYPE_ROAD_EDGE and equal id form a segment; an
 *    isolated valid road-edge point is a zero-length segment signed by its stored dir;
 *    and the nested grids of candidate lists over them (WM_OFFROAD_CULLED);
 *  - the valid roadgraph points bucketed into a uniform grid for the top-k observation (L82).
 * Keeps pointers to nothing in `rg` (everything needed is copied); `rg` must match the B of
 * later calls.  SYNCHRONISES the stream (it sizes its buffers from a device-side count).
 * `n_segments_max` (HOST, may be NULL) receives max_b S_e(b).
 */
int wm_prepare(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, void* stream);

/* reset(scenario), L122 / L78: sim rows [0, history) <- log rows; later rows are cleared
 * (valid = 0, fields 0).  *t (HOST, may be NULL) receives history - 1. */
int wm_reset(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t* t, void* stream);

/*
 * step(state, action), L123: writes row t+1 of `sim` from row t.
 *  - WM_DYN_INVERTIBLE_BICYCLE, Appendix A.1 Eq. 2 (L339-L350), action (a, kappa), C = 2;
 *  - WM_DYN_DELTA_LOCAL, Eq. 1 (L324-L333) on the body-frame delta (dx, dy, dyaw) rotated by
 *    yaw_t (D2), C = 3.
 * An agent is moved by the dynamics iff action_valid && sim.valid[t]; every other slot of
 * row t+1 is copied from log row t+1, all 8 fields (log playback, L164; D8).  Controlled
 * agents keep length/width and get valid = 1 (D9).  Actions are clipped to
 * +-max_accel / +-max_curvature (D7).  Yaw is not wrapped (D5), speed is not clamped (D6).
 * action [B][C][A]; action_valid [B][A]. Requires 0 <= t < T-1.
 */
int wm_step(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t, const float* action,
            const uint8_t* action_valid, void* stream);

/*
 * Collision metric, L102: for every pair of valid agents at row t, do the oriented
 * rectangles (centre x,y; length along yaw, width across) intersect with positive area
 * (D12: touching is not overlap; D13: no self pairs).
 * pair_bits [B][A][ceil(A/32)] uint32, bit j%32 of word j/32 of row i = overlap(i, j); may be
 * NULL.  agent_flag [B][A] = OR_j overlap(i, j).
 */
int wm_metrics_overlap(wm_handle* h, const wm_traj* sim, int32_t t, uint32_t* pair_bits,
                       uint8_t* agent_flag, void* stream);

/*
 * Off-road metric, L100: signed distance of each of the 4 box corners of every valid agent
 * at row t to the nearest road-edge segment (prepared by wm_prepare); negative on the left
 * of the oriented edge (on-road), positive on the right (D15-D17, D19).
 * signed_dist [B][A] = max over the 4 corners (D18); corner_dist [B][4][A] (corner order:
 * 0 front-left, 1 front-right, 2 rear-right, 3 rear-left), may be NULL; agent_flag [B][A] =
 * valid && signed_dist > 0.  A scenario without road-edge segments gives -FLT_MAX, flag 0
 * (D20).  Returns WM_ERR_STATE before wm_prepare.
 */
int wm_metrics_offroad(wm_handle* h, const wm_traj* sim, int32_t t, float* signed_dist,
                       float* corner_dist, uint8_t* agent_flag, void* stream);

/* Displacement error, L106: dist [B][A] = ||(x,y)_sim - (x,y)_log||_2 at row t,
 * valid [B][A] = both valid; dist = 0 where not valid. */
int wm_log_divergence(wm_handle* h, const wm_traj* log, const wm_traj* sim, int32_t t,
                      float* dist, uint8_t* valid, void* stream);

/*
 * Default observation, L82: for every ego e (every agent slot; egos invalid at t get zeros /
 * -1) at row t:
 *  - hist [B][A_ego][H][7][A], hist_valid [B][A_ego][H][A]: all agents' last H = history
 *    steps (rows t-H+1 .. t) in the ego frame at t: p' = R(-yaw_e)(p - p_e),
 *    yaw' = wrap(yaw - yaw_e) in [-pi, pi), v' = R(-yaw_e) v, length, width (D22);
 *  - rg_index [B][A_ego][k], rg_feat [B][A_ego][4][k] (x', y', dir_x', dir_y'), rg_type
 *    [B][A_ego][k]: the k = topk valid roadgraph points nearest the ego centre, ties to the
 *    lower index, emitted in ascending index order (or nearest first: wm_config.topk_order), padded
 *    with -1 / 0 (D23-D25).  The
 *    selection key is the float32 value fma(dy, dy, dx*dx), dx = px - ex, dy = py - ey.
 * Either group of outputs may be skipped by passing NULL for all of its pointers.
 * The top-k part needs wm_prepare (WM_ERR_STATE otherwise). Requires t >= history-1.
 */
int wm_observe(wm_handle* h, const wm_traj* sim, const wm_roadgraph* rg, int32_t t, float* hist,
               uint8_t* hist_valid, int32_t* rg_index, float* rg_feat, int32_t* rg_type,
               void* stream);

/*
 * The top-k half of wm_observe (L82: "sub-samples the roadgraph via distance") for callers that are not
 * allowed to allocate device memory at the point where they call the library.  Who that is:
 *  - code running inside a training or serving job whose framework has already handed (nearly) all of the
 *    GPU's memory to its own pooling allocator: a cudaMalloc issued by a library then fails, or eats into
 *    the pool's head-room;
 *  - planners and controllers with a memory budget fixed at start-up, where allocating later is forbidden;
 *  - latency-critical loops: cudaMalloc and cudaFree stall the whole device while they run.
 * The regular route cannot serve them: wm_create and wm_prepare call cudaMalloc (handle counters, the
 * bucketed roadgraph points).  This function needs NO handle and calls no cudaMalloc, cudaFree, stream- or
 * event-creating routine, nor anything else that allocates.  Its scratch memory - the roadgraph points of
 * every scenario bucketed into a uniform grid - lives in an array that is part of the library image:
 * about 13 MiB of every GPU that loads libwm_b200.so, held until the process exits, used or not.
 *
 * Same result as wm_prepare followed by wm_observe (hist = NULL) on a handle with this topk / topk_order,
 * bit for bit: the same two kernels run (bucket the points, then select), both on `stream`, so the
 * bucketing is redone on every call instead of once per episode.
 *   sim, rg, t, rg_index [B][A][topk], rg_feat [B][A][4][topk], rg_type [B][A][topk]: as for wm_observe
 *   (DEVICE pointers owned by the caller, same layouts; only x, y, yaw, valid of `sim` and x, y, dir_x,
 *   dir_y, type, valid of `rg` are read); topk_order = WM_TOPK_BY_INDEX or WM_TOPK_BY_DISTANCE.
 * Limits, fixed when the library is built: B <= WM_STATIC_MAX_B scenarios and B * R <= WM_STATIC_MAX_POINTS
 * roadgraph points per call (e.g. 32 scenarios of 30 000 points).  Anything larger returns WM_ERR_TOO_LARGE
 * and launches nothing; also A <= 1024 and 1 <= topk <= R (WM_ERR_UNSUPPORTED), as for wm_observe.
 * Sharing: there is ONE array per GPU, shared by every call from every thread.  It keeps the last call's
 * contents; nothing in it needs clearing, because the bucketing kernel rewrites every word the selection
 * kernel reads.  Two calls whose kernels may run at the same time on one GPU (different streams without an
 * event between them, or two host threads) RACE on it and return garbage: put all calls on one stream, or
 * order them with events.  The outputs are yours as soon as the work on `stream` has completed.
 * First call on each device: looks up the array's address on that device (cudaGetSymbolAddress, the device
 * being current) and remembers it.  Make that first call during start-up, outside any stream capture.
 */
#define WM_STATIC_MAX_B 64
#define WM_STATIC_MAX_POINTS (1 << 20)
int wm_observe_topk_static(const wm_traj* sim, const wm_roadgraph* rg, int32_t t, int32_t topk, int32_t topk_order,
                           int32_t* rg_index, float* rg_feat, int32_t* rg_type, void* stream);

/*
 * Expert actor = inverse kinematics on the rows of a trajectory ("Expert"; L335 delta
 * inverse; L352-L359 Eq. 3 bicycle inverse), for the dynamics model of the handle.  Step s =
 * 0 .. n_steps-1 uses rows t+s and t+s+1 of `tr`:
 *   bicycle: a = (v' - v)/dt, v = |(vx, vy)|; kappa = wrap(atan2(vy', vx') - yaw) / (v dt + a dt^2/2)
 *            (heading atan2(vy', vx'): D4; difference wrapped into [-pi, pi): D32; kappa = 0 when
 *            v and v' are both exactly 0: D31);
 *   delta:   (dx, dy) = R(-yaw)(p' - p) in the body frame of row t+s (D2), dyaw = yaw' - yaw.
 * action [B][n_steps][C][A] (the layout wm_rollout takes; n_steps = 1: what wm_step takes),
 * action_valid [B][n_steps][A] = both rows valid; action = 0 where not valid.  Replaying the
 * DeltaLocal expert of the log reproduces the log (Table 3: Log ADE 0.00).
 * Requires t >= 0, t + n_steps < T.
 */
int wm_expert_actions(wm_handle* h, const wm_traj* tr, int32_t t, int32_t n_steps, float* action,
                      uint8_t* action_valid, void* stream);

/*
 * Kinematic-infeasibility metric, L104: Eq. 3 on the transitions INTO rows t .. t+n_steps-1 (row
 * t+s-1 -> t+s), whatever the dynamics model of the handle; flag = |a| > max_accel or |kappa| >
 * max_curvature of the config (6 m/s^2, 0.3 1/m), strictly.  accel, curvature (may be NULL), flag
 * [B][n_steps][A]; a transition with an invalid end gives 0 / 0 / flag 0.  Requires t >= 1,
 * t + n_steps <= T.  (L198: actions of the bicycle model inside the limits are never flagged.)
 */
int wm_metrics_kinematic(wm_handle* h, const wm_traj* sim, int32_t t, int32_t n_steps, float* accel,
                         float* curvature, uint8_t* flag, void* stream);

/*
 * Discretised action spaces (L204: "For discrete action spaces, the inverse is computed by discretizing
 * the continuous inverse"; the Bicycle-Discrete / Delta-Discrete spaces of L373).  The paper prints no
 * grids, so they are arguments (D42): channel c has n[c] >= 1 values lo[c] + i (hi[c] - lo[c]) / (n[c] - 1),
 * i = 0 .. n[c]-1.  A continuous value maps to the nearest grid value (ties -> the even bin, values
 * beyond the range -> the end bin); the bin is decided in float32: rint((v - lo) * fl((n-1)/(hi-lo))).
 * The joint index is row-major over the C channels: (i_0 n_1 + i_1) n_2 + i_2.  Channels beyond C are ignored.
 */
typedef struct { int32_t n[3]; float lo[3], hi[3]; } wm_action_grid;

/* action [N][C][A] (N rows, e.g. B*n_steps; C = 2 or 3 as for the handle's dynamics) -> index [N][A]
 * (-1 where valid == 0; valid [N][A] may be NULL = all valid) and dequant [N][C][A], the grid values
 * (0 where not valid; may be NULL; may alias `action`). */
int wm_discretize_actions(wm_handle* h, const wm_action_grid* grid, int64_t N, int32_t A, const float* action,
                          const uint8_t* valid, int32_t* index, float* dequant, void* stream);
/* index [N][A] -> action [N][C][A]: the grid values, ready for wm_step / wm_rollout.  An index that names no
 * bin of the grid - negative, or >= n[0] * .. * n[C-1] - decodes to the zero action (D45); it never wraps
 * around into some other bin. */
int wm_actions_from_index(wm_handle* h, const wm_action_grid* grid, int64_t N, int32_t A, const int32_t* index,
                          float* action, void* stream);
/* Discrete expert (L204): wm_expert_actions followed by wm_discretize_actions in place.  action
 * [B][n_steps][C][A] receives the de-quantised expert action, index [B][n_steps][A] its joint bin. */
int wm_expert_actions_discrete(wm_handle* h, const wm_traj* tr, int32_t t, int32_t n_steps, const wm_action_grid* grid,
                               int32_t* index, float* action, uint8_t* action_valid, void* stream);

/*
 * Backward pass of the dynamics for differentiable rollouts (L252: "the entire simulation can be assembled
 * within a single ... computation graph"; Eq. 2, Eq. 1): the vector-Jacobian product of
 * the n_steps transitions that produced rows t0+1 .. t0+n_steps of `sim` from row t0 with `actions`.
 * g_rows [B][n_steps][5][A]: cotangents of a loss w.r.t. (x, y, yaw, vel_x, vel_y) of those rows.
 * g_actions [B][n_steps][C][A]: its gradient w.r.t. the actions; g_state0 [B][5][A] (may be NULL): w.r.t.
 * row t0.  A log-playback slot (D8) passes no gradient to its action or to earlier rows; an action
 * beyond the clip limits (D7) has zero gradient; dv/dv_x = 0 at v = 0 (D43).  Reads the stored rows:
 * call it after wm_rollout / wm_step with the same actions.  wm_step_vjp is the n_steps = 1 case
 * (g_next [B][5][A], g_action [B][C][A]).
 */
int wm_rollout_vjp(wm_handle* h, const wm_traj* sim, int32_t t0, int32_t n_steps, const float* actions,
                   const uint8_t* action_valid, const float* g_rows, float* g_actions, float* g_state0, void* stream);
int wm_step_vjp(wm_handle* h, const wm_traj* sim, int32_t t, const float* action, const uint8_t* action_valid,
                const float* g_next, float* g_state, float* g_action, void* stream);

/* One on-route path per agent (L84, L96): points [B][A][P] with the distance along the path from
 * its start (arc_len, an input) and validity.  DEVICE pointers, caller-owned. */
typedef struct {
  int32_t B, A, P;
  const float *x, *y, *arc_len;
  const uint8_t* valid;
} wm_paths;

/*
 * Route-progress ratio, L96: for every agent, x(t) = the valid path point closest to the simulated
 * position at row t (closest POINT, ties -> lower index; float32 key fma(dy, dy, dx*dx), D33);
 * ratio = (arc_len[x(t)] - d_p) / (d_q - d_p), d_p / d_q = arc length of the path points closest
 * to the agent's first / last VALID logged position (D34); it may exceed 1 or be negative.
 * ratio [B][A], valid [B][A] = sim valid at t, a valid path point, a valid logged row and
 * d_q != d_p (D35); ratio = 0 where not valid.  Requires 0 <= t < T and paths of the same B, A.
 */
int wm_metrics_route_progress(wm_handle* h, const wm_traj* log, const wm_traj* sim, int32_t t,
                              const wm_paths* paths, float* ratio, uint8_t* valid, void* stream);

/*
 * Off-route metric, L98: "sufficiently closer to an off-route path than on-route path or ... far
 * enough away from an on-route path".  The paper gives no thresholds: they are arguments (D36).
 * d_on / d_off = distance from the agent's position at row t to the closest valid point of its
 * on-route / off-route path (float32 key and square root; +inf without an off-route point);
 *   flag = d_on > max_dist || d_off + margin < d_on
 * for agents valid at t with an on-route path point, else flag 0 and dist_on 0.  off_route may be
 * NULL.  dist_on [B][A] (may be NULL), flag [B][A].
 */
int wm_metrics_offroute(wm_handle* h, const wm_traj* sim, int32_t t, const wm_paths* on_route,
                        const wm_paths* off_route, float max_dist, float margin, float* dist_on,
                        uint8_t* flag, void* stream);

/* Constants of the intelligent driver model (ref. [51] of the paper: Treiber, Hennecke, Helbing 2000).
 * The paper gives none (D37); typical values: v0 = 30 m/s desired speed, T = 1.5 s time headway,
 * s0 = 2 m minimum gap, a_max = 1 m/s^2, b = 1.5 m/s^2 comfortable deceleration, delta = 4,
 * b_max = 4 m/s^2 hardest braking. */
typedef struct { float v0, T, s0, a_max, b, delta, b_max; } wm_idm_params;

/*
 * IDM reactive sim agent, L110-L112: the agent "follows the logged path" (its `paths` polyline) with
 * the speed profile of the intelligent driver model,
 *   a = a_max [1 - (v/v0)^delta - (s_star/s)^2],  s_star = s0 + max(0, v T + v (v - v_lead) / (2 sqrt(a_max b))),
 * s = bumper-to-bumper gap along the path to the lead object (no lead: last term 0).  Readings
 * D38-D41: path coordinate = arc length of the projection on the nearest path segment;
 * lead = the valid other agent whose projection on this agent's path is ahead, within (W_i + W_j)/2
 * of the path, with the smallest gap sigma_j - sigma_i - (L_i + L_j)/2 (ties -> lower index), lead
 * speed |v_j|; a clamped to [-b_max, a_max], gap to >= 0.1 m; v' = max(0, v + a dt); the agent advances
 * (v + v') dt / 2 along the path (stops on its last point), yaw' = direction of the path piece it
 * lands on, velocity v' (cos yaw', sin yaw').
 * Writes row t+1 of `sim` ONLY for agents with idm_valid != 0 that are valid at row t and have a
 * path segment (valid' = 1, box kept); every other slot of row t+1 is left untouched - call wm_step
 * first (dynamics / log playback for everybody), then this.  Reads row t only.
 * accel [B][A] (may be NULL): the IDM acceleration; lead [B][A] (may be NULL): lead agent or -1.
 */
int wm_idm_step(wm_handle* h, wm_traj* sim, int32_t t, const wm_paths* paths, const uint8_t* idm_valid,
                const wm_idm_params* params, float* accel, int32_t* lead, void* stream);

/*
 * Rollout, L200: for s = 0 .. n_steps-1: wm_step at t0+s, then overlap, offroad and log
 * divergence on row t0+s+1 (D11), written to row s of the per-step outputs; aggregates over
 * the n_steps rows at the end.  The whole sequence is one CUDA graph, captured on the first
 * call for a given argument set and replayed afterwards (re-captured when any pointer or
 * shape changes); no host synchronisation inside.
 * actions [B][n_steps][C][A]; action_valid [B][n_steps][A].
 */
int wm_rollout(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t0, int32_t n_steps,
               const float* actions, const uint8_t* action_valid, const wm_rollout_out* out,
               void* stream);

/*
 * The same job from HOST memory (pinned recommended): uploads the scenario (log, roadgraph)
 * and the actions, runs wm_prepare, wm_reset and wm_rollout from t0 = history-1, downloads the
 * metric rows and aggregates into the HOST buffers of `out`, and, when sim_host is not NULL,
 * the simulated trajectory.  Device staging buffers are owned by the handle and reused.
 * Scenarios are independent (L82), so the work is pipelined over up to 16 chunks of scenarios on
 * the caller's stream (uploads) and three streams of the handle (prepare, rollout, downloads): the
 * device work hides under the PCIe upload.  The uploads are enqueued on `stream`; it is
 * synchronised once early (the record count of the road edges fixes the buffer sizes).
 * SYNCHRONISES before returning.  All pointers inside the structs are HOST pointers.
 */
int wm_rollout_host(wm_handle* h, const wm_traj* log_host, const wm_roadgraph* rg_host,
                    int32_t n_steps, const float* actions_host, const uint8_t* action_valid_host,
                    const wm_rollout_out* out_host, wm_traj* sim_host, void* stream);

/* Introspection for tests and the bench (HOST outputs; each synchronises the stream).
 * wm_segment_counts: n_seg [B] int32 copied to HOST.  wm_kernel_launches: number of kernels
 * this handle has launched (graph replays count their kernel nodes). */
int wm_segment_counts(wm_handle* h, int32_t* n_seg_host, int32_t B, void* stream);
int64_t wm_kernel_launches(const wm_handle* h);
/* wm_offroad_stats: counters of the exact grid search (WM_OFFROAD_CULLED) since the last call,
 * out_host[4] int64 on the HOST: [0] corner-segment pairs evaluated, [1] pairs a brute-force
 * search would have evaluated for the same launches, [2] corners that took the full chunk
 * search (outside the grid or a crowded cell), [3] corners queried.  Resets the counters.
 * Counting costs global atomics, so it is off until wm_offroad_stats_enable(h, 1); toggling it
 * drops a cached rollout graph.  All 0 in brute-force mode. */
int wm_offroad_stats(wm_handle* h, int64_t* out_host, void* stream);
/* wm_grid_stats: the prepared search grids (WM_OFFROAD_CULLED), summed over the scenarios of the last wm_prepare:
 * out_host[6] int64 on the HOST = {inner cells, inner cells without a list, mid cells, mid cells without a list,
 * outer cells, outer cells without a list}.  A cell "without a list" has too many candidate segments (or its
 * parent had): queries landing in it take the exact search over all segments - slower, same result.  Dense
 * roadgraphs (config 4: points 0.1 m apart) have many such cells.  Synchronises.  WM_ERR_STATE before wm_prepare. */
int wm_grid_stats(wm_handle* h, int64_t* out_host, void* stream);
int wm_offroad_stats_enable(wm_handle* h, int32_t on);

/* Diagnostics for the bench (HOST outputs; both synchronise the stream).
 * wm_rollout_kernel_times: runs the fused rollout's two kernels once, eagerly, with CUDA events around
 * each: ms_host[0] = k_rollout_dyn, ms_host[1] = k_rollout_metrics (a graph replay cannot be timed node
 * by node).  Same arguments and results as wm_rollout; WM_ERR_UNSUPPORTED outside the fused mode.
 * wm_selftest_ffma: duration of a register-resident FFMA (packed = 0) / FFMA2 (packed = 1) loop on `ctas`
 * CTAs of 256 threads, `iters` x 32 FMAs per thread, and the flop it executed: the measured FP32 peak. */
int wm_rollout_kernel_times(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t0, int32_t n_steps,
                            const float* actions, const uint8_t* action_valid, const wm_rollout_out* out,
                            float* ms_host, void* stream);
int wm_selftest_ffma(wm_handle* h, int32_t packed, int32_t ctas, int32_t iters, float* ms_host, double* flop_host, void* stream);

#ifdef __cplusplus
}
#endif
#endif /* WM_H_ */
