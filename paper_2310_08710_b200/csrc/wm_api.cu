// C-ABI entry points (include/wm.h): argument checks, handle state, rollout graph capture,
// host-buffer staging.  Every step of the path runs in the kernels of the sibling files.
#include <stdlib.h>
#include <string.h>

#include "wm_internal.cuh"

thread_local int g_wm_last_cuda_error = 0;

extern "C" int wm_last_cuda_error(void) { return g_wm_last_cuda_error; }
extern "C" const char* wm_version(void) { return "wm_b200 0.1 (sm_100a; FFMA2 offroad scan, bulk-TMA tiles, CUDA-graph rollout)"; }

static bool aligned16(const void* p) { return ((uintptr_t)p & 15u) == 0; }

static bool traj_ok(const wm_traj* t) {
  if (!t || t->B < 1 || t->A < 1 || t->T < 1) return false;
  const void* ptrs[8] = {t->x, t->y, t->yaw, t->vel_x, t->vel_y, t->length, t->width, t->valid};
  for (int i = 0; i < 8; ++i) if (!ptrs[i] || !aligned16(ptrs[i])) return false;
  return true;
}
static bool rg_ok(const wm_roadgraph* g) {
  if (!g || g->B < 1 || g->R < 1) return false;
  const void* ptrs[7] = {g->x, g->y, g->dir_x, g->dir_y, g->type, g->id, g->valid};
  for (int i = 0; i < 7; ++i) if (!ptrs[i] || !aligned16(ptrs[i])) return false;
  return true;
}
static bool same_shape(const wm_traj* a, const wm_traj* b) { return a->B == b->B && a->A == b->A && a->T == b->T; }

// Launch-shape limits, checked by EVERY entry point that launches over scenarios and agents (wm.h "Limits"):
// several kernels put the scenario in gridDim.y (<= 65 535) and hold a row of agents in one CTA (A <= 1024);
// the others run a 1-D grid of 256-thread blocks over `elems` items (<= 2^31 - 1 blocks).  A shape beyond them
// is refused here instead of coming back as a failed launch.
static int shape_guard(int64_t B, int64_t A, int64_t elems) {
  if (A > 1024 || B > WM_MAX_B) return WM_ERR_UNSUPPORTED;
  if (elems > (int64_t)0x7fffffff * 128) return WM_ERR_UNSUPPORTED;
  return WM_OK;
}
#define WM_SHAPE(B, A, elems) do { const int rc__ = shape_guard((B), (A), (elems)); if (rc__ != WM_OK) return rc__; } while (0)

extern "C" int wm_create(wm_handle** out, const wm_config* cfg) {
  if (!out || !cfg) return WM_ERR_ARG;
  if (cfg->dynamics != WM_DYN_INVERTIBLE_BICYCLE && cfg->dynamics != WM_DYN_DELTA_LOCAL && cfg->dynamics != WM_DYN_DELTA_GLOBAL) return WM_ERR_ARG;
  if (!(cfg->dt > 0.f) || cfg->history < 1 || cfg->topk < 0) return WM_ERR_ARG;
  if (cfg->offroad_mode != WM_OFFROAD_CULLED && cfg->offroad_mode != WM_OFFROAD_BRUTE_FORCE) return WM_ERR_ARG;
  if (cfg->rollout_mode != WM_ROLLOUT_FUSED && cfg->rollout_mode != WM_ROLLOUT_STEPWISE) return WM_ERR_ARG;
  if (cfg->topk_order != WM_TOPK_BY_INDEX && cfg->topk_order != WM_TOPK_BY_DISTANCE) return WM_ERR_ARG;
  wm_handle* h = (wm_handle*)calloc(1, sizeof(wm_handle));
  if (!h) return WM_ERR_ARG;
  h->cfg = *cfg;
  cudaError_t e = cudaGetDevice(&h->device);
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&h->num_sms, cudaDevAttrMultiProcessorCount, h->device);
  int major = 0;
  if (e == cudaSuccess) e = cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, h->device);
  if (e != cudaSuccess) { g_wm_last_cuda_error = (int)e; free(h); return WM_ERR_CUDA; }
  if (major != 10) { free(h); return WM_ERR_UNSUPPORTED; }    // sm_100a kernels only; no fallback
  e = cudaStreamCreateWithFlags(&h->cap_stream, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->roll_stream, cudaStreamNonBlocking);
  if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&h->d2h_stream, cudaStreamNonBlocking);
  for (int i = 0; i < WM_HOST_CHUNKS && e == cudaSuccess; ++i) {
    e = cudaEventCreateWithFlags(&h->ev_up[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_prep[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaEventCreateWithFlags(&h->ev_done[i], cudaEventDisableTiming);
  }
  if (e == cudaSuccess) e = cudaMalloc(&h->cull_stats, 16 * sizeof(unsigned long long));
  if (e == cudaSuccess) e = cudaMemset(h->cull_stats, 0, 16 * sizeof(unsigned long long));
  if (e != cudaSuccess) { g_wm_last_cuda_error = (int)e; wm_destroy(h); return WM_ERR_CUDA; }   // frees what was created so far
  *out = h;
  return WM_OK;
}

extern "C" int wm_offroad_stats(wm_handle* h, int64_t* out_host, void* stream) {
  if (!h || !out_host) return WM_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long v[4];
  WM_CUDA(cudaMemcpyAsync(v, h->cull_stats, sizeof(v), cudaMemcpyDeviceToHost, s));
  WM_CUDA(cudaMemsetAsync(h->cull_stats, 0, sizeof(v), s));
  WM_CUDA(cudaStreamSynchronize(s));
  for (int i = 0; i < 4; ++i) out_host[i] = (int64_t)v[i];
  return WM_OK;
}

extern "C" int wm_grid_stats(wm_handle* h, int64_t* out_host, void* stream) {
  if (!h || !out_host) return WM_ERR_ARG;
  if (!h->seg_ready || !h->cells) return WM_ERR_STATE;
  cudaStream_t s = (cudaStream_t)stream;
  unsigned long long v[6];
  unsigned long long* d = h->cull_stats + 8;
  WM_CUDA(cudaMemsetAsync(d, 0, sizeof(v), s));
  WM_CUDA(wm_launch_grid_cell_stats(h, d, s));
  WM_CUDA(cudaMemcpyAsync(v, d, sizeof(v), cudaMemcpyDeviceToHost, s));
  WM_CUDA(cudaStreamSynchronize(s));
  for (int i = 0; i < 6; ++i) out_host[i] = (int64_t)v[i];
  return WM_OK;
}

extern "C" int wm_offroad_stats_enable(wm_handle* h, int32_t on) {
  if (!h) return WM_ERR_ARG;
  if ((h->stats_on != 0) != (on != 0)) wm_drop_graph(h);     // the counter pointer is a kernel argument
  h->stats_on = on != 0;
  return WM_OK;
}

void wm_drop_graph(wm_handle* h) {
  if (h->graph_exec) cudaGraphExecDestroy(h->graph_exec);
  if (h->graph) cudaGraphDestroy(h->graph);
  h->graph_exec = nullptr; h->graph = nullptr; h->graph_kernels = 0;
  memset(h->graph_key, 0, sizeof(h->graph_key));
}

extern "C" int wm_destroy(wm_handle* h) {
  if (!h) return WM_ERR_ARG;
  int cur = -1;                                       // the handle's device, not whichever is current
  cudaGetDevice(&cur);
  if (cur != h->device) cudaSetDevice(h->device);
  cudaDeviceSynchronize();
  wm_drop_graph(h);
  wm_prepare_free(h);
  cudaFree(h->scratch);
  cudaFree(h->cull_stats);
  for (int i = 0; i < 16; ++i) cudaFree(h->stage[i]);
  if (h->cap_stream) cudaStreamDestroy(h->cap_stream);
  if (h->roll_stream) cudaStreamDestroy(h->roll_stream);
  if (h->d2h_stream) cudaStreamDestroy(h->d2h_stream);
  for (int i = 0; i < WM_HOST_CHUNKS; ++i) {
    if (h->ev_up[i]) cudaEventDestroy(h->ev_up[i]);
    if (h->ev_prep[i]) cudaEventDestroy(h->ev_prep[i]);
    if (h->ev_done[i]) cudaEventDestroy(h->ev_done[i]);
  }
  if (cur >= 0 && cur != h->device) cudaSetDevice(cur);
  free(h);
  return WM_OK;
}

extern "C" int64_t wm_kernel_launches(const wm_handle* h) { return h ? h->launches : 0; }

extern "C" int wm_prepare(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, void* stream) {
  if (!h || !rg_ok(rg)) return WM_ERR_ARG;
  if (rg->B > WM_MAX_B) return WM_ERR_UNSUPPORTED;
  return wm_prepare_impl(h, rg, n_segments_max, (cudaStream_t)stream);
}

extern "C" int wm_segment_counts(wm_handle* h, int32_t* n_seg_host, int32_t B, void* stream) {
  if (!h || !n_seg_host) return WM_ERR_ARG;
  if (!h->n_seg || B != h->prep_B) return WM_ERR_STATE;
  WM_CUDA(cudaMemcpyAsync(n_seg_host, h->n_seg, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToHost, (cudaStream_t)stream));
  WM_CUDA(cudaStreamSynchronize((cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_reset(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t* t, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim)) return WM_ERR_ARG;
  if (h->cfg.history > sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  WM_CUDA(wm_launch_reset(h, *log, *sim, h->cfg.history, (cudaStream_t)stream));
  if (t) *t = h->cfg.history - 1;
  return WM_OK;
}

extern "C" int wm_step(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t, const float* action,
                       const uint8_t* action_valid, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim) || !action || !action_valid) return WM_ERR_ARG;
  if (t < 0 || t + 1 >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  const int C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  WM_CUDA(wm_launch_step(h, *log, *sim, t, action, (int64_t)C * sim->A, action_valid, sim->A, nullptr, nullptr, 0,
                         (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_metrics_overlap(wm_handle* h, const wm_traj* sim, int32_t t, uint32_t* pair_bits,
                                  uint8_t* agent_flag, void* stream) {
  if (!h || !traj_ok(sim) || !agent_flag) return WM_ERR_ARG;
  if (t < 0 || t >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  WM_CUDA(wm_launch_overlap(h, *sim, t, pair_bits, agent_flag, sim->A, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_metrics_offroad(wm_handle* h, const wm_traj* sim, int32_t t, float* signed_dist,
                                  float* corner_dist, uint8_t* agent_flag, void* stream) {
  if (!h || !traj_ok(sim) || !signed_dist || !agent_flag) return WM_ERR_ARG;
  if (t < 0 || t >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  if (!h->seg_ready || h->prep_B != sim->B) return WM_ERR_STATE;
  WM_CUDA(wm_launch_offroad(h, *sim, t, signed_dist, sim->A, corner_dist, agent_flag, sim->A, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_log_divergence(wm_handle* h, const wm_traj* log, const wm_traj* sim, int32_t t, float* dist,
                                 uint8_t* valid, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim) || !dist) return WM_ERR_ARG;
  if (t < 0 || t >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  WM_CUDA(wm_launch_logdiv(h, *log, *sim, t, dist, valid, sim->A, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_expert_actions(wm_handle* h, const wm_traj* tr, int32_t t, int32_t n_steps, float* action,
                                 uint8_t* action_valid, void* stream) {
  if (!h || !traj_ok(tr) || !action || !action_valid) return WM_ERR_ARG;
  if (n_steps < 1 || t < 0 || t + n_steps >= tr->T) return WM_ERR_ARG;
  WM_SHAPE(tr->B, tr->A, (int64_t)tr->B * n_steps * tr->A);
  WM_CUDA(wm_launch_expert(h, *tr, t, n_steps, action, action_valid, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_metrics_kinematic(wm_handle* h, const wm_traj* sim, int32_t t, int32_t n_steps, float* accel,
                                    float* curvature, uint8_t* flag, void* stream) {
  if (!h || !traj_ok(sim) || !flag) return WM_ERR_ARG;
  if (n_steps < 1 || t < 1 || t + n_steps > sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * n_steps * sim->A);
  if (!(h->cfg.max_accel > 0.f) || !(h->cfg.max_curvature > 0.f)) return WM_ERR_UNSUPPORTED;   // the metric needs its limits
  WM_CUDA(wm_launch_kinematic(h, *sim, t, n_steps, accel, curvature, flag, (cudaStream_t)stream));
  return WM_OK;
}

static bool grid_ok(const wm_action_grid* g, int C) {
  if (!g) return false;
  int64_t total = 1;
  for (int c = 0; c < C; ++c) {
    if (g->n[c] < 1 || (g->n[c] > 1 && !(g->hi[c] > g->lo[c]))) return false;
    total *= g->n[c];
    if (total > 0x7fffffffLL) return false;
  }
  return true;
}

extern "C" int wm_discretize_actions(wm_handle* h, const wm_action_grid* grid, int64_t N, int32_t A, const float* action,
                                     const uint8_t* valid, int32_t* index, float* dequant, void* stream) {
  const int C = h && h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  if (!h || !grid_ok(grid, C) || N < 1 || A < 1 || !action || !index) return WM_ERR_ARG;
  if (N > (int64_t)0x7fffffff * 128 / A) return WM_ERR_UNSUPPORTED;           // the 1-D grid over N * A items
  WM_CUDA(wm_launch_discretize(h, *grid, C, N, A, action, valid, index, dequant, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_actions_from_index(wm_handle* h, const wm_action_grid* grid, int64_t N, int32_t A, const int32_t* index,
                                     float* action, void* stream) {
  const int C = h && h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  if (!h || !grid_ok(grid, C) || N < 1 || A < 1 || !action || !index) return WM_ERR_ARG;
  if (N > (int64_t)0x7fffffff * 128 / A) return WM_ERR_UNSUPPORTED;           // the 1-D grid over N * A items
  WM_CUDA(wm_launch_from_index(h, *grid, C, N, A, index, action, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_expert_actions_discrete(wm_handle* h, const wm_traj* tr, int32_t t, int32_t n_steps, const wm_action_grid* grid,
                                          int32_t* index, float* action, uint8_t* action_valid, void* stream) {
  const int C = h && h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  if (!h || !traj_ok(tr) || !grid_ok(grid, C) || !action || !action_valid || !index) return WM_ERR_ARG;
  if (n_steps < 1 || t < 0 || t + n_steps >= tr->T) return WM_ERR_ARG;
  WM_SHAPE(tr->B, tr->A, (int64_t)tr->B * n_steps * tr->A);
  WM_CUDA(wm_launch_expert(h, *tr, t, n_steps, action, action_valid, (cudaStream_t)stream));
  WM_CUDA(wm_launch_discretize(h, *grid, C, (int64_t)tr->B * n_steps, tr->A, action, action_valid, index, action, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_rollout_vjp(wm_handle* h, const wm_traj* sim, int32_t t0, int32_t n_steps, const float* actions,
                              const uint8_t* action_valid, const float* g_rows, float* g_actions, float* g_state0, void* stream) {
  if (!h || !traj_ok(sim) || !actions || !action_valid || !g_rows || !g_actions) return WM_ERR_ARG;
  if (n_steps < 1 || t0 < 0 || t0 + n_steps >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  WM_CUDA(wm_launch_rollout_vjp(h, *sim, t0, n_steps, actions, action_valid, g_rows, g_actions, g_state0, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_step_vjp(wm_handle* h, const wm_traj* sim, int32_t t, const float* action, const uint8_t* action_valid,
                           const float* g_next, float* g_state, float* g_action, void* stream) {
  return wm_rollout_vjp(h, sim, t, 1, action, action_valid, g_next, g_action, g_state, stream);
}

extern "C" int wm_metrics_route_progress(wm_handle* h, const wm_traj* log, const wm_traj* sim, int32_t t, const wm_paths* paths,
                                         float* ratio, uint8_t* valid, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim) || !paths || !ratio || !valid) return WM_ERR_ARG;
  if (t < 0 || t >= sim->T) return WM_ERR_ARG;
  if (paths->B != sim->B || paths->A != sim->A || paths->P < 1 || !paths->x || !paths->y || !paths->arc_len || !paths->valid) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);                            // the scenario is gridDim.y
  WM_CUDA(wm_launch_route_progress(h, *log, *sim, t, *paths, ratio, valid, (cudaStream_t)stream));
  return WM_OK;
}

static bool paths_ok(const wm_paths* p, const wm_traj* sim) {
  return p && p->B == sim->B && p->A == sim->A && p->P >= 1 && p->x && p->y && p->arc_len && p->valid;
}

extern "C" int wm_metrics_offroute(wm_handle* h, const wm_traj* sim, int32_t t, const wm_paths* on_route, const wm_paths* off_route,
                                   float max_dist, float margin, float* dist_on, uint8_t* flag, void* stream) {
  if (!h || !traj_ok(sim) || !paths_ok(on_route, sim) || (off_route && !paths_ok(off_route, sim)) || !flag) return WM_ERR_ARG;
  if (t < 0 || t >= sim->T || !(max_dist >= 0.f) || !(margin >= 0.f)) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A * 32);                       // a warp per agent
  WM_CUDA(wm_launch_offroute(h, *sim, t, *on_route, off_route, max_dist, margin, dist_on, flag, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_idm_step(wm_handle* h, wm_traj* sim, int32_t t, const wm_paths* paths, const uint8_t* idm_valid,
                           const wm_idm_params* params, float* accel, int32_t* lead, void* stream) {
  if (!h || !traj_ok(sim) || !paths_ok(paths, sim) || !idm_valid || !params) return WM_ERR_ARG;
  if (t < 0 || t + 1 >= sim->T) return WM_ERR_ARG;
  if (!(params->v0 > 0.f) || !(params->a_max > 0.f) || !(params->b > 0.f) || !(params->b_max > 0.f) || !(params->T >= 0.f) ||
      !(params->s0 >= 0.f) || !(params->delta > 0.f)) return WM_ERR_ARG;
  if (paths->P > 1900) return WM_ERR_UNSUPPORTED;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A * 32);                       // a warp per agent
  WM_CUDA(wm_launch_idm_step(h, *sim, t, *paths, idm_valid, *params, accel, lead, (cudaStream_t)stream));
  return WM_OK;
}

extern "C" int wm_observe(wm_handle* h, const wm_traj* sim, const wm_roadgraph* rg, int32_t t, float* hist,
                          uint8_t* hist_valid, int32_t* rg_index, float* rg_feat, int32_t* rg_type, void* stream) {
  if (!h || !traj_ok(sim)) return WM_ERR_ARG;
  const bool want_hist = hist || hist_valid, want_topk = rg_index || rg_feat || rg_type;
  if (want_hist && !(hist && hist_valid)) return WM_ERR_ARG;
  if (want_topk && !(rg_index && rg_feat && rg_type && rg_ok(rg))) return WM_ERR_ARG;
  if (t < h->cfg.history - 1 || t >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  if (want_hist) WM_CUDA(wm_launch_observe_hist(h, *sim, t, hist, hist_valid, (cudaStream_t)stream));
  if (want_topk) {
    if (h->cfg.topk < 1 || h->cfg.topk > rg->R) return WM_ERR_UNSUPPORTED;
    if (!h->pt_xy || h->prep_B != sim->B || h->prep_R != rg->R || rg->B != sim->B) return WM_ERR_STATE;
    WM_CUDA(wm_launch_observe_topk(h, *sim, *rg, t, rg_index, rg_feat, rg_type, (cudaStream_t)stream));
  }
  return WM_OK;
}

// ---------------------------------------------------------------------------------------
// rollout: n_steps x {step (+log divergence) -> overlap -> offroad}, aggregates; one graph.
// ---------------------------------------------------------------------------------------
static int ensure_scratch(wm_handle* h, size_t bytes) {
  if (h->scratch_bytes >= bytes) return WM_OK;
  wm_drop_graph(h);
  cudaFree(h->scratch); h->scratch = nullptr; h->scratch_bytes = 0;
  WM_CUDA(cudaMalloc(&h->scratch, bytes));
  h->scratch_bytes = bytes;
  return WM_OK;
}

static int enqueue_rollout(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                           const float* actions, const uint8_t* action_valid, const wm_rollout_out& o,
                           uint8_t* ld_valid_rows, cudaStream_t s) {
  const int A = sim.A;
  const int C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  const int64_t row_stride = (int64_t)n_steps * A;
  for (int k = 0; k < n_steps; ++k) {
    const int t = t0 + k;
    WM_CUDA(wm_launch_step(h, log, sim, t, actions + (int64_t)k * C * A, (int64_t)n_steps * C * A,
                           action_valid + (int64_t)k * A, row_stride, o.log_div + (int64_t)k * A,
                           ld_valid_rows + (int64_t)k * A, row_stride, s));
    WM_CUDA(wm_launch_overlap(h, sim, t + 1, nullptr, o.overlap + (int64_t)k * A, row_stride, s));
    WM_CUDA(wm_launch_offroad(h, sim, t + 1, o.offroad_dist + (int64_t)k * A, row_stride, nullptr,
                              o.offroad + (int64_t)k * A, row_stride, s));
  }
  WM_CUDA(wm_launch_aggregate(h, sim.B, A, n_steps, o, ld_valid_rows, s));
  return WM_OK;
}

extern "C" int wm_rollout(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t0, int32_t n_steps,
                          const float* actions, const uint8_t* action_valid, const wm_rollout_out* out, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim) || !actions || !action_valid || !out) return WM_ERR_ARG;
  if (n_steps < 1 || t0 < 0 || t0 + n_steps >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  if (!h->seg_ready || h->prep_B != sim->B) return WM_ERR_STATE;
  const bool fused = h->cfg.rollout_mode == WM_ROLLOUT_FUSED && h->cfg.offroad_mode == WM_OFFROAD_CULLED &&
                     n_steps < 60000;                  // its hash entries carry a 16-bit block number
  const int64_t rows = fused ? 0 : (int64_t)sim->B * n_steps * sim->A;
  // stepwise: rows the caller did not ask for still feed the aggregates: put them in scratch
  size_t need = (size_t)rows;                                  // ld_valid rows (uint8)
  need = (need + 255) / 256 * 256;
  const size_t off_ov = need;    if (!out->overlap) need += (size_t)rows;
  need = (need + 255) / 256 * 256;
  const size_t off_of = need;    if (!out->offroad) need += (size_t)rows;
  need = (need + 255) / 256 * 256;
  const size_t off_sd = need;    if (!out->offroad_dist) need += (size_t)rows * 4;
  need = (need + 255) / 256 * 256;
  const size_t off_ld = need;    if (!out->log_div) need += (size_t)rows * 4;
  int rc = ensure_scratch(h, need);
  if (rc != WM_OK) return rc;
  unsigned char* sc = (unsigned char*)h->scratch;
  wm_rollout_out o = *out;
  if (!fused) {
  if (!o.overlap) o.overlap = sc + off_ov;
  if (!o.offroad) o.offroad = sc + off_of;
  if (!o.offroad_dist) o.offroad_dist = (float*)(sc + off_sd);
  if (!o.log_div) o.log_div = (float*)(sc + off_ld);
  }
  uint8_t* ld_valid_rows = sc;

  // cache key of the captured graph: every pointer and shape in a slot of its own
  uint64_t key[WM_GRAPH_KEY_WORDS];
  memset(key, 0, sizeof(key));
  const uint64_t words[] = {
      (uint64_t)(uintptr_t)log->x, (uint64_t)(uintptr_t)log->y, (uint64_t)(uintptr_t)log->yaw, (uint64_t)(uintptr_t)log->vel_x,
      (uint64_t)(uintptr_t)log->vel_y, (uint64_t)(uintptr_t)log->length, (uint64_t)(uintptr_t)log->width, (uint64_t)(uintptr_t)log->valid,
      (uint64_t)(uintptr_t)sim->x, (uint64_t)(uintptr_t)sim->y, (uint64_t)(uintptr_t)sim->yaw, (uint64_t)(uintptr_t)sim->vel_x,
      (uint64_t)(uintptr_t)sim->vel_y, (uint64_t)(uintptr_t)sim->length, (uint64_t)(uintptr_t)sim->width, (uint64_t)(uintptr_t)sim->valid,
      (uint64_t)(uintptr_t)actions, (uint64_t)(uintptr_t)action_valid,
      (uint64_t)(uintptr_t)o.overlap, (uint64_t)(uintptr_t)o.offroad, (uint64_t)(uintptr_t)o.offroad_dist, (uint64_t)(uintptr_t)o.log_div,
      (uint64_t)(uintptr_t)o.any_overlap, (uint64_t)(uintptr_t)o.any_offroad, (uint64_t)(uintptr_t)o.ade,
      (uint64_t)sim->B, (uint64_t)sim->A, (uint64_t)sim->T, (uint64_t)(uint32_t)t0, (uint64_t)(uint32_t)n_steps,
      (uint64_t)h->cfg.dynamics, (uint64_t)(uintptr_t)h->segrec, (uint64_t)(uintptr_t)h->cells, (uint64_t)h->stats_on};
  static_assert(sizeof(words) / sizeof(words[0]) <= WM_GRAPH_KEY_WORDS, "graph key too small for its contents");
  memcpy(key, words, sizeof(words));

  if (!h->graph_exec || memcmp(key, h->graph_key, sizeof(key)) != 0) {
    wm_drop_graph(h);
    const int64_t before = h->launches;
    WM_CUDA(cudaStreamBeginCapture(h->cap_stream, cudaStreamCaptureModeThreadLocal));
    if (fused) {
      cudaError_t le = wm_launch_rollout_fused(h, *log, *sim, t0, n_steps, actions, action_valid, o, 0, h->cap_stream);
      rc = WM_OK;
      if (le != cudaSuccess) { g_wm_last_cuda_error = (int)le; rc = WM_ERR_CUDA; }
    } else {
      rc = enqueue_rollout(h, *log, *sim, t0, n_steps, actions, action_valid, o, ld_valid_rows, h->cap_stream);
    }
    cudaGraph_t g = nullptr;
    cudaError_t e = cudaStreamEndCapture(h->cap_stream, &g);
    h->graph_kernels = h->launches - before;
    h->launches = before;                    // capture launched nothing yet
    if (rc != WM_OK) { if (g) cudaGraphDestroy(g); return rc; }
    WM_CUDA(e);
    h->graph = g;
    WM_CUDA(cudaGraphInstantiate(&h->graph_exec, h->graph, 0));
    memcpy(h->graph_key, key, sizeof(key));
  }
  WM_CUDA(cudaGraphLaunch(h->graph_exec, (cudaStream_t)stream));
  h->launches += h->graph_kernels;
  return WM_OK;
}

// Diagnostics for the bench: the two kernels of the fused rollout launched eagerly with CUDA events
// between them (a graph replay cannot be timed node by node).  Synchronises.
extern "C" int wm_rollout_kernel_times(wm_handle* h, const wm_traj* log, wm_traj* sim, int32_t t0, int32_t n_steps,
                                       const float* actions, const uint8_t* action_valid, const wm_rollout_out* out,
                                       float* ms_host, void* stream) {
  if (!h || !traj_ok(log) || !traj_ok(sim) || !same_shape(log, sim) || !actions || !action_valid || !out || !ms_host) return WM_ERR_ARG;
  if (n_steps < 1 || t0 < 0 || t0 + n_steps >= sim->T) return WM_ERR_ARG;
  WM_SHAPE(sim->B, sim->A, (int64_t)sim->B * sim->A);
  if (!h->seg_ready || h->prep_B != sim->B) return WM_ERR_STATE;
  if (h->cfg.rollout_mode != WM_ROLLOUT_FUSED || h->cfg.offroad_mode != WM_OFFROAD_CULLED) return WM_ERR_UNSUPPORTED;
  cudaStream_t s = (cudaStream_t)stream;
  cudaEvent_t ev[3] = {nullptr, nullptr, nullptr};
  cudaError_t e = cudaSuccess;
  for (int i = 0; i < 3 && e == cudaSuccess; ++i) e = cudaEventCreate(&ev[i]);
  if (e == cudaSuccess) e = wm_launch_rollout_fused_timed(h, *log, *sim, t0, n_steps, actions, action_valid, *out, ev, s);
  if (e == cudaSuccess) e = cudaEventSynchronize(ev[2]);
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms_host[0], ev[0], ev[1]);
  if (e == cudaSuccess) e = cudaEventElapsedTime(&ms_host[1], ev[1], ev[2]);
  for (int i = 0; i < 3; ++i) if (ev[i]) cudaEventDestroy(ev[i]);      // whatever was created, on every exit path
  WM_CUDA(e);
  return WM_OK;
}

// Diagnostics for the bench: duration of a register-resident FFMA (packed = 0) or FFMA2 (packed = 1) loop.
// flop = ctas * 256 * iters * 32 * (packed ? 4 : 2).  Synchronises.
extern "C" int wm_selftest_ffma(wm_handle* h, int32_t packed, int32_t ctas, int32_t iters, float* ms_host, double* flop_host, void* stream) {
  if (!h || !ms_host || ctas < 1 || iters < 1) return WM_ERR_ARG;
  cudaStream_t s = (cudaStream_t)stream;
  cudaEvent_t a = nullptr, b = nullptr;
  cudaError_t e = cudaEventCreate(&a);
  if (e == cudaSuccess) e = cudaEventCreate(&b);
  if (e == cudaSuccess) e = wm_launch_ffma_peak(h, packed, ctas, iters, (float*)h->cull_stats, s);      // warm-up
  if (e == cudaSuccess) e = cudaEventRecord(a, s);
  if (e == cudaSuccess) e = wm_launch_ffma_peak(h, packed, ctas, iters, (float*)h->cull_stats, s);
  if (e == cudaSuccess) e = cudaEventRecord(b, s);
  if (e == cudaSuccess) e = cudaEventSynchronize(b);
  if (e == cudaSuccess) e = cudaEventElapsedTime(ms_host, a, b);
  if (a) cudaEventDestroy(a);
  if (b) cudaEventDestroy(b);
  WM_CUDA(e);
  if (flop_host) *flop_host = (double)ctas * 256.0 * (double)iters * 32.0 * (packed ? 4.0 : 2.0);
  return WM_OK;
}

// ---------------------------------------------------------------------------------------
// the same job from host memory
// ---------------------------------------------------------------------------------------
static int stage_alloc(wm_handle* h, int slot, size_t bytes) {
  if (h->stage_bytes[slot] >= bytes) return WM_OK;
  wm_drop_graph(h);
  cudaFree(h->stage[slot]); h->stage[slot] = nullptr; h->stage_bytes[slot] = 0;
  WM_CUDA(cudaMalloc(&h->stage[slot], bytes));
  h->stage_bytes[slot] = bytes;
  return WM_OK;
}

static size_t al256(size_t n) { return (n + 255) / 256 * 256; }

extern "C" int wm_rollout_host(wm_handle* h, const wm_traj* lh, const wm_roadgraph* gh, int32_t n_steps,
                               const float* actions_host, const uint8_t* action_valid_host,
                               const wm_rollout_out* oh, wm_traj* sim_host, void* stream) {
  if (!h || !lh || !gh || !actions_host || !action_valid_host || !oh) return WM_ERR_ARG;
  if (lh->B < 1 || lh->A < 1 || lh->T < 1 || gh->B != lh->B || gh->R < 1) return WM_ERR_ARG;
  const int B = lh->B, A = lh->A, T = lh->T, R = gh->R;
  const int t0 = h->cfg.history - 1;
  if (n_steps < 1 || t0 + n_steps >= T) return WM_ERR_ARG;
  WM_SHAPE(B, A, (int64_t)B * n_steps * A);
  cudaStream_t s = (cudaStream_t)stream;
  const int C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  const size_t nTA = (size_t)B * T * A, nR = (size_t)B * R, rows = (size_t)B * n_steps * A, nBA = (size_t)B * A;
  // slot 0: log traj, 1: sim traj, 2: roadgraph, 3: actions + valid, 4: outputs
  const size_t traj_bytes = 7 * al256(nTA * 4) + al256(nTA);
  const size_t rg_bytes = 6 * al256(nR * 4) + al256(nR);
  const size_t act_bytes = al256(rows * C * 4) + al256(rows);
  const size_t out_bytes = 2 * al256(rows) + 2 * al256(rows * 4) + 2 * al256(nBA) + al256(nBA * 4);
  int rc;
  if ((rc = stage_alloc(h, 0, traj_bytes)) != WM_OK) return rc;
  if ((rc = stage_alloc(h, 1, traj_bytes)) != WM_OK) return rc;
  if ((rc = stage_alloc(h, 2, rg_bytes)) != WM_OK) return rc;
  if ((rc = stage_alloc(h, 3, act_bytes)) != WM_OK) return rc;
  if ((rc = stage_alloc(h, 4, out_bytes)) != WM_OK) return rc;
  auto carve_traj = [&](void* base, wm_traj& t) {
    unsigned char* p = (unsigned char*)base;
    t.B = B; t.A = A; t.T = T;
    float** f[7] = {&t.x, &t.y, &t.yaw, &t.vel_x, &t.vel_y, &t.length, &t.width};
    for (int i = 0; i < 7; ++i) { *f[i] = (float*)p; p += al256(nTA * 4); }
    t.valid = p;
  };
  wm_traj dl, ds;
  carve_traj(h->stage[0], dl);
  carve_traj(h->stage[1], ds);
  wm_roadgraph dg;
  {
    unsigned char* p = (unsigned char*)h->stage[2];
    dg.B = B; dg.R = R;
    dg.x = (float*)p; p += al256(nR * 4); dg.y = (float*)p; p += al256(nR * 4);
    dg.dir_x = (float*)p; p += al256(nR * 4); dg.dir_y = (float*)p; p += al256(nR * 4);
    dg.type = (int32_t*)p; p += al256(nR * 4); dg.id = (int32_t*)p; p += al256(nR * 4);
    dg.valid = p;
  }
  float* d_act = (float*)h->stage[3];
  uint8_t* d_av = (uint8_t*)h->stage[3] + al256(rows * C * 4);
  wm_rollout_out dout;
  {
    unsigned char* p = (unsigned char*)h->stage[4];
    dout.overlap = p; p += al256(rows); dout.offroad = p; p += al256(rows);
    dout.offroad_dist = (float*)p; p += al256(rows * 4); dout.log_div = (float*)p; p += al256(rows * 4);
    dout.any_overlap = p; p += al256(nBA); dout.any_offroad = p; p += al256(nBA);
    dout.ade = (float*)p;
  }
#define H2D(dst, src, n) WM_CUDA(cudaMemcpyAsync((dst), (src), (n), cudaMemcpyHostToDevice, s))
#define D2H(dst, src, n) do { if (dst) WM_CUDA(cudaMemcpyAsync((dst), (src), (n), cudaMemcpyDeviceToHost, s3)); } while (0)
  // Pipeline over chunks of scenarios (they are independent, L82).  All uploads go down the caller's
  // stream in this order: the roadgraph's type / id / valid of the whole batch (what the record
  // count needs, which fixes the buffer capacity), then chunk by chunk the rest of the roadgraph,
  // the logged trajectories and the actions.  While chunk c + 1 crosses PCIe, chunk c is prepared
  // (cap_stream), rolled out (roll_stream) and its metric rows go back (d2h_stream).
  cudaStream_t s2 = h->cap_stream, s4 = h->roll_stream, s3 = h->d2h_stream;
  H2D(dg.type, gh->type, nR * 4); H2D(dg.id, gh->id, nR * 4); H2D(dg.valid, gh->valid, nR);
  if ((rc = wm_prepare_count(h, &dg, nullptr, s)) != WM_OK) return rc;          // synchronises s
  const bool fused = h->cfg.rollout_mode == WM_ROLLOUT_FUSED && h->cfg.offroad_mode == WM_OFFROAD_CULLED && n_steps < 60000;
  int nchunk = fused ? (B + 255) / 256 : 1;
  if (nchunk > WM_HOST_CHUNKS) nchunk = WM_HOST_CHUNKS;
  const int per = (B + nchunk - 1) / nchunk;
  for (int c = 0; c < nchunk; ++c) {
    const int b0 = c * per, nb = (b0 + per <= B ? per : B - b0);
    if (nb <= 0) break;
    const size_t oR = (size_t)b0 * R, cR = (size_t)nb * R, oT = (size_t)b0 * T * A, cT = (size_t)nb * T * A;
    const size_t oW = (size_t)b0 * n_steps * A, cW = (size_t)nb * n_steps * A, oA = (size_t)b0 * A, cA = (size_t)nb * A;
    H2D(dg.x + oR, gh->x + oR, cR * 4); H2D(dg.y + oR, gh->y + oR, cR * 4);
    H2D(dg.dir_x + oR, gh->dir_x + oR, cR * 4); H2D(dg.dir_y + oR, gh->dir_y + oR, cR * 4);
    H2D(dl.x + oT, lh->x + oT, cT * 4); H2D(dl.y + oT, lh->y + oT, cT * 4); H2D(dl.yaw + oT, lh->yaw + oT, cT * 4);
    H2D(dl.vel_x + oT, lh->vel_x + oT, cT * 4); H2D(dl.vel_y + oT, lh->vel_y + oT, cT * 4);
    H2D(dl.length + oT, lh->length + oT, cT * 4); H2D(dl.width + oT, lh->width + oT, cT * 4); H2D(dl.valid + oT, lh->valid + oT, cT);
    H2D(d_act + oW * C, actions_host + oW * C, cW * C * 4); H2D(d_av + oW, action_valid_host + oW, cW);
    WM_CUDA(cudaEventRecord(h->ev_up[c], s));
    WM_CUDA(cudaStreamWaitEvent(s2, h->ev_up[c], 0));
    if ((rc = wm_prepare_build(h, &dg, b0, nb, s2)) != WM_OK) return rc;
    WM_CUDA(cudaEventRecord(h->ev_prep[c], s2));
    WM_CUDA(cudaStreamWaitEvent(s4, h->ev_prep[c], 0));
    wm_traj cl = dl, cs = ds;
    cl.B = nb; cs.B = nb;
    cl.x += oT; cl.y += oT; cl.yaw += oT; cl.vel_x += oT; cl.vel_y += oT; cl.length += oT; cl.width += oT; cl.valid += oT;
    cs.x += oT; cs.y += oT; cs.yaw += oT; cs.vel_x += oT; cs.vel_y += oT; cs.length += oT; cs.width += oT; cs.valid += oT;
    wm_rollout_out co = dout;
    co.overlap += oW; co.offroad += oW; co.offroad_dist += oW; co.log_div += oW;
    co.any_overlap += oA; co.any_offroad += oA; co.ade += oA;
    WM_CUDA(wm_launch_reset(h, cl, cs, h->cfg.history, s4));
    if (fused) {
      WM_CUDA(wm_launch_rollout_fused(h, cl, cs, t0, n_steps, d_act + oW * C, d_av + oW, co, b0, s4));
    } else {
      // stepwise / brute-force modes: one chunk = the whole batch, through the graph path
      WM_CUDA(cudaStreamSynchronize(s4));
      if ((rc = wm_rollout(h, &dl, &ds, t0, n_steps, d_act, d_av, &dout, s4)) != WM_OK) return rc;
    }
    WM_CUDA(cudaEventRecord(h->ev_done[c], s4));
    WM_CUDA(cudaStreamWaitEvent(s3, h->ev_done[c], 0));
    D2H(oh->overlap ? oh->overlap + oW : nullptr, co.overlap, cW); D2H(oh->offroad ? oh->offroad + oW : nullptr, co.offroad, cW);
    D2H(oh->offroad_dist ? oh->offroad_dist + oW : nullptr, co.offroad_dist, cW * 4);
    D2H(oh->log_div ? oh->log_div + oW : nullptr, co.log_div, cW * 4);
    D2H(oh->any_overlap ? oh->any_overlap + oA : nullptr, co.any_overlap, cA);
    D2H(oh->any_offroad ? oh->any_offroad + oA : nullptr, co.any_offroad, cA);
    D2H(oh->ade ? oh->ade + oA : nullptr, co.ade, cA * 4);
    if (sim_host) {
      D2H(sim_host->x + oT, cs.x, cT * 4); D2H(sim_host->y + oT, cs.y, cT * 4); D2H(sim_host->yaw + oT, cs.yaw, cT * 4);
      D2H(sim_host->vel_x + oT, cs.vel_x, cT * 4); D2H(sim_host->vel_y + oT, cs.vel_y, cT * 4);
      D2H(sim_host->length + oT, cs.length, cT * 4); D2H(sim_host->width + oT, cs.width, cT * 4); D2H(sim_host->valid + oT, cs.valid, cT);
    }
  }
#undef H2D
#undef D2H
  WM_CUDA(cudaStreamSynchronize(s3));
  WM_CUDA(cudaStreamSynchronize(s4));
  WM_CUDA(cudaStreamSynchronize(s2));
  WM_CUDA(cudaStreamSynchronize(s));
  return WM_OK;
}

