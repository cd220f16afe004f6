// Internal declarations of the wm_* library (sm_100a only). Not part of the public ABI.
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "../../include/wm.h"

#if defined(__CUDA_ARCH__) && (__CUDA_ARCH__ < 1000)
#error "this library is written for sm_100a (B200) only"
#endif

// ---------------------------------------------------------------------------------------
// Layout constants of the prepared road-edge segments.
// A tile holds 512 segments = 32 lanes x 16 consecutive segments ("run") per lane, stored so
// that one LDS.128 per lane fetches the same component of two consecutive segments:
//   float4 index inside a tile = (it*3 + c)*32 + lane,  it = (s%16)/2,  lane = (s%512)/16
//   c = 0: {p0x[lo], p0x[hi], p0y[lo], p0y[hi]}   lo/hi = segments 2*it, 2*it+1 of the run
//   c = 1: {ex[lo],  ex[hi],  ey[lo],  ey[hi]}    e = p1 - p0
//   c = 2: {gx[lo],  gx[hi],  gy[lo],  gy[hi]}    g = e / (e.e)   (0 for zero-length)
// ---------------------------------------------------------------------------------------
constexpr int WM_TILE_SEGS = 512;
constexpr int WM_RUN = 16;                 // consecutive segments owned by one lane
constexpr int WM_TILE_F4 = 8 * 3 * 32;     // float4 per tile
constexpr int WM_TILE_BYTES = WM_TILE_F4 * 16;   // 12288
constexpr float WM_FAR = 1.0e18f;          // sentinel coordinate of padding segments

// Exact grid search (wm_grid.cuh): road-edge segments in ascending source order as 32-byte
// records (and two by two as 48-byte PAIR records), bounding boxes per chunk of WM_CHUNK records,
// and TWO nested grids of square cells per scenario: a fine inner grid (<= WM_GRID_NG_IN^2 cells,
// side >= 2 m) over the segments' bounding box plus a small margin, where nearly all queries land,
// and a coarse outer grid (<= WM_GRID_NG_OUT^2 cells, side >= 4 x the inner side) over the wide
// margin that agents reach when they drive off the map.  The inner grid is aligned with the outer
// one: an outer cell under it splits into 2 x 2 MID cells (a level that only wm_prepare uses) and each of
// those into 2 x 2 inner cells; a mid / inner cell takes its candidates from its PARENT's list instead of
// from all segments (wm_grid.cu).  A cell has an 8-byte header of up to three runs of pair records, 21 bits
// each (first pair << 5 | pairs, 1 <= pairs <= 31) in bits 0-20, 21-41, 42-62:
//   bit 63 clear            1-3 runs (unused fields zero); zero = nothing to walk
//   bit 63 set              two runs, and bits 42-62 = offset into the pool: pool[offset] = n further
//                           runs (n <= WM_GRID_MAXRUN - 2), pool[offset + 1 ...] = those runs
//   all ones                too many candidates: search all chunks
// Headers are stored in tiles of 2 x 2 cells (one 32-byte sector = 4 m x 4 m at the default
// inner cell side), tile-row-major: the four corners of a box and its next steps share sectors.
// The outer grid's headers follow the inner grid's at cell offset WmGrid::obase, the mid grid's at mbase.
constexpr int WM_CHUNK = 32;
constexpr int WM_GRID_NG_IN = 160;
constexpr int WM_GRID_NG_OUT = 64;
constexpr int WM_GRID_CELLS = WM_GRID_NG_IN * WM_GRID_NG_IN + WM_GRID_NG_OUT * WM_GRID_NG_OUT + (WM_GRID_NG_IN / 2) * (WM_GRID_NG_IN / 2);
constexpr int WM_POOL_CAP = WM_GRID_CELLS;       // words of overflow runs per scenario
constexpr int WM_GRID_MAXRUN = 16;               // runs per cell before the cell falls back to the full search
constexpr int WM_MAX_RECORDS = 131072;           // pair indices are 16 bits
struct WmGrid {
  float x0, y0, inv_h, h; int nx, ny, nseg, obase;        // inner grid; obase = first outer header
  float ox0, oy0, oinv_h, oh; int onx, ony, icx0, icy0;   // outer grid; the inner grid starts at its cell (icx0, icy0)
  int mbase, pad0, pad1, pad2;                            // mid grid (build only): (nx / 2) x (ny / 2) cells of side 2 h at (x0, y0); first header
};
// Prepared roadgraph points for the top-k observation (wm_observe.cu): the valid points of a
// scenario bucketed into a uniform grid of at most WM_PT_NG x WM_PT_NG cells (side >= 4 m) over
// their bounding box, stored cell by cell in row-major cell order: (x, y), original index, and the
// start of every cell.  A row of consecutive cells is one contiguous run of points.
constexpr int WM_PT_NG = 64;
constexpr int WM_PT_CELLS = WM_PT_NG * WM_PT_NG;
struct WmPtGrid { float x0, y0, inv_h, h; int nx, ny, nvalid, pad; };

constexpr int WM_MAX_B = 65535;            // scenarios per call: several launchers put the scenario in gridDim.y
constexpr int WM_GRAPH_KEY_WORDS = 40;     // cache key of the captured rollout graph (wm_api.cu)
constexpr int WM_HOST_CHUNKS = 16;          // scenario chunks of the pipelined host path

struct wm_handle {
  wm_config cfg;
  int device;
  int num_sms;
  int64_t launches;
  // prepared static data (wm_prepare)
  int32_t prep_B, prep_R;
  int32_t seg_tiles;        // tiles per scenario in `edges`
  int32_t seg_max;          // max_b n_seg[b]
  int32_t seg_ready;        // the record arrays below are allocated for prep_B x seg_tiles: wm_prepare has run ("is prepared" marker)
  int32_t* n_seg;           // [B]
  float4* edges;            // [B][seg_tiles][WM_TILE_F4]  WM_OFFROAD_BRUTE_FORCE only (NULL otherwise)
  float2* sign_dir;         // [B][seg_tiles*512]  sign direction (e, or stored dir if e == 0); WM_OFFROAD_BRUTE_FORCE only
  int32_t* seg_src;         // [B][seg_tiles*512]  first-point index of each stored segment (-1: padding)
  float4* segrec;           // [B][seg_tiles*512][2] {p0x,p0y,ex,ey} {gx,gy,sx,sy}, ascending source order
  float4* segfin;           // [B][seg_tiles*512] {p0x, p0y, sx, sy}: what the sign of the winner needs
  float4* segpair;          // [B][3][seg_tiles*256] the same records two by two, component-wise, in three planes (wm_grid.cuh)
  float4* seglk;            // [B][seg_tiles*256][2] per pair record, for the cell build only (wm_grid.cu; kept between
                            //   wm_prepare calls so that re-preparing a batch of the same size calls no cudaMalloc): what the
                            //   neighbour rules P / N need - {fx, fx', fy, fy'} {aP, aP', aN, aN'}, f = e of the NEXT record
                            //   of the same polyline (0 if none), aP / aN = |ex| + |ey| when the rule can apply, +inf otherwise
  float4* chunks;           // [B][seg_tiles*16]   bounding box of each chunk of 32 records
  WmGrid* gridp;            // [B]
  uint2* cells;             // [B][WM_GRID_CELLS]  cell headers, 2 x 2 tiles
  uint32_t* pool;           // [B][WM_POOL_CAP]    overflow runs
  int32_t* pool_cnt;        // [B]
  float2* pt_xy;            // [B][R] valid points in cell order (wm_observe.cu)
  int32_t* pt_idx;          // [B][R] their roadgraph indices
  int32_t* pt_start;        // [B][WM_PT_CELLS + 1] first point of every cell; [ny * nx] = number of valid points
  WmPtGrid* pt_grid;        // [B]
  // rollout graph cache; streams and events of the pipelined host path (wm_rollout_host)
  cudaStream_t cap_stream, roll_stream, d2h_stream;
  cudaEvent_t ev_up[WM_HOST_CHUNKS], ev_prep[WM_HOST_CHUNKS], ev_done[WM_HOST_CHUNKS];
  cudaGraph_t graph;
  cudaGraphExec_t graph_exec;
  int64_t graph_kernels;
  uint64_t graph_key[WM_GRAPH_KEY_WORDS];
  // scratch for rollouts / host staging
  void* scratch; size_t scratch_bytes;
  void* stage[16]; size_t stage_bytes[16];
  unsigned long long* cull_stats;   // device [16]: [0..3] pairs evaluated, brute-force pairs, slow-path corners, corners;
                                    //   [8..13] scratch of wm_grid_stats
  int stats_on;                     // counters are collected only when enabled (wm_offroad_stats_enable)
};

extern thread_local int g_wm_last_cuda_error;

#define WM_CUDA(call)                                   \
  do {                                                  \
    cudaError_t e__ = (call);                           \
    if (e__ != cudaSuccess) {                           \
      g_wm_last_cuda_error = (int)e__;                  \
      return WM_ERR_CUDA;                               \
    }                                                   \
  } while (0)

// A time row of a trajectory: pointers to row t of scenario 0, batch stride in elements.
struct wm_row {
  const float *x, *y, *yaw, *vel_x, *vel_y, *length, *width;
  const uint8_t* valid;
  int64_t stride_b;
};
struct wm_row_mut {
  float *x, *y, *yaw, *vel_x, *vel_y, *length, *width;
  uint8_t* valid;
  int64_t stride_b;
};
static inline wm_row wm_make_row(const wm_traj& tr, int t) {
  const int64_t o = (int64_t)t * tr.A;
  return wm_row{tr.x + o, tr.y + o, tr.yaw + o, tr.vel_x + o, tr.vel_y + o, tr.length + o,
                tr.width + o, tr.valid + o, (int64_t)tr.T * tr.A};
}
static inline wm_row_mut wm_make_row_mut(const wm_traj& tr, int t) {
  const int64_t o = (int64_t)t * tr.A;
  return wm_row_mut{tr.x + o, tr.y + o, tr.yaw + o, tr.vel_x + o, tr.vel_y + o, tr.length + o,
                    tr.width + o, tr.valid + o, (int64_t)tr.T * tr.A};
}

// ---- launchers (each enqueues on `s`, returns the launch error, bumps h->launches) ----
cudaError_t wm_launch_reset(wm_handle* h, const wm_traj& log, const wm_traj& sim, int history, cudaStream_t s);
// dynamics row t -> t+1; optional fused log divergence of row t+1 (ld_dist may be NULL)
cudaError_t wm_launch_step(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t,
                           const float* action, int64_t act_stride_b, const uint8_t* av,
                           int64_t av_stride_b, float* ld_dist, uint8_t* ld_valid,
                           int64_t ld_stride_b, cudaStream_t s);
cudaError_t wm_launch_logdiv(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t, float* dist,
                             uint8_t* valid, int64_t stride_b, cudaStream_t s);
cudaError_t wm_launch_expert(wm_handle* h, const wm_traj& tr, int t, int n_steps, float* action, uint8_t* valid, cudaStream_t s);
cudaError_t wm_launch_kinematic(wm_handle* h, const wm_traj& tr, int t, int n_steps, float* accel, float* curvature,
                                uint8_t* flag, cudaStream_t s);
cudaError_t wm_launch_rollout_vjp(wm_handle* h, const wm_traj& sim, int t0, int n_steps, const float* actions, const uint8_t* av,
                                  const float* g_rows, float* g_actions, float* g_state0, cudaStream_t s);
cudaError_t wm_launch_discretize(wm_handle* h, const wm_action_grid& g, int C, int64_t N, int A, const float* action,
                                 const uint8_t* valid, int32_t* index, float* dequant, cudaStream_t s);
cudaError_t wm_launch_from_index(wm_handle* h, const wm_action_grid& g, int C, int64_t N, int A, const int32_t* index, float* action,
                                 cudaStream_t s);
cudaError_t wm_launch_ffma_peak(wm_handle* h, int packed, int ctas, int iters, float* sink, cudaStream_t s);
cudaError_t wm_launch_route_progress(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t, const wm_paths& pa, float* ratio,
                                     uint8_t* valid, cudaStream_t s);
cudaError_t wm_launch_offroute(wm_handle* h, const wm_traj& sim, int t, const wm_paths& on, const wm_paths* off, float max_dist,
                               float margin, float* dist_on, uint8_t* flag, cudaStream_t s);
cudaError_t wm_launch_idm_step(wm_handle* h, const wm_traj& sim, int t, const wm_paths& pa, const uint8_t* idm_valid,
                               const wm_idm_params& prm, float* accel, int32_t* lead, cudaStream_t s);
cudaError_t wm_launch_overlap(wm_handle* h, const wm_traj& sim, int t, uint32_t* pair_bits,
                              uint8_t* flag, int64_t flag_stride_b, cudaStream_t s);
cudaError_t wm_launch_offroad(wm_handle* h, const wm_traj& sim, int t, float* sd, int64_t sd_stride_b,
                              float* corner, uint8_t* flag, int64_t flag_stride_b, cudaStream_t s);
cudaError_t wm_launch_offroad_grid(wm_handle* h, const wm_traj& sim, int t, float* sd, int64_t sd_stride_b,
                                     float* corner, uint8_t* flag, int64_t flag_stride_b, cudaStream_t s);
cudaError_t wm_launch_aggregate(wm_handle* h, int B, int A, int n_steps, const wm_rollout_out& out,
                                const uint8_t* ld_valid_rows, cudaStream_t s);
cudaError_t wm_launch_build_grid(wm_handle* h, int b0, int B, cudaStream_t s);   // scenarios [b0, b0 + B)
// log / sim / actions / out are views of scenarios [b0, b0 + sim.B) of the prepared batch
cudaError_t wm_launch_rollout_fused(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                    const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                    int b0, cudaStream_t s);
// the same two launches with events: ev[0] before the dynamics kernel, ev[1] between, ev[2] after the metrics kernel
cudaError_t wm_launch_rollout_fused_timed(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                          const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                          cudaEvent_t* ev, cudaStream_t s);
int wm_prepare_impl(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, cudaStream_t s);
int wm_prepare_count(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, cudaStream_t s);   // needs type, id, valid; syncs s
int wm_prepare_build(wm_handle* h, const wm_roadgraph* rg, int b0, int nb, cudaStream_t s);            // scenarios [b0, b0 + nb), no sync
cudaError_t wm_launch_grid_cell_stats(wm_handle* h, unsigned long long* out6, cudaStream_t s);   // out6: device, zeroed by the caller
void wm_prepare_free(wm_handle* h);
void wm_drop_graph(wm_handle* h);
cudaError_t wm_launch_observe_hist(wm_handle* h, const wm_traj& sim, int t, float* hist, uint8_t* hist_valid, cudaStream_t s);
cudaError_t wm_launch_point_grid(wm_handle* h, const wm_roadgraph& rg, int b0, int nb, cudaStream_t s);   // scenarios [b0, b0 + nb)
cudaError_t wm_launch_observe_topk(wm_handle* h, const wm_traj& sim, const wm_roadgraph& rg, int t,
                                   int32_t* rg_index, float* rg_feat, int32_t* rg_type, cudaStream_t s);

#ifdef __CUDACC__
// ---------------------------------------------------------------------------------------
// Device helpers: packed fp32x2 arithmetic (FFMA2/FADD2/FMUL2 on sm_100a), 3-input min,
// mbarrier + 1-D bulk TMA (cp.async.bulk -> UBLKCP).
// ---------------------------------------------------------------------------------------
typedef unsigned long long wm_u64;
__device__ __forceinline__ wm_u64 pk2(float lo, float hi) { wm_u64 r; asm("mov.b64 %0, {%1,%2};" : "=l"(r) : "f"(lo), "f"(hi)); return r; }
__device__ __forceinline__ void upk2(wm_u64 v, float& lo, float& hi) { asm("mov.b64 {%0,%1}, %2;" : "=f"(lo), "=f"(hi) : "l"(v)); }
__device__ __forceinline__ wm_u64 fma2(wm_u64 a, wm_u64 b, wm_u64 c) { wm_u64 d; asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(d) : "l"(a), "l"(b), "l"(c)); return d; }
__device__ __forceinline__ wm_u64 add2(wm_u64 a, wm_u64 b) { wm_u64 d; asm("add.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ wm_u64 sub2(wm_u64 a, wm_u64 b) { wm_u64 d; asm("sub.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ wm_u64 mul2(wm_u64 a, wm_u64 b) { wm_u64 d; asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(d) : "l"(a), "l"(b)); return d; }
__device__ __forceinline__ float min3f(float a, float b, float c) { float d; asm("min.f32 %0, %1, %2, %3;" : "=f"(d) : "f"(a), "f"(b), "f"(c)); return d; }

// corner offsets of a box: a = front-left, b = front-right; corners 0..3 = c+a, c+b, c-a, c-b
// (D30).  Explicit round-to-nearest ops so that every kernel derives bit-identical offsets.
__device__ __forceinline__ void wm_box_offsets_h(float sn, float cs, float hl, float hw, float& ax, float& ay, float& bx,
                                                 float& by) {
  const float hfx = __fmul_rn(hl, cs), hfy = __fmul_rn(hl, sn), hsx = -__fmul_rn(hw, sn), hsy = __fmul_rn(hw, cs);
  ax = __fadd_rn(hfx, hsx); ay = __fadd_rn(hfy, hsy);
  bx = __fsub_rn(hfx, hsx); by = __fsub_rn(hfy, hsy);
}
__device__ __forceinline__ void wm_box_offsets_sc(float sn, float cs, float length, float width, float& ax, float& ay,
                                                  float& bx, float& by) {
  wm_box_offsets_h(sn, cs, 0.5f * length, 0.5f * width, ax, ay, bx, by);
}
__device__ __forceinline__ void wm_box_offsets(float yaw, float length, float width, float& ax, float& ay, float& bx,
                                               float& by) {
  float sn, cs;
  sincosf(yaw, &sn, &cs);
  wm_box_offsets_sc(sn, cs, length, width, ax, ay, bx, by);
}

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void mbar_fence_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n\t.reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t}" ::"r"(smem_u32(bar)), "r"(parity) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// 1-D bulk copy global -> shared, completion counted in bytes on `bar`. bytes % 16 == 0.
__device__ __forceinline__ void tma_load_1d(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(smem_u32(dst_smem)),
               "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)) : "memory");
}
// bulk prefetch of [p, p + bytes) into L2 (bytes % 16 == 0, p 16-byte aligned); fire and forget
__device__ __forceinline__ void l2_prefetch(const void* p, uint32_t bytes) {
  asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(p), "r"(bytes) : "memory");
}
#endif
