// a4 off-road metric, PAPER.md L100 (+ L176: "the Off-Road metric needs to find nearby
// roadgraph points, which is a slow operation" — this kernel IS the cost of the step).
//
// wm_prepare: compacts road-edge segments once per scenario into 512-segment tiles laid out
// for conflict-free LDS.128 and packed fp32x2 arithmetic (wm_internal.cuh).
//
// k_offroad: one CTA per scenario.  The scenario's segment tiles are streamed into shared
// memory by 1-D bulk TMA (cp.async.bulk, mbarrier completion) into two buffers; lanes own
// SEGMENTS (a run of 16 consecutive ones per tile), a warp owns a "unit" of 2 valid agents
// = 8 box corners held in registers, and evaluates 2 segments x 8 corners per iteration
// with FFMA2/FADD2/FMUL2 (two segments packed per instruction):
//     w = (c - p0) + off_k;  t = sat(w.g);  r = w - t e;  d2 = r.r          (8.5 FP32 lane-ops)
//     min tracked per (lane, corner) with one 3-input FMNMX per packed pair
// The argmin is tracked at run granularity (tile, lane); at the end the winning run of each
// corner (16 segments) is re-scanned to get the exact segment (lowest index on ties, D17), the
// sign from the oriented edge (D16) and the signed distance.  Valid agents are compacted first,
// so invalid slots cost nothing.  Bound: FP32 pipe (see DESIGN.md roofline).
#include <float.h>
#include <stdlib.h>

#include "wm_internal.cuh"

// ======================================================================================
// wm_prepare kernels
// ======================================================================================
struct RgView {
  const float *x, *y, *dir_x, *dir_y;
  const int32_t *type, *id;
  const uint8_t* valid;
  int R;
};

__device__ __forceinline__ bool rg_is_edge(const RgView& g, int64_t o, int i) {
  return g.valid[o + i] != 0 && g.type[o + i] == WM_TYPE_ROAD_EDGE;
}
__device__ __forceinline__ bool rg_starts(const RgView& g, int64_t o, int i) {
  return i + 1 < g.R && rg_is_edge(g, o, i) && rg_is_edge(g, o, i + 1) && g.id[o + i] == g.id[o + i + 1];
}
// point i contributes a record: a segment (i, i+1), or an isolated zero-length segment (D16)
__device__ __forceinline__ bool rg_record(const RgView& g, int64_t o, int i, bool* is_seg) {
  if (i >= g.R) { *is_seg = false; return false; }
  const bool s = rg_starts(g, o, i);
  *is_seg = s;
  if (s) return true;
  return rg_is_edge(g, o, i) && !(i > 0 && rg_starts(g, o, i - 1));
}

__global__ void __launch_bounds__(1024) k_count_segments(RgView g, int32_t* n_seg) {
  __shared__ int s_cnt;
  if (threadIdx.x == 0) s_cnt = 0;
  __syncthreads();
  const int64_t o = (int64_t)blockIdx.x * g.R;
  int c = 0;
  for (int i = threadIdx.x; i < g.R; i += blockDim.x) { bool sg; c += rg_record(g, o, i, &sg) ? 1 : 0; }
  atomicAdd(&s_cnt, c);
  __syncthreads();
  if (threadIdx.x == 0) n_seg[blockIdx.x] = s_cnt;
}

// ---------------------------------------------------------------------------------------
// Segment order = ascending first-point index (order-preserving compaction), so that "lower
// stored index" IS the tie rule D17 everywhere, and polyline pieces stay contiguous (the grid
// cells of wm_grid.cu hold runs of consecutive records).  k_order_segments writes seg_src.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(1024) k_order_segments(RgView g, int cap, int32_t* seg_src) {
  __shared__ int s_w[32];
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t o = (int64_t)b * g.R;
  int32_t* out = seg_src + (int64_t)b * cap;
  // a thread owns a contiguous stretch of points: count, one block scan, write (two barriers in all)
  const int per = (g.R + 1023) / 1024, i0 = tid * per, i1 = min(g.R, i0 + per);
  int c = 0;
  bool sg;
  for (int i = i0; i < i1; ++i) c += rg_record(g, o, i, &sg) ? 1 : 0;
  int inc = c;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
  if (lane == 31) s_w[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int v = s_w[lane], w = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, w, d); if (lane >= d) w += u; }
    s_w[lane] = w - v;
  }
  __syncthreads();
  int pos = s_w[warp] + inc - c;
  for (int i = i0; i < i1; ++i) if (rg_record(g, o, i, &sg)) out[pos++] = i;
}

// position of stored segment s inside its tile: lane = (s%512)/16, it = (s%16)/2, half = s&1 (wm_internal.cuh)
__device__ __forceinline__ void store_segment(float* tile_base, float2* sign_dir, int s, float p0x, float p0y,
                                              float ex, float ey, float gx, float gy, float sx, float sy) {
  const int tau = s / WM_TILE_SEGS, r = s % WM_TILE_SEGS;
  const int it = (r & 15) >> 1, lane = r >> 4, half = r & 1;
  float* t = tile_base + (int64_t)tau * (WM_TILE_F4 * 4);
  float* q0 = t + ((it * 3 + 0) * 32 + lane) * 4;
  float* q1 = t + ((it * 3 + 1) * 32 + lane) * 4;
  float* q2 = t + ((it * 3 + 2) * 32 + lane) * 4;
  q0[half] = p0x; q0[2 + half] = p0y;
  q1[half] = ex;  q1[2 + half] = ey;
  q2[half] = gx;  q2[2 + half] = gy;
  sign_dir[s] = make_float2(sx, sy);
}

// One warp per group of 64 stored segments: writes the tile records (brute-force layout), the
// 32-byte records of the grid search and their pair form, and the bounding box of each chunk of 32.
__global__ void __launch_bounds__(256) k_fill_segments(RgView g, int seg_tiles, const int32_t* n_seg, float4* edges,
                                                       float2* sign_dir, int32_t* seg_src, float4* segrec, float4* segpair, float4* seglk, float4* segfin, float4* chunks, int tiles_on) {
  const int b = blockIdx.y, lane = threadIdx.x & 31;
  const int grp = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
  const int ngrp = seg_tiles * (WM_TILE_SEGS / 64);
  if (grp >= ngrp) return;
  const int64_t o = (int64_t)b * g.R;
  const int cap = seg_tiles * WM_TILE_SEGS, n = n_seg[b];
  float* tile_base = tiles_on ? (float*)(edges + (int64_t)b * seg_tiles * WM_TILE_F4) : nullptr;   // NULL outside the brute-force mode
  float2* sd = tiles_on ? sign_dir + (int64_t)b * cap : nullptr;
  int32_t* src = seg_src + (int64_t)b * cap;
  float x0 = 3.0e38f, y0 = 3.0e38f, x1 = -3.0e38f, y1 = -3.0e38f;
  float ax[2], ay[2], bx[2], by[2];
  float pp[2][6];                                 // p0x, p0y, -ex, -ey, gx, gy of the lane's two segments
  float lk[2][4];                                 // fx, fy, aP, aN (wm_internal.cuh: seglk)
  const float PINF = __int_as_float(0x7f800000);
  bool real[2];
#pragma unroll
  for (int hf = 0; hf < 2; ++hf) {
    const int s = grp * 64 + lane * 2 + hf;
    real[hf] = s < n;
    if (real[hf]) {
      const int i = src[s];
      const bool is_seg = rg_starts(g, o, i);
      const float p0x = g.x[o + i], p0y = g.y[o + i];
      float ex = 0.f, ey = 0.f;
      if (is_seg) { ex = g.x[o + i + 1] - p0x; ey = g.y[o + i + 1] - p0y; }
      const float ee = fmaf(ex, ex, ey * ey);
      float gx = 0.f, gy = 0.f, sx, sy;
      if (ee > 0.f) { gx = ex / ee; gy = ey / ee; sx = ex; sy = ey; }
      else { ex = 0.f; ey = 0.f; sx = g.dir_x[o + i]; sy = g.dir_y[o + i]; }     // D16 / D29
      if (tiles_on) store_segment(tile_base, sd, s, p0x, p0y, ex, ey, gx, gy, sx, sy);     // the brute-force kernel's layout: only that mode reads it
      float4* rec = segrec + ((int64_t)b * cap + s) * 2;
      rec[0] = make_float4(p0x, p0y, ex, ey);
      rec[1] = make_float4(gx, gy, sx, sy);
      segfin[(int64_t)b * cap + s] = make_float4(p0x, p0y, sx, sy);
      pp[hf][0] = p0x; pp[hf][1] = p0y; pp[hf][2] = -ex; pp[hf][3] = -ey; pp[hf][4] = gx; pp[hf][5] = gy;
      // neighbour rules of the cell build (wm_grid.cu): P needs the previous record to be the real segment
      // that ends in p0, N the next record to be the real segment that starts in p1
      lk[hf][0] = 0.f; lk[hf][1] = 0.f; lk[hf][2] = PINF; lk[hf][3] = PINF;
      if (ee > 0.f) {
        const float ae = fabsf(ex) + fabsf(ey);
        if (i > 0 && rg_starts(g, o, i - 1)) {
          const float qx = p0x - g.x[o + i - 1], qy = p0y - g.y[o + i - 1];
          if (fmaf(qx, qx, qy * qy) > 0.f) lk[hf][2] = ae;
        }
        if (rg_starts(g, o, i + 1)) {
          const float fx = g.x[o + i + 2] - g.x[o + i + 1], fy = g.y[o + i + 2] - g.y[o + i + 1];
          if (fmaf(fx, fx, fy * fy) > 0.f) { lk[hf][0] = fx; lk[hf][1] = fy; lk[hf][3] = ae; }
        }
      }
      ax[hf] = p0x; ay[hf] = p0y; bx[hf] = p0x + ex; by[hf] = p0y + ey;
      x0 = fminf(x0, fminf(ax[hf], bx[hf])); x1 = fmaxf(x1, fmaxf(ax[hf], bx[hf]));
      y0 = fminf(y0, fminf(ay[hf], by[hf])); y1 = fmaxf(y1, fmaxf(ay[hf], by[hf]));
    } else {                                      // padding: far away, never wins against a real segment
      if (tiles_on) store_segment(tile_base, sd, s, WM_FAR, WM_FAR, 0.f, 0.f, 0.f, 0.f, 1.f, 0.f);
      float4* rec = segrec + ((int64_t)b * cap + s) * 2;
      rec[0] = make_float4(WM_FAR, WM_FAR, 0.f, 0.f);
      rec[1] = make_float4(0.f, 0.f, 1.f, 0.f);
      segfin[(int64_t)b * cap + s] = make_float4(WM_FAR, WM_FAR, 1.f, 0.f);
      src[s] = -1;
      pp[hf][0] = WM_FAR; pp[hf][1] = WM_FAR; pp[hf][2] = 0.f; pp[hf][3] = 0.f; pp[hf][4] = 0.f; pp[hf][5] = 0.f;
      lk[hf][0] = 0.f; lk[hf][1] = 0.f; lk[hf][2] = PINF; lk[hf][3] = PINF;
    }
  }
  {                                               // the lane's two records as one pair record
    float4* pr = segpair + (int64_t)b * (cap / 2) * 3 + grp * 32 + lane;       // three planes of cap / 2 parts (wm_grid.cuh)
    pr[0] = make_float4(pp[0][0], pp[1][0], pp[0][1], pp[1][1]);
    pr[cap / 2] = make_float4(pp[0][2], pp[1][2], pp[0][3], pp[1][3]);
    pr[2 * (cap / 2)] = make_float4(pp[0][4], pp[1][4], pp[0][5], pp[1][5]);
    float4* pl = seglk + ((int64_t)b * (cap / 2) + grp * 32 + lane) * 2;
    pl[0] = make_float4(lk[0][0], lk[1][0], lk[0][1], lk[1][1]);
    pl[1] = make_float4(lk[0][2], lk[1][2], lk[0][3], lk[1][3]);
  }
#pragma unroll
  for (int d = 8; d > 0; d >>= 1) {             // 16 lanes = one chunk of 32 records
    x0 = fminf(x0, __shfl_xor_sync(0xffffffffu, x0, d)); y0 = fminf(y0, __shfl_xor_sync(0xffffffffu, y0, d));
    x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, d)); y1 = fmaxf(y1, __shfl_xor_sync(0xffffffffu, y1, d));
  }
  // axis-aligned bounding box {x0, y0, x1, y1} of the chunk's segments (min/max of the float32
  // endpoints; p1 = p0 + e may round by an ulp, covered by the slack of the cull tests)
  if ((lane & 15) == 0) {
    const bool any = x1 >= x0;
    chunks[(int64_t)b * ngrp * 2 + grp * 2 + (lane >> 4)] = any ? make_float4(x0, y0, x1, y1) : make_float4(WM_FAR, WM_FAR, WM_FAR, WM_FAR);
  }
}

void wm_prepare_free(wm_handle* h) {
  cudaFree(h->n_seg); cudaFree(h->edges); cudaFree(h->sign_dir); cudaFree(h->seg_src); cudaFree(h->pt_xy); cudaFree(h->pt_idx); cudaFree(h->pt_start); cudaFree(h->pt_grid);
  cudaFree(h->segrec); cudaFree(h->segpair); cudaFree(h->seglk); cudaFree(h->segfin); cudaFree(h->chunks); cudaFree(h->gridp); cudaFree(h->cells); cudaFree(h->pool); cudaFree(h->pool_cnt);
  h->n_seg = nullptr; h->edges = nullptr; h->sign_dir = nullptr; h->seg_src = nullptr; h->pt_xy = nullptr; h->pt_idx = nullptr; h->pt_start = nullptr; h->pt_grid = nullptr;
  h->segrec = nullptr; h->segpair = nullptr; h->seglk = nullptr; h->segfin = nullptr; h->chunks = nullptr; h->gridp = nullptr; h->cells = nullptr; h->pool = nullptr; h->pool_cnt = nullptr;
  h->prep_B = 0; h->prep_R = 0; h->seg_tiles = 0; h->seg_max = 0; h->seg_ready = 0;
}

// Step 1 of wm_prepare: per-scenario record counts (needs type, id, valid only), the capacity they
// call for, and the buffers.  Synchronises `s` once (the counts come back to the host).
int wm_prepare_count(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, cudaStream_t s) {
  const int B = rg->B, R = rg->R;
  RgView g{rg->x, rg->y, rg->dir_x, rg->dir_y, rg->type, rg->id, rg->valid, R};
  // Buffers are reused when the shapes fit, so device pointers (and a captured rollout graph)
  // stay valid across scenarios of the same shape.
  if (h->prep_B != B || h->prep_R != R) {
    wm_drop_graph(h);
    wm_prepare_free(h);
    WM_CUDA(cudaMalloc(&h->n_seg, (size_t)B * sizeof(int32_t)));
    WM_CUDA(cudaMalloc(&h->pt_xy, (size_t)B * R * sizeof(float2)));
    WM_CUDA(cudaMalloc(&h->pt_idx, (size_t)B * R * sizeof(int32_t)));
    WM_CUDA(cudaMalloc(&h->pt_start, (size_t)B * (WM_PT_CELLS + 1) * sizeof(int32_t)));
    WM_CUDA(cudaMalloc(&h->pt_grid, (size_t)B * sizeof(WmPtGrid)));
    WM_CUDA(cudaMalloc(&h->gridp, (size_t)B * sizeof(WmGrid)));
    WM_CUDA(cudaMalloc(&h->cells, (size_t)B * WM_GRID_CELLS * sizeof(uint2)));
    WM_CUDA(cudaMalloc(&h->pool, (size_t)B * WM_POOL_CAP * sizeof(uint32_t)));
    WM_CUDA(cudaMalloc(&h->pool_cnt, (size_t)B * sizeof(int32_t)));
    h->prep_B = B; h->prep_R = R;
  }
  k_count_segments<<<B, 1024, 0, s>>>(g, h->n_seg);
  h->launches++;
  WM_CUDA(cudaGetLastError());
  int32_t* host = (int32_t*)malloc((size_t)B * sizeof(int32_t));
  if (!host) return WM_ERR_ARG;
  cudaError_t e = cudaMemcpyAsync(host, h->n_seg, (size_t)B * sizeof(int32_t), cudaMemcpyDeviceToHost, s);
  if (e == cudaSuccess) e = cudaStreamSynchronize(s);
  int mx = 0;
  if (e == cudaSuccess) for (int b = 0; b < B; ++b) mx = host[b] > mx ? host[b] : mx;
  free(host);
  WM_CUDA(e);
  if (mx > WM_MAX_RECORDS) return WM_ERR_UNSUPPORTED;      // pair indices of the cell lists are 16 bits
  h->seg_max = mx;
  int tiles = (mx + WM_TILE_SEGS - 1) / WM_TILE_SEGS;
  if (tiles < 1) tiles = 1;
  if (tiles > h->seg_tiles || !h->seg_ready) {   // grow only: seg_tiles is the row stride of the record arrays
    wm_drop_graph(h);
    cudaFree(h->edges); cudaFree(h->sign_dir); cudaFree(h->seg_src); cudaFree(h->segrec); cudaFree(h->segpair); cudaFree(h->seglk); cudaFree(h->segfin); cudaFree(h->chunks);
    h->edges = nullptr; h->sign_dir = nullptr; h->seg_src = nullptr; h->segrec = nullptr; h->segpair = nullptr; h->seglk = nullptr; h->segfin = nullptr; h->chunks = nullptr;
    h->seg_tiles = tiles; h->seg_ready = 0;
    const size_t cap = (size_t)tiles * WM_TILE_SEGS;
    cudaError_t ea = cudaSuccess;
    if (h->cfg.offroad_mode == WM_OFFROAD_BRUTE_FORCE) {     // the tile layout and its sign directions: only k_offroad reads them
      ea = cudaMalloc(&h->edges, (size_t)B * tiles * WM_TILE_BYTES);
      if (ea == cudaSuccess) ea = cudaMalloc(&h->sign_dir, (size_t)B * cap * sizeof(float2));
    }
    if (ea == cudaSuccess) ea = cudaMalloc(&h->seg_src, (size_t)B * cap * sizeof(int32_t));
    if (ea == cudaSuccess) ea = cudaMalloc(&h->segrec, (size_t)B * cap * 2 * sizeof(float4));
    if (ea == cudaSuccess) ea = cudaMalloc(&h->segpair, (size_t)B * (cap / 2) * 3 * sizeof(float4));
    if (ea == cudaSuccess) ea = cudaMalloc(&h->seglk, (size_t)B * (cap / 2) * 2 * sizeof(float4));
    if (ea == cudaSuccess) ea = cudaMalloc(&h->segfin, (size_t)B * cap * sizeof(float4));
    if (ea == cudaSuccess) ea = cudaMalloc(&h->chunks, (size_t)B * (cap / WM_CHUNK) * sizeof(float4));
    if (ea != cudaSuccess) { wm_prepare_free(h); WM_CUDA(ea); }     // out of memory: back to the unprepared state
    h->seg_ready = 1;
  }
  if (n_segments_max) *n_segments_max = mx;
  return WM_OK;
}

// Step 2: the prepared structures of scenarios [b0, b0 + nb) (records, grid, packed points), enqueued
// on `s`; no synchronisation.  rg holds the device pointers of the whole batch.
int wm_prepare_build(wm_handle* h, const wm_roadgraph* rg, int b0, int nb, cudaStream_t s) {
  const int R = rg->R;
  const int64_t o = (int64_t)b0 * R;
  RgView g{rg->x + o, rg->y + o, rg->dir_x + o, rg->dir_y + o, rg->type + o, rg->id + o, rg->valid + o, R};
  const int tiles = h->seg_tiles;
  const int64_t cap = (int64_t)tiles * WM_TILE_SEGS;
  int32_t* seg_src = h->seg_src + b0 * cap;
  k_order_segments<<<nb, 1024, 0, s>>>(g, (int)cap, seg_src);
  h->launches++;
  WM_CUDA(cudaGetLastError());
  {
    const int ngrp = tiles * (WM_TILE_SEGS / 64);
    const bool brute = h->cfg.offroad_mode == WM_OFFROAD_BRUTE_FORCE;   // edges / sign_dir exist in that mode only
    k_fill_segments<<<dim3((ngrp + 7) / 8, nb), 256, 0, s>>>(g, tiles, h->n_seg + b0, brute ? h->edges + (int64_t)b0 * tiles * WM_TILE_F4 : nullptr,
                                                             brute ? h->sign_dir + b0 * cap : nullptr, seg_src, h->segrec + b0 * cap * 2,
                                                             h->segpair + b0 * (cap / 2) * 3, h->seglk + b0 * (cap / 2) * 2, h->segfin + b0 * cap,
                                                             h->chunks + b0 * (cap / WM_CHUNK), brute);
  }
  h->launches++;
  WM_CUDA(cudaGetLastError());
  WM_CUDA(wm_launch_build_grid(h, b0, nb, s));
  WM_CUDA(wm_launch_point_grid(h, *rg, b0, nb, s));
  return WM_OK;
}

int wm_prepare_impl(wm_handle* h, const wm_roadgraph* rg, int32_t* n_segments_max, cudaStream_t s) {
  int rc = wm_prepare_count(h, rg, n_segments_max, s);
  if (rc != WM_OK) return rc;
  if ((rc = wm_prepare_build(h, rg, 0, rg->B, s)) != WM_OK) return rc;
  WM_CUDA(cudaStreamSynchronize(s));
  return WM_OK;
}

// ======================================================================================
// k_offroad
// ======================================================================================
// CTA size is a template parameter: 512 threads x 1 CTA/SM or 256 threads x 2 CTAs/SM

constexpr int OFF_NA = 2;                  // agents per warp unit (8 corners in registers)

struct OffroadParams {
  wm_row row;
  int A;
  const float4* edges; const float2* sign_dir; const int32_t* n_seg; const int32_t* seg_src;
  int seg_tiles;          // tiles per scenario in `edges`
  int tiles_per_buf;      // capacity of one shared-memory buffer, in tiles
  float* sd; int64_t sd_stride_b;
  float* corner;          // [B][4][A] or NULL
  uint8_t* flag; int64_t flag_stride_b;
};

// shared-memory carve-up (dynamic): [bars 16 B][agent SoA 6*Ap floats][aidx Ap ints][keys 4*Ap u64][buffers]
__host__ __device__ inline size_t off_fixed_bytes(int A) {
  const size_t Ap = (size_t)((A + 31) / 32) * 32;
  size_t n = 128 + Ap * 6 * 4 + Ap * 4 + Ap * 4 * 8;
  return (n + 127) / 128 * 128;
}

// distance^2 of one corner to one segment, the arithmetic both the scan and the re-scan use
__device__ __forceinline__ float seg_d2(float wx, float wy, float ex, float ey, float gx, float gy) {
  const float t = __saturatef(fmaf(wy, gy, wx * gx));
  const float rx = fmaf(-t, ex, wx), ry = fmaf(-t, ey, wy);
  return fmaf(ry, ry, rx * rx);
}

template <int OFF_THREADS, int OFF_MINB>
__global__ void __launch_bounds__(OFF_THREADS, OFF_MINB) k_offroad(OffroadParams p) {
  constexpr int OFF_WARPS = OFF_THREADS / 32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int A = p.A, Ap = ((A + 31) / 32) * 32;
  uint64_t* bars = (uint64_t*)smem_raw;                       // [2] full barriers
  int* s_misc = (int*)(smem_raw + 16);                        // [0] nvalid, [1..] scan scratch
  float* s_ag = (float*)(smem_raw + 128);                     // [6][Ap] cx, cy, ax, ay, bx, by (compacted)
  int* s_aidx = (int*)(s_ag + 6 * Ap);                        // [Ap] compact -> agent slot
  wm_u64* s_key = (wm_u64*)(s_aidx + Ap);                     // [4*Ap] (d2 bits << 32) | run id
  float4* s_buf = (float4*)(smem_raw + off_fixed_bytes(A));   // 2 x tiles_per_buf tiles

  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nseg = p.n_seg[b];
  const int nt = (nseg + WM_TILE_SEGS - 1) / WM_TILE_SEGS;    // tiles of this scenario
  const int G = (nt + p.tiles_per_buf - 1) / p.tiles_per_buf; // tile groups
  // group g covers tiles [g*nt/G, (g+1)*nt/G): balanced, each at most tiles_per_buf
  const float4* edges_b = p.edges + (int64_t)b * p.seg_tiles * WM_TILE_F4;

  if (tid == 0) {
    mbar_init(&bars[0], 1);
    mbar_init(&bars[1], 1);
    mbar_fence_init();
  }
  __syncthreads();
  // ---- producer: start the first two groups (overlaps with the agent set-up below) ----
  if (tid == 0) {
    for (int g = 0; g < 2 && g < G; ++g) {
      const int t0 = (g * nt) / G, n = ((g + 1) * nt) / G - t0;
      mbar_expect_tx(&bars[g], (uint32_t)n * WM_TILE_BYTES);
      for (int t = 0; t < n; ++t)
        tma_load_1d(s_buf + ((int64_t)g * p.tiles_per_buf + t) * WM_TILE_F4, edges_b + (int64_t)(t0 + t) * WM_TILE_F4, WM_TILE_BYTES, &bars[g]);
    }
  }

  // ---- agent set-up: order-preserving compaction of valid agents, corner offsets ----
  const int64_t ro = (int64_t)b * p.row.stride_b;
  if (tid == 0) s_misc[0] = 0;
  __syncthreads();
  for (int base = 0; base < Ap; base += OFF_THREADS) {
    const int a = base + tid;
    const bool v = a < A && p.row.valid[ro + a] != 0;
    const uint32_t bal = __ballot_sync(0xffffffffu, v);
    if (lane == 0) s_misc[1 + warp] = __popc(bal);
    __syncthreads();
    int pre = s_misc[0];
    for (int w = 0; w < warp; ++w) pre += s_misc[1 + w];
    if (v) {
      const int ci = pre + __popc(bal & ((1u << lane) - 1u));
      const float x = p.row.x[ro + a], y = p.row.y[ro + a];
      float oax, oay, obx, oby;
      wm_box_offsets(p.row.yaw[ro + a], p.row.length[ro + a], p.row.width[ro + a], oax, oay, obx, oby);
      s_ag[0 * Ap + ci] = x;    s_ag[1 * Ap + ci] = y;
      s_ag[2 * Ap + ci] = oax;  s_ag[3 * Ap + ci] = oay;   // a: front-left offset
      s_ag[4 * Ap + ci] = obx;  s_ag[5 * Ap + ci] = oby;   // b: front-right offset
      s_aidx[ci] = a;
    } else if (a < A) {                                                 // D10: zeros for invalid agents
      p.sd[(int64_t)b * p.sd_stride_b + a] = 0.f;
      p.flag[(int64_t)b * p.flag_stride_b + a] = 0;
      if (p.corner) for (int k = 0; k < 4; ++k) p.corner[((int64_t)b * 4 + k) * A + a] = 0.f;
    }
    __syncthreads();
    if (tid == 0) { int tot = 0; for (int w = 0; w < OFF_WARPS; ++w) tot += s_misc[1 + w]; s_misc[0] += tot; }
    __syncthreads();
  }
  const int nvalid = s_misc[0];
  for (int i = tid; i < 4 * nvalid; i += OFF_THREADS) s_key[i] = ~0ull;
  __syncthreads();

  // ---- scan ----
  const int nunits = (nvalid + OFF_NA - 1) / OFF_NA;
  for (int g = 0; g < G; ++g) {
    const int t0 = (g * nt) / G, ntg = ((g + 1) * nt) / G - t0;
    const int ncells = nunits * ntg;
    const int c_begin = (int)(((long long)warp * ncells) / OFF_WARPS);
    const int c_end = (int)(((long long)(warp + 1) * ncells) / OFF_WARPS);
    // every warp waits, cells or not: no bulk copy may be in flight when the buffers are
    // recycled or the CTA exits
    mbar_wait(&bars[g & 1], (uint32_t)((g >> 1) & 1));
    const float4* buf = s_buf + (int64_t)(g & 1) * p.tiles_per_buf * WM_TILE_F4;

    int cur_u = -1;
    float cx[OFF_NA], cy[OFF_NA], ax[OFF_NA], ay[OFF_NA], bx[OFF_NA], by[OFF_NA];
    float best[OFF_NA * 4];
    int brun[OFF_NA * 4];

    auto flush = [&]() {
      if (cur_u < 0) return;
#pragma unroll
      for (int k = 0; k < OFF_NA * 4; ++k) {
        const int ci = cur_u * OFF_NA + (k >> 2);
        const uint32_t bits = __float_as_uint(best[k]);
        const uint32_t m = __reduce_min_sync(0xffffffffu, bits);
        // a lane holds 16 CONSECUTIVE stored segments of a tile, so (tile, lane) order is index order: exact
        // ties between lanes go to the lower index (D17)
        const uint32_t cand = bits == m ? (uint32_t)brun[k] * 32u + (uint32_t)lane : 0xffffffffu;
        const uint32_t r = __reduce_min_sync(0xffffffffu, cand);
        if (lane == 0 && ci < nvalid) atomicMin(&s_key[ci * 4 + (k & 3)], ((wm_u64)m << 32) | r);
      }
    };

    for (int c = c_begin; c < c_end; ++c) {
      const int u = c / ntg, tl = c - u * ntg;
      if (u != cur_u) {
        flush();
        cur_u = u;
#pragma unroll
        for (int n = 0; n < OFF_NA; ++n) {
          const int ci = min(u * OFF_NA + n, nvalid - 1);    // odd tail: duplicate (result dropped)
          cx[n] = s_ag[0 * Ap + ci]; cy[n] = s_ag[1 * Ap + ci];
          ax[n] = s_ag[2 * Ap + ci]; ay[n] = s_ag[3 * Ap + ci];
          bx[n] = s_ag[4 * Ap + ci]; by[n] = s_ag[5 * Ap + ci];
        }
#pragma unroll
        for (int k = 0; k < OFF_NA * 4; ++k) { best[k] = __int_as_float(0x7f800000); brun[k] = 0; }
      }
      const float4* tp = buf + (int64_t)tl * WM_TILE_F4 + lane;
      float cm[OFF_NA * 4];
#pragma unroll
      for (int it = 0; it < 8; ++it) {
        const float4 P = tp[(it * 3 + 0) * 32], E = tp[(it * 3 + 1) * 32], Gv = tp[(it * 3 + 2) * 32];
        const wm_u64 Px = pk2(P.x, P.y), Py = pk2(P.z, P.w), Ex = pk2(E.x, E.y), Ey = pk2(E.z, E.w), Gx = pk2(Gv.x, Gv.y);
#pragma unroll
        for (int n = 0; n < OFF_NA; ++n) {
          const wm_u64 wcx = sub2(pk2(cx[n], cx[n]), Px), wcy = sub2(pk2(cy[n], cy[n]), Py);
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            wm_u64 wx, wy;
            if (k == 0)      { wx = add2(wcx, pk2(ax[n], ax[n])); wy = add2(wcy, pk2(ay[n], ay[n])); }
            else if (k == 1) { wx = add2(wcx, pk2(bx[n], bx[n])); wy = add2(wcy, pk2(by[n], by[n])); }
            else if (k == 2) { wx = sub2(wcx, pk2(ax[n], ax[n])); wy = sub2(wcy, pk2(ay[n], ay[n])); }
            else             { wx = sub2(wcx, pk2(bx[n], bx[n])); wy = sub2(wcy, pk2(by[n], by[n])); }
            const wm_u64 tm = mul2(wx, Gx);
            float tl0, tl1, wy0, wy1;
            upk2(tm, tl0, tl1); upk2(wy, wy0, wy1);
            const float t0s = __saturatef(fmaf(wy0, Gv.z, tl0)), t1s = __saturatef(fmaf(wy1, Gv.w, tl1));
            const wm_u64 nt2 = pk2(-t0s, -t1s);
            const wm_u64 rx = fma2(nt2, Ex, wx), ry = fma2(nt2, Ey, wy);
            const wm_u64 d2 = fma2(ry, ry, mul2(rx, rx));
            float d0, d1;
            upk2(d2, d0, d1);
            if (it == 0) cm[n * 4 + k] = fminf(d0, d1); else cm[n * 4 + k] = min3f(cm[n * 4 + k], d0, d1);
          }
        }
      }
#pragma unroll
      for (int k = 0; k < OFF_NA * 4; ++k) {
        if (cm[k] < best[k]) brun[k] = t0 + tl;
        best[k] = fminf(best[k], cm[k]);
      }
    }
    flush();
    if (g + 2 < G) {                       // recycle this buffer for group g+2
      __syncthreads();
      if (tid == 0) {
        fence_proxy_async();
        const int g2 = g + 2, t2 = (g2 * nt) / G, n2 = ((g2 + 1) * nt) / G - t2;
        mbar_expect_tx(&bars[g & 1], (uint32_t)n2 * WM_TILE_BYTES);
        for (int t = 0; t < n2; ++t)
          tma_load_1d(s_buf + ((int64_t)(g & 1) * p.tiles_per_buf + t) * WM_TILE_F4, edges_b + (int64_t)(t2 + t) * WM_TILE_F4, WM_TILE_BYTES, &bars[g & 1]);
      }
    }
  }
  __syncthreads();

  // ---- finalize: exact segment inside the winning run, sign, signed distance ----
  float* s_csd = (float*)s_buf;            // [4*nvalid] corner signed distances (buffers are free now)
  for (int i = tid; i < 4 * nvalid; i += OFF_THREADS) {
    const int ci = i >> 2, k = i & 3;
    float sd = -FLT_MAX;                                                   // D20
    if (nseg > 0) {
      const uint32_t run = (uint32_t)(s_key[i] & 0xffffffffull);
      const int tau = (int)(run >> 5), ln = (int)(run & 31u);
      const float offx = (k & 1) ? s_ag[4 * Ap + ci] : s_ag[2 * Ap + ci];
      const float offy = (k & 1) ? s_ag[5 * Ap + ci] : s_ag[3 * Ap + ci];
      const float sgn = (k & 2) ? -1.f : 1.f;
      const float qx = s_ag[0 * Ap + ci], qy = s_ag[1 * Ap + ci];
      const float4* tp = edges_b + (int64_t)tau * WM_TILE_F4 + ln;
      // the lane's 16 stored segments of this tile sit at lane*16 + it*2 + {0,1}; exact ties
      // inside the run go to the lower source point index (D17)
      const int32_t* srcp = p.seg_src + (int64_t)b * p.seg_tiles * WM_TILE_SEGS + tau * WM_TILE_SEGS + ln * WM_RUN;
      float bd2 = __int_as_float(0x7f800000), bwx = 0.f, bwy = 0.f;
      int bs = 0, bsrc = 0x7fffffff;
#pragma unroll
      for (int it = 0; it < 8; ++it) {
        const float4 P = __ldg(&tp[(it * 3 + 0) * 32]), E = __ldg(&tp[(it * 3 + 1) * 32]), Gv = __ldg(&tp[(it * 3 + 2) * 32]);
        const int2 sr = __ldg((const int2*)(srcp + it * 2));
        const float w0x = fmaf(sgn, offx, qx - P.x), w0y = fmaf(sgn, offy, qy - P.z);
        const float w1x = fmaf(sgn, offx, qx - P.y), w1y = fmaf(sgn, offy, qy - P.w);
        const float d0 = seg_d2(w0x, w0y, E.x, E.z, Gv.x, Gv.z);
        const float d1 = seg_d2(w1x, w1y, E.y, E.w, Gv.y, Gv.w);
        if (sr.x >= 0 && (d0 < bd2 || (d0 == bd2 && sr.x < bsrc))) { bd2 = d0; bwx = w0x; bwy = w0y; bs = it * 2; bsrc = sr.x; }
        if (sr.y >= 0 && (d1 < bd2 || (d1 == bd2 && sr.y < bsrc))) { bd2 = d1; bwx = w1x; bwy = w1y; bs = it * 2 + 1; bsrc = sr.y; }
      }
      const int s = tau * WM_TILE_SEGS + ln * WM_RUN + bs;
      const float2 sdir = __ldg(&p.sign_dir[(int64_t)b * p.seg_tiles * WM_TILE_SEGS + s]);
      const float side = fmaf(sdir.x, bwy, -sdir.y * bwx);                 // e x (q - p0), D16
      const float d = sqrtf(bd2);
      sd = side > 0.f ? -d : d;                                            // left = on-road = negative
    }
    s_csd[i] = sd;
    if (p.corner) p.corner[((int64_t)b * 4 + k) * A + s_aidx[ci]] = sd;
  }
  __syncthreads();
  for (int ci = tid; ci < nvalid; ci += OFF_THREADS) {
    const float m = fmaxf(fmaxf(s_csd[4 * ci], s_csd[4 * ci + 1]), fmaxf(s_csd[4 * ci + 2], s_csd[4 * ci + 3]));  // D18
    const int a = s_aidx[ci];
    p.sd[(int64_t)b * p.sd_stride_b + a] = m;
    p.flag[(int64_t)b * p.flag_stride_b + a] = (uint8_t)(m > 0.f);         // D19
  }
}

cudaError_t wm_launch_offroad(wm_handle* h, const wm_traj& sim, int t, float* sd, int64_t sd_stride_b,
                              float* corner, uint8_t* flag, int64_t flag_stride_b, cudaStream_t s) {
  if (h->cfg.offroad_mode != WM_OFFROAD_BRUTE_FORCE)
    return wm_launch_offroad_grid(h, sim, t, sd, sd_stride_b, corner, flag, flag_stride_b, s);
  OffroadParams p;
  p.row = wm_make_row(sim, t);
  p.A = sim.A;
  p.edges = h->edges; p.sign_dir = h->sign_dir; p.n_seg = h->n_seg; p.seg_src = h->seg_src; p.seg_tiles = h->seg_tiles;
  p.sd = sd; p.sd_stride_b = sd_stride_b; p.corner = corner; p.flag = flag; p.flag_stride_b = flag_stride_b;
  const size_t fixed = off_fixed_bytes(sim.A);
  // Two 256-thread CTAs per SM (each <= 113 KB of shared memory) so that one CTA's set-up,
  // flushes and re-scan overlap the other's main loop; one 512-thread CTA per SM when the
  // per-agent arrays leave too little room (large A).
  const size_t sm_total = 227 * 1024, per_cta2 = (sm_total - 2048) / 2;
  const bool two = fixed + 2 * 2 * (size_t)WM_TILE_BYTES <= per_cta2;
  const size_t max_smem = two ? per_cta2 : sm_total;
  int tpb = (int)((max_smem - fixed) / (2 * (size_t)WM_TILE_BYTES));
  const int need = (h->seg_tiles + 1) / 2;        // two buffers hold the whole scenario if they can
  if (tpb > need) tpb = need;
  if (tpb < 1) tpb = 1;
  p.tiles_per_buf = tpb;
  const size_t smem = fixed + 2 * (size_t)tpb * WM_TILE_BYTES;
  {                                                // per-device attributes: set at every launch (cheap)
    cudaError_t e = cudaFuncSetAttribute(k_offroad<512, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_total);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_offroad<256, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)per_cta2);
    if (e != cudaSuccess) return e;
  }
  if (two) k_offroad<256, 2><<<sim.B, 256, smem, s>>>(p);
  else k_offroad<512, 1><<<sim.B, 512, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
