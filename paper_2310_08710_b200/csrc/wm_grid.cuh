// a4 off-road metric: exact nearest-segment search through a uniform grid of
// per-cell candidate runs — device side of the query, shared by k_offroad_grid (wm_grid.cu)
// and the fused rollout kernel (wm_rollout_fused.cu).
//
// wm_prepare stores the road-edge segments of a scenario in ascending source order as 32-byte
// records and lays a grid of square cells (side h) over their bounding box.  For a cell with
// centre c and half diagonal rho, every segment that can be the nearest one of ANY point q of
// the cell satisfies  dist(c, s) <= dmin(c) + 2 rho   (triangle inequality, twice), where
// dmin(c) is the distance from c to its own nearest segment.  The cell keeps exactly those
// segments, as runs of consecutive record indices (polyline pieces are contiguous, so a road
// cell holds 1-3 runs).  A query is then: one 16-byte header load, a walk over ~20-40
// candidate records, no bounding tests.  Cells with too many runs, and points outside the
// grid, take a per-thread search over all 32-record chunks with bounding-box culling, which
// is exact as well.  Per-pair arithmetic is the same as in the brute-force kernel
// (wm_offroad.cu), so both modes return the same distances bit for bit.
#pragma once
#include <float.h>

#include "wm_internal.cuh"

constexpr float WM_CULL_REL = 1.0005f;   // slack of the chunk cull test: lb^2 > best^2*REL + ABS
constexpr float WM_CULL_ABS = 1e-5f;     //   (float32 rounding of 200 m-scale coordinates)

struct WmGridView {          // one scenario's prepared search structures
  const float4* rec;         // [nseg][2] {p0x,p0y,ex,ey} {gx,gy,sx,sy}
  const float4* chunks;      // [ceil(nseg/32)] bounding boxes {x0,y0,x1,y1}
  const uint4* cells;        // [ny*nx] headers
  const uint32_t* pool;      // overflow runs
  WmGrid g;
};

__device__ __forceinline__ WmGridView wm_grid_view(const float4* segrec, const float4* chunks, const uint4* cells,
                                                   const uint32_t* pool, const WmGrid* gridp, int seg_cap,
                                                   int pool_cap, int b) {
  WmGridView v;
  v.rec = segrec + (int64_t)b * seg_cap * 2;
  v.chunks = chunks + (int64_t)b * (seg_cap / WM_CHUNK);
  v.cells = cells + (int64_t)b * WM_GRID_CELLS;
  v.pool = pool + (int64_t)b * pool_cap;
  v.g = gridp[b];
  return v;
}

// squared distance of corner (c + off) to a record; w = (c - p0) + off keeps the rounding error
// independent of the map coordinates (DESIGN.md tolerances).  Same operations, in the same order
// and rounding, as the brute-force kernel (wm_offroad.cu).
__device__ __forceinline__ float wm_rec_d2(const float4 r0, const float4 r1, float cx, float cy, float offx, float offy) {
  const float wx = __fadd_rn(__fsub_rn(cx, r0.x), offx), wy = __fadd_rn(__fsub_rn(cy, r0.y), offy);
  const float t = __saturatef(__fmaf_rn(wy, r1.y, __fmul_rn(wx, r1.x)));
  const float rx = __fmaf_rn(-t, r0.z, wx), ry = __fmaf_rn(-t, r0.w, wy);
  return __fmaf_rn(ry, ry, __fmul_rn(rx, rx));
}

__device__ __forceinline__ void wm_grid_run(const float4* __restrict__ rec, uint32_t run, float cx, float cy,
                                            float offx, float offy, float& best, int& bs, int& n_eval) {
  int s = (int)(run >> 8);
  const int e = s + (int)(run & 255u);
  n_eval += e - s;
#pragma unroll 4
  for (; s < e; ++s) {
    const float d2 = wm_rec_d2(__ldg(rec + 2 * s), __ldg(rec + 2 * s + 1), cx, cy, offx, offy);
    if (d2 < best) { best = d2; bs = s; }      // ascending s + strict '<': exact ties -> lower index (D17)
  }
}

// Exact search over all chunks with bounding-box culling, by a whole warp for ONE corner (points
// outside the grid, crowded cells): lanes over chunks for the bounds, then lanes over the 32
// records of each surviving chunk.  All 32 lanes call with the same arguments and get the same
// result.  Chunks are visited in ascending order and a chunk replaces the incumbent only on
// strict '<', inside a chunk the lowest lane wins: exact ties -> lower index (D17).
__device__ __forceinline__ void wm_grid_search_warp(const WmGridView& v, float cx, float cy, float offx, float offy,
                                                    float& best, int& bs, int& n_eval) {
  const int lane = threadIdx.x & 31;
  const int nseg = v.g.nseg, nch = (nseg + WM_CHUNK - 1) / WM_CHUNK;
  const float qx = cx + offx, qy = cy + offy;
  const float INF = __int_as_float(0x7f800000);
  float U2 = INF;                                // some segment lies within the farthest corner of any chunk box
  for (int c = lane; c < nch; c += 32) {
    const float4 bb = __ldg(v.chunks + c);
    const float dx = fmaxf(fabsf(qx - bb.x), fabsf(qx - bb.z)), dy = fmaxf(fabsf(qy - bb.y), fabsf(qy - bb.w));
    U2 = fminf(U2, fmaf(dx, dx, dy * dy));
  }
  U2 = __uint_as_float(__reduce_min_sync(0xffffffffu, __float_as_uint(U2)));
  best = INF; bs = 0;
  for (int c0 = 0; c0 < nch; c0 += 32) {
    const int c = c0 + lane;
    float lb2 = INF;
    if (c < nch) {
      const float4 bb = __ldg(v.chunks + c);
      const float dx = fmaxf(fmaxf(bb.x - qx, qx - bb.z), 0.f), dy = fmaxf(fmaxf(bb.y - qy, qy - bb.w), 0.f);
      lb2 = fmaf(dx, dx, dy * dy);
    }
    uint32_t mask = __ballot_sync(0xffffffffu, lb2 <= fmaf(U2, WM_CULL_REL, WM_CULL_ABS));
    while (mask) {
      const int l = __ffs(mask) - 1;
      mask &= mask - 1;
      if (__shfl_sync(0xffffffffu, lb2, l) > fmaf(best, WM_CULL_REL, WM_CULL_ABS)) continue;   // warp-uniform
      const int s = (c0 + l) * WM_CHUNK + lane;
      float d2 = INF;
      if (s < nseg) d2 = wm_rec_d2(__ldg(v.rec + 2 * s), __ldg(v.rec + 2 * s + 1), cx, cy, offx, offy);
      n_eval += (lane == 0) ? min(WM_CHUNK, nseg - (c0 + l) * WM_CHUNK) : 0;
      const uint32_t m = __reduce_min_sync(0xffffffffu, __float_as_uint(d2));   // d2 >= +0: bits order as floats
      if (m < __float_as_uint(best)) {
        best = __uint_as_float(m);
        bs = (c0 + l) * WM_CHUNK + __ffs(__ballot_sync(0xffffffffu, __float_as_uint(d2) == m)) - 1;
      }
    }
  }
}

// Signed distance of the box corner (c + off) to the nearest road-edge segment (D15-D17, D19,
// D20).  Must be called by all 32 lanes of a warp (inactive lanes pass active = false): corners
// that cannot use their cell's candidate list are searched one at a time by the whole warp.
// n_eval counts evaluated pairs, fell_back is set for those corners.
__device__ __forceinline__ float wm_grid_corner_sd(const WmGridView& v, bool active, float cx, float cy, float offx,
                                                   float offy, int& n_eval, bool& fell_back) {
  const int lane = threadIdx.x & 31;
  float best = __int_as_float(0x7f800000);
  int bs = 0;
  bool slow = false;
  if (active && v.g.nseg > 0) {
    const float fx = (cx + offx - v.g.x0) * v.g.inv_h, fy = (cy + offy - v.g.y0) * v.g.inv_h;
    const int ix = (int)floorf(fx), iy = (int)floorf(fy);
    slow = !(fx >= 0.f && fy >= 0.f && ix < v.g.nx && iy < v.g.ny);
    if (!slow) {
      const uint4 hd = __ldg(v.cells + iy * v.g.nx + ix);
      if (hd.x != 0xffffffffu) {
        wm_grid_run(v.rec, hd.x, cx, cy, offx, offy, best, bs, n_eval);
        if (hd.y) wm_grid_run(v.rec, hd.y, cx, cy, offx, offy, best, bs, n_eval);
        if (hd.z) wm_grid_run(v.rec, hd.z, cx, cy, offx, offy, best, bs, n_eval);
        if (hd.w) wm_grid_run(v.rec, hd.w, cx, cy, offx, offy, best, bs, n_eval);
      } else if (hd.y != 0xffffffffu) {
        const uint32_t* pr = v.pool + hd.y;
        for (uint32_t i = 0; i < hd.z; ++i) wm_grid_run(v.rec, __ldg(pr + i), cx, cy, offx, offy, best, bs, n_eval);
      } else {
        slow = true;
      }
    }
  }
  fell_back = slow;
  uint32_t todo = __ballot_sync(0xffffffffu, slow);
  while (todo) {
    const int l = __ffs(todo) - 1;
    todo &= todo - 1;
    float b2; int s2, ne = 0;
    wm_grid_search_warp(v, __shfl_sync(0xffffffffu, cx, l), __shfl_sync(0xffffffffu, cy, l),
                        __shfl_sync(0xffffffffu, offx, l), __shfl_sync(0xffffffffu, offy, l), b2, s2, ne);
    ne = __shfl_sync(0xffffffffu, ne, 0);
    if (lane == l) { best = b2; bs = s2; n_eval += ne; }
  }
  if (!active) return 0.f;
  if (v.g.nseg <= 0) return -FLT_MAX;                                      // D20
  // sign from the oriented winning segment: e x (q - p0) > 0 is the left side = on-road (D16)
  const float4 r0 = __ldg(v.rec + 2 * bs), r1 = __ldg(v.rec + 2 * bs + 1);
  const float wx = __fadd_rn(__fsub_rn(cx, r0.x), offx), wy = __fadd_rn(__fsub_rn(cy, r0.y), offy);
  const float side = __fmaf_rn(r1.z, wy, -__fmul_rn(r1.w, wx));
  const float d = sqrtf(best);
  return side > 0.f ? -d : d;
}
