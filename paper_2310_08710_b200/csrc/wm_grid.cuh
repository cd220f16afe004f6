// a4 off-road metric: exact nearest-segment search through a uniform grid of
// per-cell candidate runs — device side of the query, shared by k_offroad_grid (wm_grid.cu)
// and the fused rollout kernel (wm_rollout_fused.cu).
//
// wm_prepare stores the road-edge segments of a scenario in ascending source order (32-byte
// records, and the same two by two as 48-byte pair records for packed arithmetic) and lays two
// nested grids of square cells over them (wm_internal.cuh): a fine inner one over the segments'
// bounding box, a coarse outer one over the wide margin around it.  For a cell with centre c and
// half diagonal rho, every segment that can be the nearest one of ANY point q of the cell satisfies
//     dist(c, s) <= dmin(c) + 2 rho        (triangle inequality, twice)
// where dmin(c) is the distance from c to its own nearest segment.  The cell keeps those segments
// (minus the ones a neighbour on the same polyline always beats, wm_grid.cu), as runs of
// consecutive pair records: polyline pieces are contiguous, so a road cell holds 1-3 runs.  A
// query is then: one 8-byte header load, a walk over ~4 pair records, no bounding tests.
// Cells with too many runs, and points outside both grids, take a warp search over all 32-record
// chunks with bounding-box culling, which is exact as well.  Per-pair arithmetic is the same as in
// the brute-force kernel (wm_offroad.cu): both modes return the same bits whenever they pick the
// same segment; at a polyline vertex, where rules P / N keep only the neighbour that wins in exact
// arithmetic, the float32 distances of the two neighbours can differ by an ulp, and so can the modes.
#pragma once
#include <float.h>

#include "wm_internal.cuh"

constexpr float WM_CULL_REL = 1.0005f;   // slack of the chunk cull test: lb^2 > best^2*REL + ABS
constexpr float WM_CULL_ABS = 1e-5f;     //   (float32 rounding of 200 m-scale coordinates)

// position of cell (ix, iy) in the header array: tiles of 2 x 2 cells, tile-row-major
__host__ __device__ __forceinline__ int wm_cell_index(int ix, int iy, int nx) {
  return (((iy >> 1) * ((nx + 1) >> 1) + (ix >> 1)) << 2) | ((iy & 1) << 1) | (ix & 1);
}

struct WmGridView {          // one scenario's prepared search structures
  const float4* rec;         // [nseg][2] {p0x,p0y,ex,ey} {gx,gy,sx,sy}
  const float4* fin;         // [nseg] {p0x, p0y, sx, sy}
  const float4* pair;        // [3][seg_cap/2] three planes; pair record p = records 2p (e) and 2p+1 (o): {p0x_e,p0x_o,p0y_e,p0y_o} | {-ex_e,-ex_o,-ey_e,-ey_o} | {gx_e,gx_o,gy_e,gy_o}
  const char* pair0;         // pair records of scenario 0 of the launch; this scenario's start at byte pair_off (< 2^32: the launchers see to it)
  uint32_t pair_off;
  uint32_t plane;            // bytes between the planes of a scenario = seg_cap / 2 * 16
  const float4* chunks;      // [ceil(nseg/32)] bounding boxes {x0,y0,x1,y1}
  const uint2* cells;        // headers, 2 x 2 tiles (wm_cell_index)
  const uint32_t* pool;      // overflow runs
  WmGrid g;
};

__device__ __forceinline__ WmGridView wm_grid_view(const float4* segrec, const float4* segpair, const float4* segfin, const float4* chunks, const uint2* cells,
                                                   const uint32_t* pool, const WmGrid* gridp, int seg_cap,
                                                   int pool_cap, int b) {
  WmGridView v;
  v.rec = segrec + (int64_t)b * seg_cap * 2;
  v.pair = segpair + (int64_t)b * (seg_cap / 2) * 3;
  v.pair0 = (const char*)segpair;
  v.pair_off = (uint32_t)b * (uint32_t)(seg_cap / 2) * 48u;
  v.plane = (uint32_t)(seg_cap / 2) * 16u;
  v.fin = segfin + (int64_t)b * seg_cap;
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

// The same squared distances for the two records of a pair record at once, with packed float32x2
// arithmetic (FADD2 / FMUL2 / FFMA2): component for component the operations and roundings of
// wm_rec_d2, so both give the same bits (fma(-t, e, w) == fma(t, -e, w); the pair stores -e).
__device__ __forceinline__ void wm_pair_d2(const float4 P, const float4 NE, const float4 G, wm_u64 cx2, wm_u64 cy2,
                                           wm_u64 ox2, wm_u64 oy2, float& d_e, float& d_o) {
  const wm_u64 wx = add2(sub2(cx2, pk2(P.x, P.y)), ox2), wy = add2(sub2(cy2, pk2(P.z, P.w)), oy2);
  const wm_u64 m = mul2(wx, pk2(G.x, G.y));
  float wy_e, wy_o, m_e, m_o;
  upk2(wy, wy_e, wy_o); upk2(m, m_e, m_o);
  const wm_u64 t = pk2(__saturatef(__fmaf_rn(wy_e, G.z, m_e)), __saturatef(__fmaf_rn(wy_o, G.w, m_o)));
  const wm_u64 rx = fma2(t, pk2(NE.x, NE.y), wx), ry = fma2(t, pk2(NE.z, NE.w), wy);
  upk2(fma2(ry, ry, mul2(rx, rx)), d_e, d_o);
}

// Cell header (8 bytes, wm_internal.cuh): up to three runs of PAIR records, 21 bits each
// (first pair << 5 | pairs, pairs <= 31), in bits 0-20, 21-41, 42-62.  Bit 63 set: the third field is
// an offset into the pool instead, pool[offset] = n further runs, pool[offset + 1 ...] = the runs.
// All ones = too many candidates: search all chunks.  Zero = nothing to walk.
//
// Walk of a cell's candidate runs as ONE flat loop (a warp runs max-over-lanes of the total
// count, not the sum of per-run maxima), one pair record = 2 records per iteration.  A run counts
// whole pair records: evaluating a real segment that is not a candidate cannot change the result
// (it is no nearer than the winner, and on an exact tie the winner has the lower index: D17;
// indices are visited in ascending order with strict '<').  Padding records sit at 1e18.
// The current run is one word, (pair << 5 | pairs left): an iteration adds 31 to it; the next two
// runs wait in registers, further ones come from the pool.
// The three 16-byte parts of a pair record live in three PLANES of the scenario's block (all first parts, all
// second parts, all third parts): the lanes of a warp walk neighbouring records, and eight neighbouring parts
// share a 128-byte line where the 48-byte records of an array-of-structures share it between 2.7 (the walk's
// loads are bound by the LSU's line wavefronts, profiles/r02_k_rollout_ncu.md).
// The winner comes back as `bso` = byte offset of its first part from the scenario's first (a multiple
// of 16) + 1 for the odd record of the pair; wm_bso_of / wm_rec_of convert.  Inside the walk offsets
// count from the first pair record of the LAUNCH (32 bits: one uniform base + a 32-bit lane offset).
__device__ __forceinline__ uint32_t wm_bso_of(int rec) { return (uint32_t)(rec >> 1) * 16u + (uint32_t)(rec & 1); }
__device__ __forceinline__ int wm_rec_of(uint32_t bso) { return (int)(2u * (bso >> 4) + (bso & 1u)); }

__device__ __forceinline__ void wm_grid_walk(const char* __restrict__ base, uint32_t off0, uint32_t plane, uint32_t r0, uint32_t r1, uint32_t r2,
                                             const uint32_t* __restrict__ pool, float cx, float cy, float offx, float offy,
                                             float& best, uint32_t& bso, int& n_eval) {
  const wm_u64 cx2 = pk2(cx, cx), cy2 = pk2(cy, cy), ox2 = pk2(offx, offx), oy2 = pk2(offy, offy);
  int n_pool = 0;
  if (r2 & 0x200000u) {                                             // the third field points into the pool
    pool += r2 & 0x1fffffu;
    n_pool = (int)__ldg(pool);
    r2 = __ldg(pool + 1);
    pool += 2; n_pool -= 1;
  }
  uint32_t off = off0 + (r0 >> 5) * 16u, cnt = r0 & 31u;            // the open run: byte offset of its next pair record, pairs left
  for (;;) {
    if (cnt == 0u) {                                                // run finished: the next one
      if (r1 == 0u) break;
      off = off0 + (r1 >> 5) * 16u; cnt = r1 & 31u;
      r1 = r2; r2 = 0u;
      if (n_pool > 0) { r2 = __ldg(pool); ++pool; --n_pool; }
    }
    const char* a = base + off;
    const float4 a0 = __ldg((const float4*)a), a1 = __ldg((const float4*)(a + plane)), a2 = __ldg((const float4*)(a + 2u * plane));
    float d0, d1;
    wm_pair_d2(a0, a1, a2, cx2, cy2, ox2, oy2, d0, d1);
    if (d0 < best) { best = d0; bso = off; }                        // ascending index, strict '<': exact ties -> lower index (D17)
    if (d1 < best) { best = d1; bso = off + 1u; }
    off += 16u; --cnt;
    n_eval += 2;
  }
  bso -= off0;
}

// Exact search over all chunks with bounding-box culling, by a whole warp for ONE corner (points
// outside the grid, crowded cells).  Best-first: lanes over chunks find the chunk whose box is
// nearest and evaluate it (lanes over its 32 records), which gives a tight bound at once; then
// every other chunk whose box can still reach that bound is evaluated.  All 32 lanes call with the
// same arguments and get the same result.  The incumbent is replaced on a smaller distance, or
// on an equal distance and a lower record index: exact ties -> lower index (D17).
__device__ __forceinline__ void wm_grid_eval_chunk(const WmGridView& v, int c, float cx, float cy, float offx, float offy,
                                                   float& best, int& bs, int& n_eval) {
  const int lane = threadIdx.x & 31;
  const int s = c * WM_CHUNK + lane;
  float d2 = __int_as_float(0x7f800000);
  if (s < v.g.nseg) d2 = wm_rec_d2(__ldg(v.rec + 2 * s), __ldg(v.rec + 2 * s + 1), cx, cy, offx, offy);
  n_eval += (lane == 0) ? min(WM_CHUNK, v.g.nseg - c * WM_CHUNK) : 0;
  const uint32_t m = __reduce_min_sync(0xffffffffu, __float_as_uint(d2));       // d2 >= +0: bits order as floats
  const int idx = c * WM_CHUNK + __ffs(__ballot_sync(0xffffffffu, __float_as_uint(d2) == m)) - 1;
  if (m < __float_as_uint(best) || (m == __float_as_uint(best) && idx < bs)) { best = __uint_as_float(m); bs = idx; }
}

__device__ __forceinline__ float wm_chunk_lb2(const float4 bb, float qx, float qy) {
  const float dx = fmaxf(fmaxf(bb.x - qx, qx - bb.z), 0.f), dy = fmaxf(fmaxf(bb.y - qy, qy - bb.w), 0.f);
  return fmaf(dx, dx, dy * dy);
}

__device__ __forceinline__ void wm_grid_search_warp(const WmGridView& v, float cx, float cy, float offx, float offy,
                                                    float& best, int& bs, int& n_eval) {
  const int lane = threadIdx.x & 31;
  const int nch = (v.g.nseg + WM_CHUNK - 1) / WM_CHUNK;
  const float qx = cx + offx, qy = cy + offy;
  const float INF = __int_as_float(0x7f800000);
  float lmin = INF;
  int cmin = 0;
  for (int c = lane; c < nch; c += 32) {
    const float lb2 = wm_chunk_lb2(__ldg(v.chunks + c), qx, qy);
    if (lb2 < lmin) { lmin = lb2; cmin = c; }
  }
  const uint32_t mm = __reduce_min_sync(0xffffffffu, __float_as_uint(lmin));
  const int c_first = __shfl_sync(0xffffffffu, cmin, __ffs(__ballot_sync(0xffffffffu, __float_as_uint(lmin) == mm)) - 1);
  best = INF; bs = 0x7fffffff;
  wm_grid_eval_chunk(v, c_first, cx, cy, offx, offy, best, bs, n_eval);
  for (int c0 = 0; c0 < nch; c0 += 32) {
    const int c = c0 + lane;
    float lb2 = INF;
    if (c < nch && c != c_first) lb2 = wm_chunk_lb2(__ldg(v.chunks + c), qx, qy);
    uint32_t mask = __ballot_sync(0xffffffffu, lb2 <= fmaf(best, WM_CULL_REL, WM_CULL_ABS));
    while (mask) {
      const int l = __ffs(mask) - 1;
      mask &= mask - 1;
      if (__shfl_sync(0xffffffffu, lb2, l) > fmaf(best, WM_CULL_REL, WM_CULL_ABS)) continue;   // warp-uniform
      wm_grid_eval_chunk(v, c0 + l, cx, cy, offx, offy, best, bs, n_eval);
    }
  }
}

// The same search for the four corners of ONE box at once (the fused rollout queues whole
// agents): chunk boxes are bounded against the box centre and its circumradius R, records are
// loaded once and evaluated for the four corners.  off[k] = corner k - centre.
__device__ __forceinline__ void wm_grid_search_warp4(const WmGridView& v, float cx, float cy, const float (&offx)[4],
                                                     const float (&offy)[4], float R, float (&best)[4], int (&bs)[4],
                                                     int& n_eval) {
  const int lane = threadIdx.x & 31;
  const int nseg = v.g.nseg, nch = (nseg + WM_CHUNK - 1) / WM_CHUNK;
  const float INF = __int_as_float(0x7f800000);
  auto eval4 = [&](int c) {
    const int s = c * WM_CHUNK + lane;
    float4 r0 = make_float4(0.f, 0.f, 0.f, 0.f), r1 = r0;
    const bool in = s < nseg;
    if (in) { r0 = __ldg(v.rec + 2 * s); r1 = __ldg(v.rec + 2 * s + 1); }
    n_eval += (lane == 0) ? 4 * min(WM_CHUNK, nseg - c * WM_CHUNK) : 0;
#pragma unroll
    for (int k = 0; k < 4; ++k) {
      const float d2 = in ? wm_rec_d2(r0, r1, cx, cy, offx[k], offy[k]) : INF;
      const uint32_t m = __reduce_min_sync(0xffffffffu, __float_as_uint(d2));
      if (m <= __float_as_uint(best[k])) {                       // warp-uniform
        const int idx = c * WM_CHUNK + __ffs(__ballot_sync(0xffffffffu, __float_as_uint(d2) == m)) - 1;
        if (m < __float_as_uint(best[k]) || idx < bs[k]) { best[k] = __uint_as_float(m); bs[k] = idx; }
      }
    }
  };
  float lmin = INF;
  int cmin = 0;
  for (int c = lane; c < nch; c += 32) {
    const float lb2 = wm_chunk_lb2(__ldg(v.chunks + c), cx, cy);
    if (lb2 < lmin) { lmin = lb2; cmin = c; }
  }
  const uint32_t mm = __reduce_min_sync(0xffffffffu, __float_as_uint(lmin));
  const int c_first = __shfl_sync(0xffffffffu, cmin, __ffs(__ballot_sync(0xffffffffu, __float_as_uint(lmin) == mm)) - 1);
#pragma unroll
  for (int k = 0; k < 4; ++k) { best[k] = INF; bs[k] = 0x7fffffff; }
  eval4(c_first);
  // a chunk matters if its box comes within max_k dist_k of some corner: lb(centre) - R <= max_k sqrt(best_k)
  auto reach2 = [&]() {
    const float bm = fmaxf(fmaxf(best[0], best[1]), fmaxf(best[2], best[3]));
    const float r = fmaf(sqrtf(bm), 1.0005f, R + 2e-3f);
    return r * r;
  };
  float B2 = reach2();
  for (int c0 = 0; c0 < nch; c0 += 32) {
    const int c = c0 + lane;
    float lb2 = INF;
    if (c < nch && c != c_first) lb2 = wm_chunk_lb2(__ldg(v.chunks + c), cx, cy);
    uint32_t mask = __ballot_sync(0xffffffffu, lb2 <= B2);
    while (mask) {
      const int l = __ffs(mask) - 1;
      mask &= mask - 1;
      if (__shfl_sync(0xffffffffu, lb2, l) > B2) continue;     // warp-uniform
      eval4(c0 + l);
      B2 = reach2();
    }
  }
}

// ---- query API (D15-D17, D19, D20) -------------------------------------------------------
// wm_grid_header: per thread; the header of the corner's cell: 0 = nothing to walk (inactive lane,
//                 no segments), all ones = the corner needs the warp search (outside both grids,
//                 crowded cell).
// wm_grid_fast_hd: per thread; walks the candidate list.  Returns true when the corner needs the
//                 warp search instead.
// wm_grid_search_warp: above.
// wm_grid_finish: per thread; sign from the oriented winning segment and the signed distance.
// wm_grid_corner_sd: the three combined for a warp of corners (k_offroad_grid).
__device__ __forceinline__ uint2 wm_grid_header(const WmGridView& v, bool active, float cx, float cy, float offx, float offy) {
  uint2 hd = make_uint2(0u, 0u);
  if (active && v.g.nseg > 0) {
    const float qx = cx + offx, qy = cy + offy;
    const float fx = (qx - v.g.x0) * v.g.inv_h, fy = (qy - v.g.y0) * v.g.inv_h;
    const int ix = (int)floorf(fx), iy = (int)floorf(fy);
    if (fx >= 0.f && fy >= 0.f && ix < v.g.nx && iy < v.g.ny) hd = __ldg(v.cells + wm_cell_index(ix, iy, v.g.nx));
    else {                                                        // off the inner grid: the coarse outer one
      const float gx = (qx - v.g.ox0) * v.g.oinv_h, gy = (qy - v.g.oy0) * v.g.oinv_h;
      const int jx = (int)floorf(gx), jy = (int)floorf(gy);
      if (gx >= 0.f && gy >= 0.f && jx < v.g.onx && jy < v.g.ony) hd = __ldg(v.cells + v.g.obase + wm_cell_index(jx, jy, v.g.onx));
      else hd = make_uint2(0xffffffffu, 0xffffffffu);
    }
  }
  return hd;
}

__device__ __forceinline__ bool wm_grid_fast_hd(const WmGridView& v, uint2 hd, float cx, float cy, float offx, float offy,
                                                float& best, uint32_t& bso, int& n_eval) {
  best = __int_as_float(0x7f800000);
  bso = 0u;
  const bool slow = (hd.x & hd.y) == 0xffffffffu;
  if (slow) { hd.x = 0u; hd.y = 0u; }
  // the three 21-bit fields; bit 21 of the third = "pool offset"
  const uint32_t r0 = hd.x & 0x1fffffu, r1 = ((hd.x >> 21) | (hd.y << 11)) & 0x1fffffu, r2 = hd.y >> 10;
  bso = v.pair_off;
  wm_grid_walk(v.pair0, v.pair_off, v.plane, r0, r1, r2, v.pool, cx, cy, offx, offy, best, bso, n_eval);   // no-op without runs
  return slow;
}

__device__ __forceinline__ float wm_grid_finish(const WmGridView& v, float cx, float cy, float offx, float offy, float best,
                                                uint32_t bso) {
  if (v.g.nseg <= 0) return -FLT_MAX;                                      // D20
  // e x (q - p0) > 0 is the left side of the oriented segment = on-road (D16).  p0 and e come from
  // the winner's pair record, which the walk has just pulled into L1 (no third dependent miss);
  // only a zero-length segment needs its stored direction from the finish record (D16 / D29).
  const char* a = (const char*)v.pair + (bso & ~1u);
  const float4 P = __ldg((const float4*)a), NE = __ldg((const float4*)(a + v.plane));
  const bool odd = (bso & 1u) != 0u;
  const float p0x = odd ? P.y : P.x, p0y = odd ? P.w : P.z;
  float sx = -(odd ? NE.y : NE.x), sy = -(odd ? NE.w : NE.z);
  if (sx == 0.f && sy == 0.f) { const float4 f = __ldg(v.fin + wm_rec_of(bso)); sx = f.z; sy = f.w; }
  const float wx = __fadd_rn(__fsub_rn(cx, p0x), offx), wy = __fadd_rn(__fsub_rn(cy, p0y), offy);
  const float side = __fmaf_rn(sx, wy, -__fmul_rn(sy, wx));
  const float d = sqrtf(best);
  return side > 0.f ? -d : d;
}

// Must be called by all 32 lanes of a warp (inactive lanes pass active = false): corners that
// cannot use their cell's candidate list are searched one at a time by the whole warp.
// n_eval counts evaluated pairs, fell_back is set for those corners.
__device__ __forceinline__ float wm_grid_corner_sd(const WmGridView& v, bool active, float cx, float cy, float offx,
                                                   float offy, int& n_eval, bool& fell_back) {
  const int lane = threadIdx.x & 31;
  float best;
  uint32_t bso;
  const bool slow = wm_grid_fast_hd(v, wm_grid_header(v, active, cx, cy, offx, offy), cx, cy, offx, offy, best, bso, n_eval);
  fell_back = slow;
  uint32_t todo = __ballot_sync(0xffffffffu, slow);
  while (todo) {
    const int l = __ffs(todo) - 1;
    todo &= todo - 1;
    float b2; int s2, ne = 0;
    wm_grid_search_warp(v, __shfl_sync(0xffffffffu, cx, l), __shfl_sync(0xffffffffu, cy, l),
                        __shfl_sync(0xffffffffu, offx, l), __shfl_sync(0xffffffffu, offy, l), b2, s2, ne);
    ne = __shfl_sync(0xffffffffu, ne, 0);
    if (lane == l) { best = b2; bso = wm_bso_of(s2); n_eval += ne; }
  }
  if (!active) return 0.f;
  return wm_grid_finish(v, cx, cy, offx, offy, best, bso);
}
