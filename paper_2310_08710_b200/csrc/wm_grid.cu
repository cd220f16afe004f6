// a4 off-road metric, exact grid search — the default mode (WM_OFFROAD_CULLED).
// See wm_grid.cuh for the structure and the argument why no nearest segment can be missed.
//
//   k_grid_params        per scenario: bounding box of the segments -> the outer grid (box + wide margin,
//                        coarse cells) and, aligned with it, the mid grid (the outer cells under box + small
//                        margin split 2 x 2) and the inner grid (the mid cells split 2 x 2)
//   k_build_cells<0>     per outer cell: dmin(c), then the runs of records with dist(c, s) <= dmin + 2 rho,
//                        from the chunks whose boxes can matter (one warp per 8 x 4 cells)
//   k_build_cells<1>     per mid cell: the same two passes over its PARENT's list only
//   k_build_cells<2>     per inner cell: likewise, over its mid parent's list
//   k_offroad_grid       one thread per box corner, 4 lanes per agent: header load, candidate walk,
//                        sign of the winner; max over the corners by shuffles
//
// Bound of k_offroad_grid: instruction issue (about 14 instructions per evaluated pair, ~7 pairs
// per corner) and L1/L2 gather latency; HBM traffic is the touched 32-byte sectors only.
#include <stdlib.h>

#include "wm_grid.cuh"

// ======================================================================================
// grid construction (wm_prepare)
// ======================================================================================
constexpr int BUILD_MAXRUN = WM_GRID_MAXRUN;   // runs per cell before the cell falls back to the full search
constexpr int BUILD_MAXCAND = 256;        // candidates per cell before it falls back
constexpr int BUILD_WARPS = 4;            // warps per CTA of the build kernels (8: 0.6 ms slower, the warps of a CTA end at very different times)
constexpr int BUILD_AHEAD = 8;            // scenarios between a CTA and the one whose records it prefetches into L2

__global__ void __launch_bounds__(128) k_grid_params(const int32_t* n_seg, const float4* chunks, int seg_cap, float h_min,
                                                     float margin_in, float margin, WmGrid* gridp, int32_t* pool_cnt) {
  __shared__ float s_red[4][4];
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int n = n_seg[b], nch = (n + WM_CHUNK - 1) / WM_CHUNK;
  const float4* ch = chunks + (int64_t)b * (seg_cap / WM_CHUNK);
  float x0 = 3.0e38f, y0 = 3.0e38f, x1 = -3.0e38f, y1 = -3.0e38f;
  for (int c = tid; c < nch; c += blockDim.x) {
    const float4 bb = ch[c];
    x0 = fminf(x0, bb.x); y0 = fminf(y0, bb.y); x1 = fmaxf(x1, bb.z); y1 = fmaxf(y1, bb.w);
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    x0 = fminf(x0, __shfl_xor_sync(0xffffffffu, x0, d)); y0 = fminf(y0, __shfl_xor_sync(0xffffffffu, y0, d));
    x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, d)); y1 = fmaxf(y1, __shfl_xor_sync(0xffffffffu, y1, d));
  }
  if (lane == 0) { s_red[0][warp] = x0; s_red[1][warp] = y0; s_red[2][warp] = x1; s_red[3][warp] = y1; }
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < 4; ++w) {
      x0 = fminf(x0, s_red[0][w]); y0 = fminf(y0, s_red[1][w]); x1 = fmaxf(x1, s_red[2][w]); y1 = fmaxf(y1, s_red[3][w]);
    }
    WmGrid g;
    g.nseg = n; g.icx0 = 0; g.icy0 = 0; g.mbase = 0; g.pad0 = 0; g.pad1 = 0; g.pad2 = 0;
    if (n <= 0) {
      g.x0 = 0.f; g.y0 = 0.f; g.h = h_min; g.inv_h = 1.f / h_min; g.nx = 0; g.ny = 0; g.obase = 0;
      g.ox0 = 0.f; g.oy0 = 0.f; g.oh = 4.f * h_min; g.oinv_h = 1.f / g.oh; g.onx = 0; g.ony = 0;
    } else {
      // outer: the bounding box + margin; its cell side is 4 inner sides, and at most
      // WM_GRID_NG_IN / 4 of its cells per axis lie under the inner grid
      const float W = (x1 - x0) + 2.f * margin, H = (y1 - y0) + 2.f * margin;
      const float Wi = (x1 - x0) + 2.f * margin_in, Hi = (y1 - y0) + 2.f * margin_in;
      const float oh = fmaxf(4.f * h_min, fmaxf(fmaxf(W, H) * (1.0001f / WM_GRID_NG_OUT),
                                                fmaxf(Wi, Hi) * (1.0001f / (WM_GRID_NG_IN / 4 - 1))));
      g.ox0 = x0 - margin; g.oy0 = y0 - margin; g.oh = oh; g.oinv_h = 1.f / oh;
      g.onx = min(WM_GRID_NG_OUT, (int)ceilf(W / oh)); g.ony = min(WM_GRID_NG_OUT, (int)ceilf(H / oh));
      // inner: the outer cells that meet the bounding box + margin_in, each split 4 x 4 (2 x 2 mid cells of 2 x 2)
      const int cx0 = max(0, (int)floorf((x0 - margin_in - g.ox0) / oh)), cy0 = max(0, (int)floorf((y0 - margin_in - g.oy0) / oh));
      int cx1 = min(g.onx, (int)ceilf((x1 + margin_in - g.ox0) / oh)), cy1 = min(g.ony, (int)ceilf((y1 + margin_in - g.oy0) / oh));
      cx1 = min(cx1, cx0 + WM_GRID_NG_IN / 4); cy1 = min(cy1, cy0 + WM_GRID_NG_IN / 4);
      g.icx0 = cx0; g.icy0 = cy0;
      g.h = 0.25f * oh; g.inv_h = 1.f / g.h;
      g.x0 = g.ox0 + (float)cx0 * oh; g.y0 = g.oy0 + (float)cy0 * oh;
      g.nx = 4 * (cx1 - cx0); g.ny = 4 * (cy1 - cy0);
      g.obase = 4 * ((g.nx + 1) >> 1) * ((g.ny + 1) >> 1);
      g.mbase = g.obase + 4 * ((g.onx + 1) >> 1) * ((g.ony + 1) >> 1);
    }
    gridp[b] = g;
    pool_cnt[b] = 0;
  }
}

// plain float32 distance^2 from a cell centre to a record (safety comes from the slack below)
__device__ __forceinline__ float centre_d2(const float4 r0, const float4 r1, float cx, float cy) {
  const float wx = cx - r0.x, wy = cy - r0.y;
  const float t = __saturatef(fmaf(wy, r1.y, wx * r1.x));
  const float rx = fmaf(-t, r0.z, wx), ry = fmaf(-t, r0.w, wy);
  return fmaf(ry, ry, rx * rx);
}
// The same for the two records of a pair record (P, NE, G: wm_grid.cuh), packed; w = c - p0 comes back too.
__device__ __forceinline__ void centre_pair_d2(const float4 P, const float4 NE, const float4 G, wm_u64 cx2, wm_u64 cy2,
                                               wm_u64& wx, wm_u64& wy, float& d_e, float& d_o) {
  wx = sub2(cx2, pk2(P.x, P.y)); wy = sub2(cy2, pk2(P.z, P.w));
  const wm_u64 m = mul2(wx, pk2(G.x, G.y));
  float wy_e, wy_o, m_e, m_o;
  upk2(wy, wy_e, wy_o); upk2(m, m_e, m_o);
  const wm_u64 t = pk2(__saturatef(fmaf(wy_e, G.z, m_e)), __saturatef(fmaf(wy_o, G.w, m_o)));
  const wm_u64 rx = fma2(t, pk2(NE.x, NE.y), wx), ry = fma2(t, pk2(NE.z, NE.w), wy);
  upk2(fma2(ry, ry, mul2(rx, rx)), d_e, d_o);
}

// A record that passes the distance test is still dropped when it can never be the REPORTED
// nearest segment of any point of the cell (exact in real arithmetic, tested on the four corners
// of the inflated cell because the conditions are linear in q):
//   P  the whole cell projects before p0 of s, and s-1 ends in that same stored point: then
//      d(q, s-1) <= |q - p0| = d(q, s) and the tie rule prefers the lower index (D17);
//   N  the whole cell projects beyond p1 of s AND onto the interior side of s+1, which starts in
//      that same stored point: then d(q, s+1) < |q - p1| = d(q, s).
// Along a polyline this leaves the few segments whose perpendicular slab meets the cell (about
// h/spacing + 2) instead of everything within dmin + 2 rho.  Whether a rule can apply to a record, the
// next record's edge vector f and |ex| + |ey| come precomputed per pair record (seglk, k_fill_segments), so
// the test is a dozen packed operations on w = c - p0 with no further loads and no branches:
//   P   w.e + hh ae < -eps                          <=>  w.(-e) > kk aP          kk = hh + 2 mm, eps = 2 mm ae
//   N   (w - e).e - hh ae > eps  and  (w - e).f - hh af > 2 mm af     (w - e = c - p1 up to an ulp of the coordinates)
// aP / aN are +inf when the rule cannot apply.  Returns the keep flags of the even and the odd record.
__device__ __forceinline__ void slab_keep(const float4 NE, const float4 L0, const float4 L1, wm_u64 wx, wm_u64 wy, float kk,
                                          bool& keep_e, bool& keep_o) {
  const wm_u64 nex = pk2(NE.x, NE.y), ney = pk2(NE.z, NE.w);
  float pn_e, pn_o, vn_e, vn_o, vf_e, vf_o;
  upk2(fma2(wy, ney, mul2(wx, nex)), pn_e, pn_o);                        // w.(-e)
  const wm_u64 vx = add2(wx, nex), vy = add2(wy, ney);                   // c - p1
  upk2(fma2(vy, ney, mul2(vx, nex)), vn_e, vn_o);                        // (c - p1).(-e)
  upk2(fma2(vy, pk2(L0.z, L0.w), mul2(vx, pk2(L0.x, L0.y))), vf_e, vf_o);   // (c - p1).f
  const float af_e = fabsf(L0.x) + fabsf(L0.z), af_o = fabsf(L0.y) + fabsf(L0.w);
  const bool drop_e = pn_e > kk * L1.x || (-vn_e > kk * L1.z && vf_e > kk * af_e);
  const bool drop_o = pn_o > kk * L1.y || (-vn_o > kk * L1.w && vf_o > kk * af_o);
  keep_e = !drop_e; keep_o = !drop_o;
}

// One warp per block of 8 x 4 cells, one lane per cell.  Outer cells: chunks that cannot hold a candidate
// of any cell of the block are dropped with one box-box test per chunk (lanes over chunks); the survivors
// are walked twice: dmin(c), then the candidates.  Mid and inner cells: both passes walk the parent's runs;
// there is no chunk pass at these levels, so a cell whose parent has no list (all-ones header: too many runs
// or candidates, or the pool was full) gets the all-ones header too and its queries take the exact search
// over all chunks.  wm_grid_stats counts such cells per level (the bench prints the shares).
//
// Both passes take the records two by two (pair records, packed arithmetic).  Pass 2 marks the pair
// records that hold a candidate in a bit mask over the run (or chunk) being walked; the set stretches
// of the mask are the cell's runs, already in the header's format (first pair << 5 | pairs).
// LEVEL 0: outer cells, 1: mid cells, 2: inner cells
template <int LEVEL>
__global__ void __launch_bounds__(32 * BUILD_WARPS, 1024 / (32 * BUILD_WARPS)) k_build_cells(const float4* segrec, const float4* segpair, const float4* seglk, const float4* chunks,
                                                     int seg_cap, const WmGrid* gridp, uint2* cells, uint32_t* pool,
                                                     int32_t* pool_cnt) {
  __shared__ uint32_t s_runs[BUILD_WARPS][BUILD_MAXRUN][32];
  const int b = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const WmGrid g = gridp[b];
  // A scenario's records are read by its own CTAs only, all at about the same time: every first touch
  // would be a DRAM miss in a dependent chain.  Each CTA asks L2 for its share of the pair and link records of
  // the scenario BUILD_AHEAD places further on (bulk prefetch: no registers, no waiting).
  if (threadIdx.x == 0 && b + BUILD_AHEAD < (int)gridDim.y) {
    const int bn = b + BUILD_AHEAD;
    const uint32_t np = (uint32_t)((gridp[bn].nseg + 1) >> 1), per = (np + gridDim.x - 1) / gridDim.x;
    const uint32_t p0 = min(np, per * blockIdx.x), p1 = min(np, p0 + per);
    if (p1 > p0) {
      const float4* pn = segpair + (int64_t)bn * (seg_cap / 2) * 3 + p0;
      l2_prefetch(pn, (p1 - p0) * 16u); l2_prefetch(pn + seg_cap / 2, (p1 - p0) * 16u); l2_prefetch(pn + 2 * (seg_cap / 2), (p1 - p0) * 16u);
      l2_prefetch(seglk + ((int64_t)bn * (seg_cap / 2) + p0) * 2, (p1 - p0) * 32u);
    }
  }
  // the warp's block of 8 x 4 cells of its level
  constexpr bool FINE = LEVEL > 0;
  const int wg = blockIdx.x * BUILD_WARPS + warp;
  const int gnx = LEVEL == 0 ? g.onx : LEVEL == 1 ? (g.nx >> 1) : g.nx, gny = LEVEL == 0 ? g.ony : LEVEL == 1 ? (g.ny >> 1) : g.ny;
  const float gx0 = FINE ? g.x0 : g.ox0, gy0 = FINE ? g.y0 : g.oy0, h = LEVEL == 0 ? g.oh : LEVEL == 1 ? 2.f * g.h : g.h;
  const int cbase = LEVEL == 0 ? g.obase : LEVEL == 1 ? g.mbase : 0;
  const int nbx = (gnx + 7) >> 3, nby = (gny + 3) >> 2;
  if (wg >= nbx * nby) return;                                  // warp-uniform
  const int bx = wg % nbx, by = wg / nbx;
  const int ix = bx * 8 + (lane & 7), iy = by * 4 + (lane >> 3);
  const float4* rec = segrec + (int64_t)b * seg_cap * 2;
  const float4* pair = segpair + (int64_t)b * (seg_cap / 2) * 3;     // three planes of PS parts (wm_grid.cuh)
  const int PS = seg_cap / 2;
  const float4* lk = seglk + (int64_t)b * (seg_cap / 2) * 2;
  const float4* ch = chunks + (int64_t)b * (seg_cap / WM_CHUNK);
  uint2* cells_b = cells + (int64_t)b * WM_GRID_CELLS;
  uint32_t* pool_b = pool + (int64_t)b * WM_POOL_CAP;
  const int n = g.nseg, nch = (n + WM_CHUNK - 1) / WM_CHUNK;
  const float cx = gx0 + ((float)ix + 0.5f) * h, cy = gy0 + ((float)iy + 0.5f) * h;
  const wm_u64 cx2 = pk2(cx, cx), cy2 = pk2(cy, cy);
  // cell box inflated by delta (float32 rounding of the query's cell index), half diagonal rho
  const float delta = 1e-3f + 1e-4f * h;
  const float hh = 0.5f * h + delta;
  const float kk = hh + 2e-3f;                                    // rules P / N: half side + 2 mm along the edge
  const float rho = 1.41421362f * hh;
  const bool in = ix < gnx && iy < gny;
  const float INF = __int_as_float(0x7f800000);

  float dmin2 = INF;
  int nr = 0, npair = 0;
  uint32_t open_run = 0u;                                         // the last run, not yet stored: first pair << 5 | pairs
  // the set stretches of `m` (bit j = pair record first + j holds a candidate) join the cell's runs
  auto add_mask = [&](uint32_t m, int first) {
    while (m) {
      const int a = __ffs(m) - 1;
      const uint32_t t = ~(m >> a);
      const int len = t ? __ffs(t) - 1 : 32 - a;
      m = len + a >= 32 ? 0u : (m & (0xffffffffu << (a + len)));
      npair += len;
      int f0 = first + a, left = len;
      // continue the open run when it ends where this stretch begins
      if (open_run && (int)(open_run >> 5) + (int)(open_run & 31u) == f0 && (open_run & 31u) < 31u) {
        const int take = min(left, 31 - (int)(open_run & 31u));
        open_run += (uint32_t)take; f0 += take; left -= take;
      }
      while (left > 0) {
        if (open_run) { if (nr < BUILD_MAXRUN) s_runs[warp][nr][lane] = open_run; ++nr; }
        const int take = min(left, 31);
        open_run = ((uint32_t)f0 << 5) | (uint32_t)take; f0 += take; left -= take;
      }
    }
  };
  // pass 2 on one pair record: does it hold a candidate of this cell?
  auto pair_hit = [&](int pid, float thr2) -> bool {
    const float4 P = __ldg(pair + pid), NE = __ldg(pair + PS + pid), G = __ldg(pair + 2 * PS + pid);
    const float4 L0 = __ldg(lk + 2 * pid), L1 = __ldg(lk + 2 * pid + 1);
    wm_u64 wx, wy;
    float de, dq;
    bool ke, ko;
    centre_pair_d2(P, NE, G, cx2, cy2, wx, wy, de, dq);
    slab_keep(NE, L0, L1, wx, wy, kk, ke, ko);
    return (de <= thr2 && ke) || (dq <= thr2 && ko);              // padding records (1e18) never pass
  };
  bool crowded = false;                                           // under a crowded parent: crowded as well
  if constexpr (FINE) {
    // Mid / inner cell: its inflated box lies inside its parent's (the cell above it, 2 x 2 children),
    // so every segment that is the reported nearest one of a point of this cell is in the
    // parent's list, and so is the nearest segment of the cell centre: both passes walk the
    // parent's runs (a few dozen records) instead of the surviving chunks.  The children of a crowded
    // parent (no list: its queries search all chunks) are crowded too.
    uint2 ph = make_uint2(0u, 0u);
    if (in) ph = LEVEL == 1 ? cells_b[g.obase + wm_cell_index(g.icx0 + (ix >> 1), g.icy0 + (iy >> 1), g.onx)]
                            : cells_b[g.mbase + wm_cell_index(ix >> 1, iy >> 1, g.nx >> 1)];
    crowded = (ph.x & ph.y) == 0xffffffffu;
    if (crowded) ph = make_uint2(0u, 0u);
    {
      auto walk_runs = [&](auto&& f) {                  // the parent's pair runs (wm_internal.cuh): f(first pair, pairs)
        uint32_t r = ph.x & 0x1fffffu, r1 = ((ph.x >> 21) | (ph.y << 11)) & 0x1fffffu, r2 = ph.y >> 10;
        const uint32_t* pl = pool_b;
        int np = 0;
        if (r2 & 0x200000u) { pl += r2 & 0x1fffffu; np = (int)pl[0]; r2 = pl[1]; pl += 2; --np; }
        while (r != 0u) {
          f((int)(r >> 5), (int)(r & 31u));
          r = r1; r1 = r2; r2 = 0u;
          if (np > 0) { r2 = *pl++; --np; }
        }
      };
      walk_runs([&](int first, int cnt) {
        for (int q = 0; q < cnt; ++q) {
          const int pid = first + q;
          wm_u64 wx, wy;
          float de, dq;
          centre_pair_d2(__ldg(pair + pid), __ldg(pair + PS + pid), __ldg(pair + 2 * PS + pid), cx2, cy2, wx, wy, de, dq);
          dmin2 = fminf(dmin2, fminf(de, dq));
        }
      });
      const float dmin = sqrtf(dmin2);
      const float thr = dmin + 2.f * rho + (1e-3f + 1e-4f * dmin);
      const float thr2 = thr * thr;
      walk_runs([&](int first, int cnt) {
        uint32_t m = 0u;
        for (int q = 0; q < cnt; ++q) m |= (uint32_t)pair_hit(first + q, thr2) << q;
        if (in) add_mask(m, first);
      });
    }
  } else {
  // block box
  const float X0 = gx0 + (float)(bx * 8) * h - delta, X1 = gx0 + (float)(bx * 8 + 8) * h + delta;
  const float Y0 = gy0 + (float)(by * 4) * h - delta, Y1 = gy0 + (float)(by * 4 + 4) * h + delta;

  // bound for the whole block: the chunk whose box is nearest to the block centre is evaluated
  // exactly (lanes over its records); every cell centre of the block then has a segment within
  // d_centre + (half diagonal of the block's cell centres), and no candidate of any cell lies
  // farther than that + 2 rho from its cell centre, hence from the block box.
  const float bcx = 0.5f * (X0 + X1), bcy = 0.5f * (Y0 + Y1);
  float lmin = INF;
  int cmin = 0;
  for (int c = lane; c < nch; c += 32) {
    const float lb2 = wm_chunk_lb2(__ldg(ch + c), bcx, bcy);
    if (lb2 < lmin) { lmin = lb2; cmin = c; }
  }
  {
    const uint32_t mm = __reduce_min_sync(0xffffffffu, __float_as_uint(lmin));
    cmin = __shfl_sync(0xffffffffu, cmin, __ffs(__ballot_sync(0xffffffffu, __float_as_uint(lmin) == mm)) - 1);
  }
  float dc2 = INF;
  {
    const int sidx = cmin * WM_CHUNK + lane;
    if (sidx < n) dc2 = centre_d2(__ldg(rec + 2 * sidx), __ldg(rec + 2 * sidx + 1), bcx, bcy);
    dc2 = __uint_as_float(__reduce_min_sync(0xffffffffu, __float_as_uint(dc2)));
  }
  const float hdiag = 0.5f * h * 7.6157732f;                        // sqrt(7^2 + 3^2) cells between the extreme centres
  const float reach = (sqrtf(dc2) + hdiag) * 1.001f + 2.f * rho + 4e-3f;
  const float reach2 = reach * reach;
  auto survivors = [&](int r) -> uint32_t {
    const int c = r * 32 + lane;
    bool sv = false;
    if (c < nch) {
      const float4 bb = __ldg(ch + c);
      const float dx = fmaxf(fmaxf(bb.x - X1, X0 - bb.z), 0.f), dy = fmaxf(fmaxf(bb.y - Y1, Y0 - bb.w), 0.f);
      sv = fmaf(dx, dx, dy * dy) <= reach2;
    }
    return __ballot_sync(0xffffffffu, sv);
  };
  const int nround = (nch + 31) >> 5;
  constexpr int CP = WM_CHUNK / 2;                                  // pair records per chunk

  {
    // Both passes run chunk by chunk with the roles turned: the lanes hold the chunk's 16 pair records
    // (twice: lanes 0-15 and 16-31), and only the cells whose own bound reaches the chunk's box are taken,
    // two at a time, one per half warp.  A cell far from a chunk that its block neighbours need costs nothing.
    const int half = lane >> 4, q = lane & 15;
    auto cell_centre = [&](int i, float& x, float& y) { x = __shfl_sync(0xffffffffu, cx, i); y = __shfl_sync(0xffffffffu, cy, i); };
    auto half_min = [&](float v) {                          // min over the 16 lanes of a half warp
#pragma unroll
      for (int d = 8; d > 0; d >>= 1) v = fminf(v, __shfl_xor_sync(0xffffffffu, v, d));
      return v;
    };
    // pass 1: dmin(c).  The block's nearest chunk first (a tight start); a cell takes a chunk only if
    // the chunk's box can still improve it.
    auto pass1_chunk = [&](int c) {
      uint32_t need = __ballot_sync(0xffffffffu, in && wm_chunk_lb2(__ldg(ch + c), cx, cy) < dmin2);
      if (!need) return;
      const int pid = c * CP + q;
      const float4 P = __ldg(pair + pid), NE = __ldg(pair + PS + pid), G = __ldg(pair + 2 * PS + pid);
      while (need) {
        const int i0 = __ffs(need) - 1;
        need &= need - 1;
        const int i1 = need ? __ffs(need) - 1 : i0;
        need &= need - 1;                                           // 0 & (0 - 1) = 0
        float x, y;
        cell_centre(half ? i1 : i0, x, y);
        wm_u64 wx, wy;
        float de, dq;
        centre_pair_d2(P, NE, G, pk2(x, x), pk2(y, y), wx, wy, de, dq);
        const float mb = half_min(fminf(de, dq));
        const float m0 = __shfl_sync(0xffffffffu, mb, 0), m1 = __shfl_sync(0xffffffffu, mb, 16);
        if (lane == i0) dmin2 = fminf(dmin2, m0);
        if (lane == i1) dmin2 = fminf(dmin2, m1);
      }
    };
    // a bound for every cell first: its distance to the first and the middle point of every surviving chunk
    // (lanes over cells, 2 loads per chunk); the chunks that can still improve a cell are then few
    for (int r = 0; r < nround; ++r) {
      uint32_t mask = survivors(r);
      while (mask) {
        const int c = r * 32 + __ffs(mask) - 1;
        mask &= mask - 1;
        const float4 Pa = __ldg(pair + c * CP), Pb = __ldg(pair + c * CP + CP / 2);      // p0 of records 32 c and 32 c + 16 (1e18 if padding)
        const float ax = cx - Pa.x, ay = cy - Pa.z, bx2 = cx - Pb.x, by2 = cy - Pb.z;
        dmin2 = fminf(dmin2, fminf(fmaf(ax, ax, ay * ay), fmaf(bx2, bx2, by2 * by2)));
      }
    }
    dmin2 = dmin2 * 1.00001f + 1e-6f;                       // the bound is a point distance in other roundings than centre_pair_d2's
    if (nch > 0) pass1_chunk(cmin);
    for (int r = 0; r < nround; ++r) {
      uint32_t mask = survivors(r);
      while (mask) {
        const int c = r * 32 + __ffs(mask) - 1;
        mask &= mask - 1;
        if (c != cmin) pass1_chunk(c);
      }
    }
    // pass 2: candidates dist(c, s) <= dmin + 2 rho (+ slack)
    const float dmin = sqrtf(dmin2);
    const float thr = dmin + 2.f * rho + (1e-3f + 1e-4f * dmin);
    const float thr2 = thr * thr;
    const float thr2c = in ? thr2 * 1.0001f + 1e-5f : -1.f;         // chunk-level test, a little wider
    for (int r = 0; r < nround; ++r) {
      uint32_t mask = survivors(r);
      while (mask) {
        const int c = r * 32 + __ffs(mask) - 1;
        mask &= mask - 1;
        uint32_t need = __ballot_sync(0xffffffffu, wm_chunk_lb2(__ldg(ch + c), cx, cy) <= thr2c);
        if (!need) continue;
        const int pid = c * CP + q;
        const float4 P = __ldg(pair + pid), NE = __ldg(pair + PS + pid), G = __ldg(pair + 2 * PS + pid);
        const float4 L0 = __ldg(lk + 2 * pid), L1 = __ldg(lk + 2 * pid + 1);
        uint32_t mine = 0u;
        while (need) {
          const int i0 = __ffs(need) - 1;
          need &= need - 1;
          const int i1 = need ? __ffs(need) - 1 : i0;
          need &= need - 1;
          const int i = half ? i1 : i0;
          float x, y;
          cell_centre(i, x, y);
          const float t2 = __shfl_sync(0xffffffffu, thr2, i);
          wm_u64 wx, wy;
          float de, dq;
          bool ke, ko;
          centre_pair_d2(P, NE, G, pk2(x, x), pk2(y, y), wx, wy, de, dq);
          slab_keep(NE, L0, L1, wx, wy, kk, ke, ko);
          const uint32_t bal = __ballot_sync(0xffffffffu, (de <= t2 && ke) || (dq <= t2 && ko));
          if (lane == i0) mine = bal & 0xffffu;                     // bit j = pair record c * 16 + j holds a candidate of cell i0
          if (lane == i1 && i1 != i0) mine = bal >> 16;
        }
        if (mine) add_mask(mine, c * CP);
      }
    }
  }
  }
  if (open_run) { if (nr < BUILD_MAXRUN) s_runs[warp][nr][lane] = open_run; ++nr; }
  if (!in) return;
  // query header (wm_internal.cuh): three runs in the header, or two + the rest in the pool
  uint2 hd = make_uint2(0xffffffffu, 0xffffffffu);              // fall back to the full search
  if (n <= 0) hd = make_uint2(0u, 0u);
  else if (!crowded && nr <= BUILD_MAXRUN && 2 * npair <= BUILD_MAXCAND) {
    uint32_t f0 = nr > 0 ? s_runs[warp][0][lane] : 0u, f1 = nr > 1 ? s_runs[warp][1][lane] : 0u, f2 = nr > 2 ? s_runs[warp][2][lane] : 0u;
    bool ok = true;
    if (nr > 3) {
      const int off = atomicAdd(&pool_cnt[b], nr - 1);        // count word + (nr - 2) runs
      if (off + nr - 1 <= WM_POOL_CAP && off < (1 << 21)) {
        uint32_t* pw = pool_b + off;
        pw[0] = (uint32_t)(nr - 2);
        for (int i = 2; i < nr; ++i) pw[i - 1] = s_runs[warp][i][lane];
        f2 = 0x200000u | (uint32_t)off;
      } else ok = false;
    }
    if (ok) { hd.x = f0 | (f1 << 21); hd.y = (f1 >> 11) | (f2 << 10); }
  }
  cells_b[cbase + wm_cell_index(ix, iy, gnx)] = hd;
}

cudaError_t wm_launch_build_grid(wm_handle* h, int b0, int B, cudaStream_t s) {
  // inner cell side (lower bound), metres of outer / inner grid beyond the segments' bounding box (an agent at
  // 15 m/s leaves the map by up to 120 m in 8 s); the cell sides grow when the boxes do not fit
  // WM_GRID_NG_OUT / WM_GRID_NG_IN cells
  const float h_min = 2.0f, margin = 120.f, margin_in = 32.f;
  const int seg_cap = h->seg_tiles * WM_TILE_SEGS;
  const float4* segrec = h->segrec + (int64_t)b0 * seg_cap * 2;
  const float4* chunks = h->chunks + (int64_t)b0 * (seg_cap / WM_CHUNK);
  k_grid_params<<<B, 128, 0, s>>>(h->n_seg + b0, chunks, seg_cap, h_min, margin_in, margin, h->gridp + b0, h->pool_cnt + b0);
  h->launches++;
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  const float4* segpair = h->segpair + (int64_t)b0 * (seg_cap / 2) * 3;
  const float4* seglk = h->seglk + (int64_t)b0 * (seg_cap / 2) * 2;
  uint2* cells = h->cells + (int64_t)b0 * WM_GRID_CELLS;
  uint32_t* pool = h->pool + (int64_t)b0 * WM_POOL_CAP;
  // the outer grid first: its cells are the parents the inner cells build from
  k_build_cells<0><<<dim3((WM_GRID_NG_OUT / 8) * (WM_GRID_NG_OUT / 4) / BUILD_WARPS, B), 32 * BUILD_WARPS, 0, s>>>(segrec, segpair, seglk, chunks, seg_cap, h->gridp + b0, cells, pool, h->pool_cnt + b0);
  h->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_build_cells<1><<<dim3((WM_GRID_NG_IN / 16) * (WM_GRID_NG_IN / 8) / BUILD_WARPS, B), 32 * BUILD_WARPS, 0, s>>>(segrec, segpair, seglk, chunks, seg_cap, h->gridp + b0, cells, pool, h->pool_cnt + b0);
  h->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  k_build_cells<2><<<dim3((WM_GRID_NG_IN / 8) * (WM_GRID_NG_IN / 4) / BUILD_WARPS, B), 32 * BUILD_WARPS, 0, s>>>(segrec, segpair, seglk, chunks, seg_cap, h->gridp + b0, cells, pool, h->pool_cnt + b0);
  h->launches++;
  return cudaGetLastError();
}

// Diagnostics (wm_grid_stats): how many cells of each level exist and how many of them carry the
// "search all chunks" header.  One CTA per scenario; out[2 l] += cells, out[2 l + 1] += all-ones headers of
// level l = 0 inner, 1 mid, 2 outer.
__global__ void __launch_bounds__(256) k_grid_cell_stats(const WmGrid* gridp, const uint2* cells, unsigned long long* out) {
  const int b = blockIdx.x;
  const WmGrid g = gridp[b];
  const uint2* cb = cells + (int64_t)b * WM_GRID_CELLS;
  const int nx[3] = {g.nx, g.nx >> 1, g.onx}, ny[3] = {g.ny, g.ny >> 1, g.ony}, base[3] = {0, g.mbase, g.obase};
  for (int l = 0; l < 3; ++l) {
    int full = 0;
    const int n = nx[l] * ny[l];
    for (int i = threadIdx.x; i < n; i += blockDim.x) {
      const uint2 hd = cb[base[l] + wm_cell_index(i % nx[l], i / nx[l], nx[l])];
      full += (hd.x & hd.y) == 0xffffffffu;
    }
    full = __reduce_add_sync(0xffffffffu, full);
    if ((threadIdx.x & 31) == 0 && full) atomicAdd(&out[2 * l + 1], (unsigned long long)full);
    if (threadIdx.x == 0) atomicAdd(&out[2 * l], (unsigned long long)n);
  }
}

cudaError_t wm_launch_grid_cell_stats(wm_handle* h, unsigned long long* out, cudaStream_t s) {
  k_grid_cell_stats<<<h->prep_B, 256, 0, s>>>(h->gridp, h->cells, out);
  h->launches++;
  return cudaGetLastError();
}

// ======================================================================================
// k_offroad_grid
// ======================================================================================
struct GridParams {
  wm_row row;
  int A;
  const float4* segrec; const float4* segpair; const float4* segfin; const float4* chunks; const uint2* cells; const uint32_t* pool; const WmGrid* gridp;
  int seg_cap;
  float* sd; int64_t sd_stride_b;
  float* corner;
  uint8_t* flag; int64_t flag_stride_b;
  unsigned long long* stats;
};

__global__ void __launch_bounds__(128) k_offroad_grid(GridParams p) {
  const int b = blockIdx.y, tid = threadIdx.x, lane = tid & 31;
  const int a = blockIdx.x * 32 + (tid >> 2), k = tid & 3;
  const int A = p.A;
  const int64_t ro = (int64_t)b * p.row.stride_b;
  const bool v = a < A && p.row.valid[ro + a] != 0;
  const WmGridView gv = wm_grid_view(p.segrec, p.segpair, p.segfin, p.chunks, p.cells, p.pool, p.gridp, p.seg_cap, WM_POOL_CAP, b);
  int n_eval = 0;
  bool slow = false;
  float cx = 0.f, cy = 0.f, offx = 0.f, offy = 0.f;
  if (v) {
    cx = p.row.x[ro + a]; cy = p.row.y[ro + a];
    float ax, ay, bx, by;
    wm_box_offsets(p.row.yaw[ro + a], p.row.length[ro + a], p.row.width[ro + a], ax, ay, bx, by);
    const float ox = (k & 1) ? bx : ax, oy = (k & 1) ? by : ay;
    offx = (k & 2) ? -ox : ox; offy = (k & 2) ? -oy : oy;
  }
  const float sd = wm_grid_corner_sd(gv, v, cx, cy, offx, offy, n_eval, slow);     // 0 for invalid agents (D10)
  if (a < A && p.corner) p.corner[((int64_t)b * 4 + k) * A + a] = sd;
  float m = fmaxf(sd, __shfl_xor_sync(0xffffffffu, sd, 1));                  // D18: max over the 4 corners
  m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
  if (k == 0 && a < A) {
    p.sd[(int64_t)b * p.sd_stride_b + a] = v ? m : 0.f;
    p.flag[(int64_t)b * p.flag_stride_b + a] = (uint8_t)(v && m > 0.f);      // D19
  }
  if (p.stats) {
    const unsigned ne = __reduce_add_sync(0xffffffffu, (unsigned)n_eval);
    const unsigned nv = __popc(__ballot_sync(0xffffffffu, v)), ns = __popc(__ballot_sync(0xffffffffu, slow));
    if (lane == 0 && nv) {
      atomicAdd(&p.stats[0], (unsigned long long)ne);
      atomicAdd(&p.stats[1], (unsigned long long)nv * (unsigned long long)max(gv.g.nseg, 0));
      if (ns) atomicAdd(&p.stats[2], (unsigned long long)ns);
      atomicAdd(&p.stats[3], (unsigned long long)nv);
    }
  }
}

cudaError_t wm_launch_offroad_grid(wm_handle* h, const wm_traj& sim, int t, float* sd, int64_t sd_stride_b,
                                   float* corner, uint8_t* flag, int64_t flag_stride_b, cudaStream_t s) {
  const int64_t cap = (int64_t)h->seg_tiles * WM_TILE_SEGS;
  int64_t nbmax = cap > 0 ? (int64_t)0xffffffffLL / (cap * 24) : sim.B;     // pair records of a launch span < 4 GB (wm_grid.cuh)
  if (nbmax < 1) nbmax = 1;
  if (nbmax > 65535) nbmax = 65535;                                         // gridDim.y
  for (int64_t c0 = 0; c0 < sim.B; c0 += nbmax) {
    const int nb = (int)(sim.B - c0 < nbmax ? sim.B - c0 : nbmax);
    GridParams p;
    p.row = wm_make_row(sim, t);
    const int64_t ro = c0 * p.row.stride_b;
    p.row.x += ro; p.row.y += ro; p.row.yaw += ro; p.row.vel_x += ro; p.row.vel_y += ro; p.row.length += ro; p.row.width += ro; p.row.valid += ro;
    p.A = sim.A;
    p.segrec = h->segrec + c0 * cap * 2; p.segpair = h->segpair + c0 * (cap / 2) * 3; p.segfin = h->segfin + c0 * cap;
    p.chunks = h->chunks + c0 * (cap / WM_CHUNK); p.cells = h->cells + c0 * WM_GRID_CELLS; p.pool = h->pool + c0 * WM_POOL_CAP;
    p.gridp = h->gridp + c0;
    p.seg_cap = (int)cap;
    p.sd = sd + c0 * sd_stride_b; p.sd_stride_b = sd_stride_b; p.corner = corner ? corner + c0 * 4 * sim.A : nullptr;
    p.flag = flag + c0 * flag_stride_b; p.flag_stride_b = flag_stride_b;
    p.stats = h->stats_on ? h->cull_stats : nullptr;
    k_offroad_grid<<<dim3((sim.A + 31) / 32, nb), 128, 0, s>>>(p);
    h->launches++;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}
