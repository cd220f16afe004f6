// a4 off-road metric, exact search with group culling — the default mode.
//
// Same definition and same per-pair arithmetic as k_offroad (wm_offroad.cu); what changes is
// which pairs are evaluated.  wm_prepare stores the segments in spatial (Morton-cell) order
// and keeps one axis-aligned bounding box per group of 64 stored segments.  A warp owns one
// valid agent at a time (4 corners in registers), lanes own 2 segments of a group (packed
// FFMA2 math):
//   1. every lane computes, for one group per round, the squared distance v_k from each box
//      corner q_k to the group's bounding box: v_k <= squared distance of q_k to any segment
//      of the group;
//   2. on the first pass the group with the smallest bound is evaluated first, which gives
//      near-final per-corner bests;
//   3. a group is evaluated only if v_k <= best_k (with a rounding slack) for some corner k;
//      the warp-wide bests are refreshed (REDUX.MIN) once per round of 32 groups, and two
//      surviving groups are in flight per loop iteration.
// A group is skipped only when it cannot improve any corner, so the nearest segment is never
// missed: results equal the brute-force kernel's bit for bit (up to which of two exactly tied
// segments wins, which only matters inside the ambiguity band).  Segment tiles are streamed
// by bulk TMA into double-buffered shared memory, so the kernel's floor is the HBM time of
// the segment tiles (24 B/segment/scenario per launch): bound = HBM.
#include <float.h>
#include <stdlib.h>

#include "wm_internal.cuh"

constexpr int CULL_MAXR = 4;        // rounds of 32 groups resident at once
constexpr int CULL_CAP = CULL_MAXR * 4;   // tile slots resident at once (16 tiles = 8192 segments), one mbarrier each
constexpr float CULL_REL = 1.0005f; // slack of the cull test: v > best*REL + ABS  (float32 rounding
constexpr float CULL_ABS = 1e-5f;   //   of the 200 m-scale corner coordinates)

struct CullParams {
  wm_row row;
  int A;
  const float4* edges; const float2* sign_dir; const int32_t* n_seg; const float4* groups;
  int seg_tiles, cap_tiles;   // tiles per scenario in `edges`; resident tile slots (<= CULL_CAP)
  float* sd; int64_t sd_stride_b;
  float* corner;
  uint8_t* flag; int64_t flag_stride_b;
  unsigned long long* stats;   // [0] groups evaluated, [1] groups considered (wm_offroad_stats)
};

// [bars 128 B][misc 128 B][agent SoA 6*Ap floats][aidx Ap][best 4*Ap floats][win 4*Ap ints][group boxes][buffers]
static inline size_t cull_fixed_bytes(int A, int seg_tiles) {
  const size_t Ap = (size_t)((A + 31) / 32) * 32;
  size_t n = 256 + Ap * (6 * 4 + 4 + 16 + 16) + (size_t)seg_tiles * 8 * 16;
  return (n + 127) / 128 * 128;
}

struct CullAgent {            // one agent's state while a warp works on it (registers)
  float cx, cy, ax, ay, bx, by;
  float best[4];              // per-lane best squared distance per corner
  int bpos[4];                // stored position of the segment that gave it
};

// 2 segments (packed) x 4 corners of one agent against group `gi` of the resident buffer
__device__ __forceinline__ void cull_evaluate(CullAgent& a, const float4* buf, int gi, int pos0, int lane) {
  const float4* tp = buf + (int64_t)(gi >> 3) * WM_TILE_F4 + (gi & 7) * 96 + lane;
  const float4 P = tp[0], E = tp[32], Gv = tp[64];
  const wm_u64 Px = pk2(P.x, P.y), Py = pk2(P.z, P.w), Ex = pk2(E.x, E.y), Ey = pk2(E.z, E.w), Gx = pk2(Gv.x, Gv.y);
  const wm_u64 wcx = sub2(pk2(a.cx, a.cx), Px), wcy = sub2(pk2(a.cy, a.cy), Py);
  const int pos = pos0 + (gi >> 3) * WM_TILE_SEGS + (gi & 7) * 64 + lane * 2;
#pragma unroll
  for (int k = 0; k < 4; ++k) {
    wm_u64 wx, wy;
    if (k == 0)      { wx = add2(wcx, pk2(a.ax, a.ax)); wy = add2(wcy, pk2(a.ay, a.ay)); }
    else if (k == 1) { wx = add2(wcx, pk2(a.bx, a.bx)); wy = add2(wcy, pk2(a.by, a.by)); }
    else if (k == 2) { wx = sub2(wcx, pk2(a.ax, a.ax)); wy = sub2(wcy, pk2(a.ay, a.ay)); }
    else             { wx = sub2(wcx, pk2(a.bx, a.bx)); wy = sub2(wcy, pk2(a.by, a.by)); }
    const wm_u64 tm = mul2(wx, Gx);
    float tl0, tl1, wy0, wy1;
    upk2(tm, tl0, tl1); upk2(wy, wy0, wy1);
    const float t0s = __saturatef(fmaf(wy0, Gv.z, tl0)), t1s = __saturatef(fmaf(wy1, Gv.w, tl1));
    const wm_u64 nt2 = pk2(-t0s, -t1s);
    const wm_u64 rx = fma2(nt2, Ex, wx), ry = fma2(nt2, Ey, wy);
    const wm_u64 d2 = fma2(ry, ry, mul2(rx, rx));
    float d0, d1;
    upk2(d2, d0, d1);
    const float cm = fminf(d0, d1);
    if (cm < a.best[k]) { a.best[k] = cm; a.bpos[k] = pos + (d1 < d0 ? 1 : 0); }
  }
}

template <int NT, int MINB>
__global__ void __launch_bounds__(NT, MINB) k_offroad_cull(CullParams p, int fixed_bytes) {
  constexpr int NW = NT / 32;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  const int A = p.A, Ap = ((A + 31) / 32) * 32;
  uint64_t* bars = (uint64_t*)smem_raw;                    // [CULL_CAP] one full-barrier per resident tile slot
  int* s_misc = (int*)(smem_raw + 128);
  float* s_ag = (float*)(smem_raw + 256);                  // [6][Ap] cx, cy, ax, ay, bx, by (compacted)
  int* s_aidx = (int*)(s_ag + 6 * Ap);
  float* s_best = (float*)(s_aidx + Ap);                   // [4*Ap] best squared distance per corner
  int* s_win = (int*)(s_best + 4 * Ap);                    // [4*Ap] stored position of the winning segment
  float4* s_grp = (float4*)(s_win + 4 * Ap);               // [nt*8] bounding boxes {x0,y0,x1,y1}
  float4* s_buf = (float4*)(smem_raw + fixed_bytes);

  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int nseg = p.n_seg[b];
  const int nt = (nseg + WM_TILE_SEGS - 1) / WM_TILE_SEGS;
  const int G = (nt + p.cap_tiles - 1) / p.cap_tiles;      // passes (1 when the scenario fits: the usual case)
  const float4* edges_b = p.edges + (int64_t)b * p.seg_tiles * WM_TILE_F4;
  const float4* groups_b = p.groups + (int64_t)b * p.seg_tiles * 8;

  // every pass arms all CULL_CAP barriers (unused slots with 0 bytes) so their phases stay in step
  auto issue_pass = [&](int g) {
    const int t0 = (g * nt) / G, n = ((g + 1) * nt) / G - t0;
    for (int t = 0; t < CULL_CAP; ++t) {
      mbar_expect_tx(&bars[t], t < n ? (uint32_t)WM_TILE_BYTES : 0u);
      if (t < n) tma_load_1d(s_buf + (int64_t)t * WM_TILE_F4, edges_b + (int64_t)(t0 + t) * WM_TILE_F4, WM_TILE_BYTES, &bars[t]);
    }
  };
  if (tid == 0) { for (int t = 0; t < CULL_CAP; ++t) mbar_init(&bars[t], 1); mbar_fence_init(); }
  __syncthreads();
  if (tid == 0 && G > 0) issue_pass(0);
  // ---- agent set-up: order-preserving compaction of valid agents, corner offsets ----
  const int64_t ro = (int64_t)b * p.row.stride_b;
  if (tid == 0) s_misc[0] = 0;
  for (int i = tid; i < nt * 8; i += NT) s_grp[i] = __ldg(&groups_b[i]);
  __syncthreads();
  for (int base = 0; base < Ap; base += NT) {
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
      float sn, cs;
      sincosf(p.row.yaw[ro + a], &sn, &cs);
      const float hl = 0.5f * p.row.length[ro + a], hw = 0.5f * p.row.width[ro + a];
      const float hfx = hl * cs, hfy = hl * sn, hsx = -hw * sn, hsy = hw * cs;
      s_ag[0 * Ap + ci] = x;          s_ag[1 * Ap + ci] = y;
      s_ag[2 * Ap + ci] = hfx + hsx;  s_ag[3 * Ap + ci] = hfy + hsy;   // a: front-left offset
      s_ag[4 * Ap + ci] = hfx - hsx;  s_ag[5 * Ap + ci] = hfy - hsy;   // b: front-right offset
      s_aidx[ci] = a;
    } else if (a < A) {                                                 // D10
      p.sd[(int64_t)b * p.sd_stride_b + a] = 0.f;
      p.flag[(int64_t)b * p.flag_stride_b + a] = 0;
      if (p.corner) for (int k = 0; k < 4; ++k) p.corner[((int64_t)b * 4 + k) * A + a] = 0.f;
    }
    __syncthreads();
    if (tid == 0) { int tot = 0; for (int w = 0; w < NW; ++w) tot += s_misc[1 + w]; s_misc[0] += tot; }
    __syncthreads();
  }
  const int nvalid = s_misc[0];
  for (int i = tid; i < 4 * nvalid; i += NT) { s_best[i] = __int_as_float(0x7f800000); s_win[i] = -1; }
  __syncthreads();

  // ---- search ----
  const float INF = __int_as_float(0x7f800000);
  unsigned int n_eval = 0, n_cand = 0;       // warp-uniform counters for wm_offroad_stats
  for (int g = 0; g < G; ++g) {
    const int t0 = (g * nt) / G, ntg = ((g + 1) * nt) / G - t0;
    const uint32_t par = (uint32_t)(g & 1);
    const float4* buf = s_buf;
    const int ng = ntg * 8, pos0 = t0 * WM_TILE_SEGS;

    for (int ci = warp; ci < nvalid; ci += NW) {
      CullAgent a;
      a.cx = s_ag[0 * Ap + ci]; a.cy = s_ag[1 * Ap + ci];
      a.ax = s_ag[2 * Ap + ci]; a.ay = s_ag[3 * Ap + ci]; a.bx = s_ag[4 * Ap + ci]; a.by = s_ag[5 * Ap + ci];
      float wb[4];                                         // warp-wide best per corner (uniform)
#pragma unroll
      for (int k = 0; k < 4; ++k) { wb[k] = a.best[k] = s_best[ci * 4 + k]; a.bpos[k] = s_win[ci * 4 + k]; }
      const bool first = wb[0] == INF;
      n_cand += (unsigned)((min((t0 + ntg) * WM_TILE_SEGS, nseg) - pos0 + 63) / 64);
      const float qx[4] = {a.cx + a.ax, a.cx + a.bx, a.cx - a.ax, a.cx - a.bx};
      const float qy[4] = {a.cy + a.ay, a.cy + a.by, a.cy - a.ay, a.cy - a.by};

      // squared distance of each corner to each resident group's box, one group per lane per round
      float v[CULL_MAXR][4], vmin[CULL_MAXR];
#pragma unroll
      for (int r = 0; r < CULL_MAXR; ++r) {
        const int gi = r * 32 + lane;
        const bool in = gi < ng;
        const float4 c = in ? s_grp[t0 * 8 + gi] : make_float4(WM_FAR, WM_FAR, WM_FAR, WM_FAR);
        float m = INF;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
          const float dx = fmaxf(fmaxf(c.x - qx[k], qx[k] - c.z), 0.f), dy = fmaxf(fmaxf(c.y - qy[k], qy[k] - c.w), 0.f);
          v[r][k] = in ? fmaf(dx, dx, dy * dy) : INF;
          m = fminf(m, v[r][k]);
        }
        vmin[r] = m;
      }
      auto refresh = [&]() {
#pragma unroll
        for (int k = 0; k < 4; ++k) wb[k] = __uint_as_float(__reduce_min_sync(0xffffffffu, __float_as_uint(a.best[k])));
      };
      // first pass: seed with the group of the smallest bound
      if (first) {
        float lm = vmin[0]; int lr = 0;
#pragma unroll
        for (int r = 1; r < CULL_MAXR; ++r) if (vmin[r] < lm) { lm = vmin[r]; lr = r; }
        const uint32_t mw = __reduce_min_sync(0xffffffffu, __float_as_uint(lm));
        const uint32_t bal = __ballot_sync(0xffffffffu, __float_as_uint(lm) == mw);
        const int l = __ffs(bal) - 1;
        const int r = __shfl_sync(0xffffffffu, lr, l);
        if (__uint_as_float(mw) < 1e30f) {
          mbar_wait(&bars[(r * 32 + l) >> 3], par);            // only the tile that holds the seed group
          cull_evaluate(a, buf, r * 32 + l, pos0, lane); ++n_eval;
          refresh();
#pragma unroll
          for (int rr = 0; rr < CULL_MAXR; ++rr)
            if (lane == l && rr == r) { v[rr][0] = INF; v[rr][1] = INF; v[rr][2] = INF; v[rr][3] = INF; }
        }
      }
      // sweep: a group survives if it can still improve some corner
#pragma unroll
      for (int r = 0; r < CULL_MAXR; ++r) {
        if (r * 32 < ng) {
          bool surv = false;
#pragma unroll
          for (int k = 0; k < 4; ++k) surv = surv || (v[r][k] <= fmaf(wb[k], CULL_REL, CULL_ABS));
          uint32_t mask = __ballot_sync(0xffffffffu, surv);
          if (mask) {
#pragma unroll
            for (int q = 0; q < 4; ++q) if (r * 4 + q < ntg) mbar_wait(&bars[r * 4 + q], par);   // this round's tiles
            while (mask) {
              const int l1 = __ffs(mask) - 1;
              mask &= mask - 1;
              cull_evaluate(a, buf, r * 32 + l1, pos0, lane); ++n_eval;
              if (mask) {
                const int l2 = __ffs(mask) - 1;
                mask &= mask - 1;
                cull_evaluate(a, buf, r * 32 + l2, pos0, lane); ++n_eval;
              }
            }
            refresh();
          }
        }
      }
      // warp-wide winner per corner: min squared distance, then lowest stored position
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        const uint32_t bits = __float_as_uint(a.best[k]);
        const uint32_t m = __reduce_min_sync(0xffffffffu, bits);
        const uint32_t cand = bits == m ? (uint32_t)a.bpos[k] : 0x7fffffffu;
        const uint32_t w = __reduce_min_sync(0xffffffffu, cand);
        if (lane == 0) { s_best[ci * 4 + k] = __uint_as_float(m); s_win[ci * 4 + k] = (int)w; }
      }
      __syncwarp();
    }
    // no bulk copy may be in flight when the slots are recycled or the CTA exits
    for (int t = 0; t < CULL_CAP; ++t) mbar_wait(&bars[t], par);
    if (g + 1 < G) {
      __syncthreads();
      if (tid == 0) { fence_proxy_async(); issue_pass(g + 1); }
    }
  }
  if (lane == 0 && p.stats) { atomicAdd(&p.stats[0], (unsigned long long)n_eval); atomicAdd(&p.stats[1], (unsigned long long)n_cand); }
  __syncthreads();

  // ---- finalize: sign from the oriented winning segment, signed distance ----
  float* s_csd = (float*)s_buf;
  for (int i = tid; i < 4 * nvalid; i += NT) {
    const int ci = i >> 2, k = i & 3;
    float sd = -FLT_MAX;                                                   // D20
    const int s = s_win[i];
    if (nseg > 0 && s >= 0) {
      const int tau = s / WM_TILE_SEGS, r = s % WM_TILE_SEGS;
      const float4 P = __ldg(&edges_b[(int64_t)tau * WM_TILE_F4 + ((r >> 6) * 3) * 32 + ((r >> 1) & 31)]);
      const float p0x = (r & 1) ? P.y : P.x, p0y = (r & 1) ? P.w : P.z;
      const float offx = (k & 1) ? s_ag[4 * Ap + ci] : s_ag[2 * Ap + ci];
      const float offy = (k & 1) ? s_ag[5 * Ap + ci] : s_ag[3 * Ap + ci];
      const float sgn = (k & 2) ? -1.f : 1.f;
      const float wx = fmaf(sgn, offx, s_ag[0 * Ap + ci] - p0x), wy = fmaf(sgn, offy, s_ag[1 * Ap + ci] - p0y);
      const float2 sdir = __ldg(&p.sign_dir[(int64_t)b * p.seg_tiles * WM_TILE_SEGS + s]);
      const float side = fmaf(sdir.x, wy, -sdir.y * wx);                   // e x (q - p0), D16
      const float d = sqrtf(s_best[i]);
      sd = side > 0.f ? -d : d;
    }
    s_csd[i] = sd;
    if (p.corner) p.corner[((int64_t)b * 4 + k) * A + s_aidx[ci]] = sd;
  }
  __syncthreads();
  for (int ci = tid; ci < nvalid; ci += NT) {
    const float m = fmaxf(fmaxf(s_csd[4 * ci], s_csd[4 * ci + 1]), fmaxf(s_csd[4 * ci + 2], s_csd[4 * ci + 3]));  // D18
    const int a = s_aidx[ci];
    p.sd[(int64_t)b * p.sd_stride_b + a] = m;
    p.flag[(int64_t)b * p.flag_stride_b + a] = (uint8_t)(m > 0.f);         // D19
  }
}

cudaError_t wm_launch_offroad_culled(wm_handle* h, const wm_traj& sim, int t, float* sd, int64_t sd_stride_b,
                                     float* corner, uint8_t* flag, int64_t flag_stride_b, cudaStream_t s) {
  CullParams p;
  p.row = wm_make_row(sim, t);
  p.A = sim.A;
  p.edges = h->edges; p.sign_dir = h->sign_dir; p.n_seg = h->n_seg; p.groups = h->groups; p.seg_tiles = h->seg_tiles;
  p.sd = sd; p.sd_stride_b = sd_stride_b; p.corner = corner; p.flag = flag; p.flag_stride_b = flag_stride_b;
  p.stats = h->cull_stats;
  const size_t fixed = cull_fixed_bytes(sim.A, h->seg_tiles);
  static int forced = -1;
  if (forced < 0) { const char* e = getenv("WM_OFFROAD_CTA"); forced = e ? atoi(e) : 0; }
  const size_t sm_total = 227 * 1024, per_cta2 = (sm_total - 2048) / 2;
  // two 256-thread CTAs per SM only if the whole scenario still fits in each one's share
  bool two = fixed + (size_t)h->seg_tiles * WM_TILE_BYTES <= per_cta2;
  if (forced == 512) two = false;
  if (forced == 256 && fixed + 2 * (size_t)WM_TILE_BYTES <= per_cta2) two = true;
  const size_t max_smem = two ? per_cta2 : sm_total;
  if (fixed + (size_t)WM_TILE_BYTES > max_smem) return cudaErrorInvalidConfiguration;
  int cap = (int)((max_smem - fixed) / (size_t)WM_TILE_BYTES);
  if (cap > h->seg_tiles) cap = h->seg_tiles;
  if (cap > CULL_CAP) cap = CULL_CAP;
  if (cap < 1) cap = 1;
  p.cap_tiles = cap;
  const size_t smem = fixed + (size_t)cap * WM_TILE_BYTES;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_offroad_cull<512, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_total);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_offroad_cull<768, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_total);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_offroad_cull<1024, 1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm_total);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_offroad_cull<256, 2>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)per_cta2);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  if (two) k_offroad_cull<256, 2><<<sim.B, 256, smem, s>>>(p, (int)fixed);
  else if (forced == 768) k_offroad_cull<768, 1><<<sim.B, 768, smem, s>>>(p, (int)fixed);
  else if (forced == 1024) k_offroad_cull<1024, 1><<<sim.B, 1024, smem, s>>>(p, (int)fixed);
  else k_offroad_cull<512, 1><<<sim.B, 512, smem, s>>>(p, (int)fixed);
  h->launches++;
  return cudaGetLastError();
}
