// a6 / a7 default observation: "transforms the location of all other vehicles to
// the agent's own coordinate frame, and sub-samples the roadgraph via distance".
//
// k_observe_hist: HBM-write bound (1.29 GB of features at config 3).  One CTA per (scenario,
// group of egos) stages the H history rows in shared memory once and streams out rows of A
// floats, fully coalesced.
//
// k_observe_topk: exact top-k by MSB radix select on the float32 key d2 = fma(dy,dy,dx*dx)
// (bit pattern of a non-negative float is order preserving).  One warp per valid ego, 16 egos
// per CTA share each roadgraph tile, which is streamed through shared memory by bulk TMA in
// double-buffered tiles.  Passes over the R points:
//   1. histogram of the key's top bits in lane-private shared-memory counters (no atomics)
//      -> bin of the k-th key (repeated on the bin's sub-range only if the bin is too large);
//   2. collect the (key, index) pairs of that bin (<= 1024) -> bitwise descent gives the exact
//      k-th key T and the number of ties to take;
//   3. emit, in ascending index order (ballot + popc compaction): key < T, or key == T and
//      among the first `quota` such points (ties -> lower index), with ego-frame features.
#include "wm_internal.cuh"

// ======================================================================================
// history -> ego frames
// ======================================================================================
constexpr int HIST_EGOS = 8;     // egos per CTA
constexpr float WM_PI = 3.14159265358979323846f;
constexpr float WM_TWO_PI = 6.28318530717958647692f;

__global__ void __launch_bounds__(256) k_observe_hist(wm_traj sim, int t, int H, float* hist, uint8_t* hist_valid) {
  extern __shared__ float sh[];                       // [H][7][A] floats + [H][A] valid bytes
  const int A = sim.A;
  const int b = blockIdx.y, e0 = blockIdx.x * HIST_EGOS;
  float* s_f = sh;
  uint8_t* s_v = (uint8_t*)(sh + (size_t)H * 7 * A);
  const float* src[7] = {sim.x, sim.y, sim.yaw, sim.vel_x, sim.vel_y, sim.length, sim.width};
  for (int i = threadIdx.x; i < H * A; i += blockDim.x) {
    const int h = i / A, a = i - h * A;
    const int64_t g = ((int64_t)b * sim.T + (t - H + 1 + h)) * A + a;
    const uint8_t v = sim.valid[g];
    s_v[i] = v;
#pragma unroll
    for (int f = 0; f < 7; ++f) s_f[(h * 7 + f) * A + a] = v ? src[f][g] : 0.f;   // D10: never use invalid data
  }
  __syncthreads();
  const int cur = H - 1;                              // row t
  for (int ee = 0; ee < HIST_EGOS; ++ee) {
    const int e = e0 + ee;
    if (e >= A) break;
    const bool ev = s_v[cur * A + e] != 0;
    const float ex = s_f[(cur * 7 + 0) * A + e], ey = s_f[(cur * 7 + 1) * A + e], eth = s_f[(cur * 7 + 2) * A + e];
    float sn, cs;
    sincosf(eth, &sn, &cs);
    float* out = hist + ((int64_t)b * A + e) * H * 7 * A;
    uint8_t* outv = hist_valid + ((int64_t)b * A + e) * H * A;
    for (int i = threadIdx.x; i < H * A; i += blockDim.x) {
      const int h = i / A, a = i - h * A;
      const bool v = ev && s_v[i] != 0;
      float o[7] = {0.f, 0.f, 0.f, 0.f, 0.f, 0.f, 0.f};
      if (v) {
        const float* r = s_f + (size_t)h * 7 * A + a;
        const float dx = r[0] - ex, dy = r[A] - ey;
        o[0] = fmaf(cs, dx, sn * dy);
        o[1] = fmaf(cs, dy, -sn * dx);
        const float d = r[2 * A] - eth;
        o[2] = d - WM_TWO_PI * floorf((d + WM_PI) * (1.f / WM_TWO_PI));   // wrap to [-pi, pi), D5
        const float vx = r[3 * A], vy = r[4 * A];
        o[3] = fmaf(cs, vx, sn * vy);
        o[4] = fmaf(cs, vy, -sn * vx);
        o[5] = r[5 * A];
        o[6] = r[6 * A];
      }
#pragma unroll
      for (int f = 0; f < 7; ++f) __stcs(&out[((int64_t)h * 7 + f) * A + a], o[f]);   // streaming store
      outv[i] = v;
    }
  }
}

cudaError_t wm_launch_observe_hist(wm_handle* h, const wm_traj& sim, int t, float* hist, uint8_t* hist_valid, cudaStream_t s) {
  const int H = h->cfg.history;
  const size_t smem = (size_t)H * 7 * sim.A * 4 + (size_t)H * sim.A;
  static size_t configured = 0;
  if (smem > 48 * 1024 && smem > configured) {
    cudaError_t e = cudaFuncSetAttribute(k_observe_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = smem;
  }
  dim3 grid((sim.A + HIST_EGOS - 1) / HIST_EGOS, sim.B);
  k_observe_hist<<<grid, 256, smem, s>>>(sim, t, H, hist, hist_valid);
  h->launches++;
  return cudaGetLastError();
}

// ======================================================================================
// top-k roadgraph points
// ======================================================================================
constexpr int TK_WARPS = 16;                 // egos per CTA
constexpr int TK_THREADS = TK_WARPS * 32;
constexpr int TK_BINS = 128;
constexpr int TK_CAPB = 1024;                // boundary (key, index) pairs per ego: 8 KB, aliases the histogram
constexpr uint32_t TK_KEY_FAR = 0x7149F2CAu; // bits of 1e30f: keys at or above are padding / invalid points
constexpr int TK_BASE = 119 << 2;            // level-0 bins start at d2 = 2^-8 (2 mantissa bits per bin)

struct TopkParams {
  wm_row row;
  int A, R, k;
  const float2* pts; int pts_pad;
  const float *dir_x, *dir_y; const int32_t* type;
  int32_t* rg_index; float* rg_feat; int32_t* rg_type;
};

enum { TK_HIST0 = 0, TK_HISTN = 1, TK_COLLECT = 2, TK_EMIT = 3 };

struct TkWarp {          // per-warp (per-ego) selection state, in registers
  float ex, ey, cs, sn;
  uint32_t lo, hi;       // undecided key range [lo, hi)
  int shift;             // linear sub-bin shift for TK_HISTN
  int c_less;            // points with key < lo
  int kk;                // min(k, number of real points)
  int in_bin;            // points with key in [lo, hi)
  uint32_t T; int quota; // exact threshold and ties to take
  int n_out, n_tie, n_col;
  int ego;               // agent slot of this warp's ego (-1: none)
  bool active, refine;
};

__device__ __forceinline__ int tk_bin0(uint32_t key) {
  if (key >= TK_KEY_FAR) return TK_BINS - 1;
  const int v = (int)(key >> 21) - TK_BASE;
  return min(max(v, 0), TK_BINS - 2);
}
__device__ __forceinline__ uint32_t tk_bin0_lo(int bin) { return bin <= 0 ? 0u : (uint32_t)(bin + TK_BASE) << 21; }
__device__ __forceinline__ uint32_t tk_bin0_hi(int bin) {
  return bin >= TK_BINS - 2 ? (bin == TK_BINS - 2 ? TK_KEY_FAR : 0xffffffffu) : (uint32_t)(bin + TK_BASE + 1) << 21;
}

// One streaming pass over the scenario's points.  All warps of the CTA walk the same tiles
// (double-buffered bulk TMA); each applies MODE to its own ego.
template <int MODE>
__device__ __forceinline__ void tk_pass(const TopkParams& p, int b, TkWarp& w, uint64_t* bars, float2* s_tiles,
                                        uint16_t* s_hist, uint2* s_col, uint32_t& tile_seq) {
  const int lane = threadIdx.x & 31;
  const int ntile = p.pts_pad / WM_PT_TILE;
  const float2* src = p.pts + (int64_t)b * p.pts_pad;
  const uint32_t lt = (1u << lane) - 1u;
  if (threadIdx.x == 0) {
    fence_proxy_async();
    for (int i = 0; i < 2 && i < ntile; ++i) {
      const uint32_t q = tile_seq + i;
      mbar_expect_tx(&bars[q & 1], WM_PT_TILE * 8);
      tma_load_1d(s_tiles + (q & 1) * WM_PT_TILE, src + (int64_t)i * WM_PT_TILE, WM_PT_TILE * 8, &bars[q & 1]);
    }
  }
  for (int ti = 0; ti < ntile; ++ti) {
    const uint32_t q = tile_seq + ti;
    mbar_wait(&bars[q & 1], (q >> 1) & 1);
    const float2* tile = s_tiles + (q & 1) * WM_PT_TILE;
    if (w.active && (MODE != TK_HISTN || w.refine)) {
#pragma unroll 4
      for (int j = 0; j < WM_PT_TILE / 32; ++j) {
        const int li = j * 32 + lane;
        const float2 pt = tile[li];
        const float dx = __fsub_rn(pt.x, w.ex), dy = __fsub_rn(pt.y, w.ey);
        const uint32_t key = __float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
        if (MODE == TK_HIST0) {
          uint16_t* c = s_hist + tk_bin0(key) * 32 + lane;
          *c = (uint16_t)(*c + 1);
        } else if (MODE == TK_HISTN) {
          if (key >= w.lo && key < w.hi) {
            uint16_t* c = s_hist + (int)((key - w.lo) >> w.shift) * 32 + lane;
            *c = (uint16_t)(*c + 1);
          }
        } else if (MODE == TK_COLLECT) {
          const bool in = key >= w.lo && key < w.hi;
          const uint32_t bal = __ballot_sync(0xffffffffu, in);
          if (in) s_col[w.n_col + __popc(bal & lt)] = make_uint2(key, (uint32_t)(ti * WM_PT_TILE + li));
          w.n_col += __popc(bal);
        } else {
          const bool tie = key == w.T;
          const uint32_t tb = __ballot_sync(0xffffffffu, tie);
          const bool take = key < w.T || (tie && w.n_tie + __popc(tb & lt) < w.quota);
          const uint32_t kb = __ballot_sync(0xffffffffu, take);
          if (take) {
            const int pos = w.n_out + __popc(kb & lt);
            const int idx = ti * WM_PT_TILE + li;
            const int64_t g = (int64_t)b * p.R + idx;
            const float ux = __ldg(&p.dir_x[g]), uy = __ldg(&p.dir_y[g]);
            const int64_t o_idx = ((int64_t)b * p.A + w.ego) * p.k + pos;
            p.rg_index[o_idx] = idx;
            p.rg_type[o_idx] = __ldg(&p.type[g]);
            float* f = p.rg_feat + ((int64_t)b * p.A + w.ego) * 4 * p.k + pos;
            f[0] = fmaf(w.cs, dx, w.sn * dy);
            f[p.k] = fmaf(w.cs, dy, -w.sn * dx);
            f[2 * (int64_t)p.k] = fmaf(w.cs, ux, w.sn * uy);
            f[3 * (int64_t)p.k] = fmaf(w.cs, uy, -w.sn * ux);
          }
          w.n_tie += __popc(tb);
          w.n_out += __popc(kb);
        }
      }
    }
    __syncthreads();                          // everyone is done with this buffer
    if (threadIdx.x == 0 && ti + 2 < ntile) {
      fence_proxy_async();
      mbar_expect_tx(&bars[q & 1], WM_PT_TILE * 8);
      tma_load_1d(s_tiles + (q & 1) * WM_PT_TILE, src + (int64_t)(ti + 2) * WM_PT_TILE, WM_PT_TILE * 8, &bars[q & 1]);
    }
  }
  tile_seq += ntile;
}

// after a histogram pass: fold the lane-private counters, locate the bin holding rank kk
__device__ __forceinline__ void tk_locate(TkWarp& w, uint16_t* s_hist, bool level0) {
  const int lane = threadIdx.x & 31;
  // lane l owns bins 4l .. 4l+3
  int tot[4];
#pragma unroll
  for (int q = 0; q < 4; ++q) {
    const uint16_t* r = s_hist + (lane * 4 + q) * 32;
    int s = 0;
    for (int i = 0; i < 32; ++i) s += r[(i + lane) & 31];     // rotate to spread banks
    tot[q] = s;
  }
  __syncwarp();
  if (level0) {                                // real points = everything but the far bin
    const int far = __shfl_sync(0xffffffffu, tot[3], 31);
    int all = tot[0] + tot[1] + tot[2] + tot[3];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) all += __shfl_xor_sync(0xffffffffu, all, o);
    w.kk = min(w.kk, all - far);
  }
  const int mine = tot[0] + tot[1] + tot[2] + tot[3];
  int inc = mine;
#pragma unroll
  for (int o = 1; o < 32; o <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, o); if (lane >= o) inc += v; }
  const int need = w.kk - w.c_less;            // 1-based rank inside the current range
  const uint32_t has = __ballot_sync(0xffffffffu, inc >= need);
  int bin = 0, below = 0, cnt = 0;
  if (need >= 1 && has) {
    const int L = __ffs(has) - 1;
    int ex = inc - mine, bq = 0, cq = 0, found = 0;
#pragma unroll
    for (int q = 0; q < 4; ++q) if (!found) { if (ex + tot[q] >= need) { bq = q; cq = tot[q]; found = 1; } else ex += tot[q]; }
    bin = __shfl_sync(0xffffffffu, lane * 4 + bq, L);
    below = __shfl_sync(0xffffffffu, ex, L);
    cnt = __shfl_sync(0xffffffffu, cq, L);
  }
  if (w.kk <= 0) { w.in_bin = 0; w.hi = w.lo; return; }
  if (level0) { w.lo = tk_bin0_lo(bin); w.hi = tk_bin0_hi(bin); }
  else { const uint32_t base = w.lo; w.lo = base + ((uint32_t)bin << w.shift); w.hi = min(w.hi, base + ((uint32_t)(bin + 1) << w.shift)); }
  w.c_less += below;
  w.in_bin = cnt;
}

__global__ void __launch_bounds__(TK_THREADS, 1) k_observe_topk(TopkParams p) {
  extern __shared__ __align__(128) unsigned char smem_raw[];
  uint64_t* bars = (uint64_t*)smem_raw;                                  // [2]
  int* s_ego = (int*)(smem_raw + 16);                                    // [TK_WARPS] ego slots of this CTA
  float2* s_tiles = (float2*)(smem_raw + 128);                           // 2 x WM_PT_TILE
  uint16_t* s_hist_all = (uint16_t*)(smem_raw + 128 + 2 * WM_PT_TILE * 8);  // TK_WARPS x 8 KB
  const int b = blockIdx.y, lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  uint16_t* s_hist = s_hist_all + warp * (TK_BINS * 32);
  uint2* s_col = (uint2*)s_hist;
  const int A = p.A, k = p.k;
  const int64_t ro = (int64_t)b * p.row.stride_b;

  // the valid egos [16*blockIdx.x, +16) of the compacted list; invalid ego slots are filled by
  // the CTA that covers the same slot range
  if (threadIdx.x < TK_WARPS) s_ego[threadIdx.x] = -1;
  if (threadIdx.x == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_fence_init(); }
  __syncthreads();
  if (warp == 0) {
    int run = 0;
    const int first = blockIdx.x * TK_WARPS;
    for (int base = 0; base < A; base += 32) {
      const int a = base + lane;
      const bool v = a < A && p.row.valid[ro + a] != 0;
      const uint32_t bal = __ballot_sync(0xffffffffu, v);
      const int ci = run + __popc(bal & ((1u << lane) - 1u));
      if (v && ci >= first && ci < first + TK_WARPS) s_ego[ci - first] = a;
      run += __popc(bal);
    }
  }
  // fill the outputs of invalid ego slots in this CTA's slot range (D10 / D25)
  for (int a = blockIdx.x * TK_WARPS + warp; a < min(A, (int)(blockIdx.x + 1) * TK_WARPS); a += TK_WARPS) {
    if (p.row.valid[ro + a] == 0) {
      for (int j = lane; j < k; j += 32) {
        const int64_t o = ((int64_t)b * A + a) * k + j;
        p.rg_index[o] = -1; p.rg_type[o] = 0;
        float* f = p.rg_feat + ((int64_t)b * A + a) * 4 * k + j;
        f[0] = 0.f; f[k] = 0.f; f[2 * (int64_t)k] = 0.f; f[3 * (int64_t)k] = 0.f;
      }
    }
  }
  __syncthreads();
  if (s_ego[0] < 0) return;                     // no valid ego left for this CTA (uniform)

  TkWarp w;
  const int ego = s_ego[warp];
  w.ego = ego;
  w.active = ego >= 0;
  w.ex = w.ey = 0.f; w.cs = 1.f; w.sn = 0.f;
  if (w.active) { w.ex = p.row.x[ro + ego]; w.ey = p.row.y[ro + ego]; sincosf(p.row.yaw[ro + ego], &w.sn, &w.cs); }
  w.lo = 0; w.hi = 0xffffffffu; w.shift = 0; w.c_less = 0; w.kk = k; w.in_bin = 0;
  w.T = 0; w.quota = 0; w.n_out = 0; w.n_tie = 0; w.n_col = 0; w.refine = false;
  uint32_t tile_seq = 0;

  // ---- pass 1: level-0 histogram ----
  for (int i = lane; i < TK_BINS * 32 / 2; i += 32) ((uint32_t*)s_hist)[i] = 0;
  __syncwarp();
  tk_pass<TK_HIST0>(p, b, w, bars, s_tiles, s_hist, s_col, tile_seq);
  if (w.active) tk_locate(w, s_hist, true);
  // ---- refine while the bin of the k-th key is too large for the collect buffer ----
  for (;;) {
    w.refine = w.active && w.in_bin > TK_CAPB && (w.hi - w.lo) > 1u;
    if (!__syncthreads_or(w.refine ? 1 : 0)) break;
    if (w.refine) {
      const uint32_t span = w.hi - w.lo;
      w.shift = max(0, 32 - __clz(span - 1) - 7);        // (span-1) >> shift < 128
      for (int i = lane; i < TK_BINS * 32 / 2; i += 32) ((uint32_t*)s_hist)[i] = 0;
      __syncwarp();
    }
    tk_pass<TK_HISTN>(p, b, w, bars, s_tiles, s_hist, s_col, tile_seq);
    if (w.refine) tk_locate(w, s_hist, false);
  }
  __syncwarp();
  // ---- pass 2: collect the undecided bin, then exact threshold by bitwise descent ----
  const bool single = w.active && w.in_bin > TK_CAPB;     // one key value with > CAPB ties
  {
    TkWarp wc = w;
    if (single || !w.active || w.kk <= 0) wc.hi = wc.lo;  // nothing to collect
    wc.n_col = 0;
    tk_pass<TK_COLLECT>(p, b, wc, bars, s_tiles, s_hist, s_col, tile_seq);
    w.n_col = wc.n_col;
  }
  __syncwarp();
  if (w.active && w.kk > 0) {
    int r = w.kk - w.c_less;                               // 1-based rank inside [lo, hi)
    if (single) { w.T = w.lo; w.quota = r; }
    else {
      uint32_t pfx = 0, mask = 0;
      const uint32_t diff = w.lo ^ (w.hi - 1u);
      const int top = diff ? 31 - __clz(diff) : -1;        // bits above `top` are common to the range
      if (top < 31) { mask = ~((top >= 0 ? (2u << top) : 1u) - 1u); pfx = w.lo & mask; }
      for (int bit = top; bit >= 0; --bit) {
        const uint32_t m2 = mask | (1u << bit);
        int c0 = 0;
        for (int i = lane; i < w.n_col; i += 32) c0 += ((s_col[i].x & m2) == pfx) ? 1 : 0;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) c0 += __shfl_xor_sync(0xffffffffu, c0, o);
        if (r > c0) { r -= c0; pfx |= 1u << bit; }
        mask = m2;
      }
      w.T = pfx; w.quota = r;                              // r = ties (key == T) to take, in index order
    }
  } else { w.T = 0; w.quota = 0; }
  // ---- pass 3: emit in ascending index order ----
  {
    TkWarp we = w;
    we.n_out = 0; we.n_tie = 0;
    if (!w.active || w.kk <= 0) { we.T = 0; we.quota = 0; }
    tk_pass<TK_EMIT>(p, b, we, bars, s_tiles, s_hist, s_col, tile_seq);
    w.n_out = we.n_out;
  }
  if (w.active) {                                           // D25 padding
    for (int j = w.n_out + lane; j < k; j += 32) {
      const int64_t o = ((int64_t)b * A + ego) * k + j;
      p.rg_index[o] = -1; p.rg_type[o] = 0;
      float* f = p.rg_feat + ((int64_t)b * A + ego) * 4 * k + j;
      f[0] = 0.f; f[k] = 0.f; f[2 * (int64_t)k] = 0.f; f[3 * (int64_t)k] = 0.f;
    }
  }
}

cudaError_t wm_launch_observe_topk(wm_handle* h, const wm_traj& sim, const wm_roadgraph& rg, int t,
                                   int32_t* rg_index, float* rg_feat, int32_t* rg_type, cudaStream_t s) {
  TopkParams p;
  p.row = wm_make_row(sim, t);
  p.A = sim.A; p.R = rg.R; p.k = h->cfg.topk;
  p.pts = h->pts; p.pts_pad = h->pts_pad;
  p.dir_x = rg.dir_x; p.dir_y = rg.dir_y; p.type = rg.type;
  p.rg_index = rg_index; p.rg_feat = rg_feat; p.rg_type = rg_type;
  const size_t smem = 128 + 2 * (size_t)WM_PT_TILE * 8 + (size_t)TK_WARPS * TK_BINS * 32 * 2;
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_observe_topk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
    configured = true;
  }
  dim3 grid((sim.A + TK_WARPS - 1) / TK_WARPS, sim.B);
  k_observe_topk<<<grid, TK_THREADS, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
