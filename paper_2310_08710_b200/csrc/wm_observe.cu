// a6 / a7 default observation: "transforms the location of all other vehicles to
// the agent's own coordinate frame, and sub-samples the roadgraph via distance".
//
// k_observe_hist: HBM-write bound (1.29 GB of features at config 3).  One CTA per (scenario,
// group of egos) stages the H history rows in shared memory once and streams out rows of A
// floats, fully coalesced.
//
// k_observe_topk: exact top-k on the float32 key d2 = fma(dy,dy,dx*dx) (the bit pattern of a
// non-negative float is order preserving; DESIGN.md R-topk).  wm_prepare buckets the valid points of
// a scenario into a uniform grid (k_point_grid).  One 128-thread CTA per ego:
//   0. the square of cells around the ego's cell that holds ~1.6 k points (cell counts only);
//   1. histogram of the keys' top bits over the points of that square (shared-memory atomics)
//      -> bin of the k-th key (repeated on the bin's sub-range only if the bin is too large);
//   2. collect the (key, index) pairs of that bin (<= 512) -> bitwise descent gives the exact k-th
//      key T and the number of ties to take;
//   3. every point outside a square of m rings is farther than m h, so if sqrt(T) < m h the k
//      nearest points of the square are the k nearest of the scenario; otherwise the square grows
//      to hold the disc of radius sqrt(T) and 1-2 run again (T of a subset is never too small);
//   4. mark key < T in a bitmap over the roadgraph indices, key == T in a second one; the first
//      `quota` tie bits in index order join (ties -> lower index, D23);
//   5. emit the set bits in ascending index order (block scan of popcounts) with ego-frame features.
// It reads ~2.3 k of the scenario's 30 k points per ego instead of all of them three times.
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
  if (smem > 48 * 1024) {                          // per-device attribute: set whenever a launch needs it (cheap)
    cudaError_t e = cudaFuncSetAttribute(k_observe_hist, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  dim3 grid((sim.A + HIST_EGOS - 1) / HIST_EGOS, sim.B);
  k_observe_hist<<<grid, 256, smem, s>>>(sim, t, H, hist, hist_valid);
  h->launches++;
  return cudaGetLastError();
}

// ======================================================================================
// top-k roadgraph points
// ======================================================================================
constexpr int PG_THREADS = 1024;

// wm_prepare: bucket the valid points of one scenario (one CTA) into the point grid.
__global__ void __launch_bounds__(PG_THREADS) k_point_grid(const float* x, const float* y, const uint8_t* valid, int R,
                                                           float2* pt_xy, int32_t* pt_idx, int32_t* pt_start, WmPtGrid* pt_grid) {
  __shared__ int s_cnt[WM_PT_CELLS];
  __shared__ float s_red[4][32];
  __shared__ int s_scan[32];
  __shared__ WmPtGrid s_g;
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t o = (int64_t)b * R;
  x += o; y += o; valid += o; pt_xy += o; pt_idx += o;
  pt_start += (int64_t)b * (WM_PT_CELLS + 1);
  // bounding box of the valid points
  float x0 = 3.0e38f, y0 = 3.0e38f, x1 = -3.0e38f, y1 = -3.0e38f;
  for (int i = tid; i < R; i += PG_THREADS)
    if (valid[i] != 0) { const float px = x[i], py = y[i]; x0 = fminf(x0, px); x1 = fmaxf(x1, px); y0 = fminf(y0, py); y1 = fmaxf(y1, py); }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    x0 = fminf(x0, __shfl_xor_sync(0xffffffffu, x0, d)); y0 = fminf(y0, __shfl_xor_sync(0xffffffffu, y0, d));
    x1 = fmaxf(x1, __shfl_xor_sync(0xffffffffu, x1, d)); y1 = fmaxf(y1, __shfl_xor_sync(0xffffffffu, y1, d));
  }
  if (lane == 0) { s_red[0][warp] = x0; s_red[1][warp] = y0; s_red[2][warp] = x1; s_red[3][warp] = y1; }
  for (int c = tid; c < WM_PT_CELLS; c += PG_THREADS) s_cnt[c] = 0;
  __syncthreads();
  if (tid == 0) {
    for (int w = 1; w < PG_THREADS / 32; ++w) {
      x0 = fminf(x0, s_red[0][w]); y0 = fminf(y0, s_red[1][w]); x1 = fmaxf(x1, s_red[2][w]); y1 = fmaxf(y1, s_red[3][w]);
    }
    WmPtGrid g;
    g.pad = 0; g.nvalid = 0;
    if (!(x1 >= x0)) { g.x0 = 0.f; g.y0 = 0.f; g.h = 4.f; g.inv_h = 0.25f; g.nx = 0; g.ny = 0; }
    else {
      const float W = x1 - x0, H = y1 - y0;
      const float h = fmaxf(4.f, fmaxf(W, H) * (1.0001f / WM_PT_NG));
      g.x0 = x0; g.y0 = y0; g.h = h; g.inv_h = 1.f / h;
      g.nx = min(WM_PT_NG, (int)floorf(W / h) + 1); g.ny = min(WM_PT_NG, (int)floorf(H / h) + 1);
    }
    s_g = g;
  }
  __syncthreads();
  const WmPtGrid g = s_g;
  const int ncell = g.nx * g.ny;
  auto cell_of = [&](float px, float py) {
    const int i = min(g.nx - 1, max(0, (int)floorf((px - g.x0) * g.inv_h)));
    const int j = min(g.ny - 1, max(0, (int)floorf((py - g.y0) * g.inv_h)));
    return j * g.nx + i;
  };
  for (int i = tid; i < R; i += PG_THREADS) if (valid[i] != 0) atomicAdd(&s_cnt[cell_of(x[i], y[i])], 1);
  __syncthreads();
  // exclusive scan of the cell counts: each thread owns WM_PT_CELLS / PG_THREADS consecutive cells
  constexpr int PER = WM_PT_CELLS / PG_THREADS;
  int loc[PER], sum = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { loc[q] = sum; sum += s_cnt[tid * PER + q]; }
  int inc = sum;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int v = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += v; }
  if (lane == 31) s_scan[warp] = inc;
  __syncthreads();
  if (warp == 0) {
    int v = s_scan[lane], w = v;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, w, d); if (lane >= d) w += u; }
    s_scan[lane] = w - v;
  }
  __syncthreads();
  const int base = s_scan[warp] + inc - sum;
#pragma unroll
  for (int q = 0; q < PER; ++q) {
    const int c = tid * PER + q;
    s_cnt[c] = base + loc[q];                       // now the running cursor of the cell
    if (c <= ncell) pt_start[c] = base + loc[q];    // cells >= ncell are empty: [ncell] = number of valid points
  }
  if (tid == PG_THREADS - 1) {
    if (ncell == WM_PT_CELLS) pt_start[WM_PT_CELLS] = base + sum;
    WmPtGrid gg = g; gg.nvalid = base + sum;
    pt_grid[b] = gg;
  }
  __syncthreads();
  for (int i = tid; i < R; i += PG_THREADS)
    if (valid[i] != 0) {
      const float px = x[i], py = y[i];
      const int pos = atomicAdd(&s_cnt[cell_of(px, py)], 1);
      pt_xy[pos] = make_float2(px, py);
      pt_idx[pos] = i;
    }
}

cudaError_t wm_launch_point_grid(wm_handle* h, const wm_roadgraph& rg, int b0, int nb, cudaStream_t s) {
  const int64_t o = (int64_t)b0 * rg.R;
  k_point_grid<<<nb, PG_THREADS, 0, s>>>(rg.x + o, rg.y + o, rg.valid + o, rg.R, h->pt_xy + o, h->pt_idx + o,
                                         h->pt_start + (int64_t)b0 * (WM_PT_CELLS + 1), h->pt_grid + b0);
  h->launches++;
  return cudaGetLastError();
}

constexpr int TK_THREADS = 128;              // one CTA per ego
constexpr int TK_BINS = 256;
constexpr int TK_CAP = 512;                  // boundary (key, index) pairs
constexpr int TK_BASE = 119 << 3;            // level-0 bins start at d2 = 2^-8, 3 mantissa bits per bin

struct TopkParams {
  wm_row row;
  int A, R, k, by_distance;
  const float2* pt_xy; const int32_t* pt_idx; const int32_t* pt_start; const WmPtGrid* pt_grid;
  const float *x, *y, *dir_x, *dir_y; const int32_t* type;
  int32_t* rg_index; float* rg_feat; int32_t* rg_type;
};

__device__ __forceinline__ int tk_bin0(uint32_t key) { return min(max((int)(key >> 20) - TK_BASE, 0), TK_BINS - 1); }
__device__ __forceinline__ uint32_t tk_bin0_lo(int bin) { return bin <= 0 ? 0u : (uint32_t)(bin + TK_BASE) << 20; }
__device__ __forceinline__ uint32_t tk_bin0_hi(int bin) { return bin >= TK_BINS - 1 ? 0xffffffffu : (uint32_t)(bin + TK_BASE + 1) << 20; }

struct TkShared {
  uint32_t hist[TK_BINS];
  uint2 col[TK_CAP];
  int scan[TK_THREADS / 32];
  uint32_t lo, hi, T;            // undecided key range [lo, hi); exact threshold
  int shift, c_less, in_bin, n_col, quota, m, count, again, n_tie;
};

// exclusive prefix sum of v over the CTA; total in `total`
__device__ __forceinline__ int tk_block_scan(int v, int* s_scan, int& total) {
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  int inc = v;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
  __syncthreads();                              // s_scan may still be read from a previous call
  if (lane == 31) s_scan[warp] = inc;
  __syncthreads();
  int base = 0; total = 0;
#pragma unroll
  for (int w = 0; w < TK_THREADS / 32; ++w) { const int t = s_scan[w]; if (w < warp) base += t; total += t; }
  return base + inc - v;
}

// warp 0, after a histogram pass: the bin that holds rank `need` (1-based) of the current range
__device__ __forceinline__ void tk_locate(TkShared& S, int need, bool level0) {
  const int lane = threadIdx.x & 31;
  constexpr int PER = TK_BINS / 32;
  int tot[PER], mine = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) { tot[q] = (int)S.hist[lane * PER + q]; mine += tot[q]; }
  int inc = mine;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
  const uint32_t has = __ballot_sync(0xffffffffu, inc >= need);
  const int L = has ? __ffs(has) - 1 : 31;
  int ex = inc - mine, bq = PER - 1, cq = 0, found = 0;
#pragma unroll
  for (int q = 0; q < PER; ++q) if (!found) { if (ex + tot[q] >= need) { bq = q; cq = tot[q]; found = 1; } else ex += tot[q]; }
  const int bin = __shfl_sync(0xffffffffu, lane * PER + bq, L);
  const int below = __shfl_sync(0xffffffffu, ex, L);
  const int cnt = __shfl_sync(0xffffffffu, cq, L);
  if (lane == 0) {
    if (level0) { S.lo = tk_bin0_lo(bin); S.hi = tk_bin0_hi(bin); }
    else { const uint32_t base = S.lo; S.lo = base + ((uint32_t)bin << S.shift); S.hi = min(S.hi, base + ((uint32_t)(bin + 1) << S.shift)); }
    S.c_less += below;
    S.in_bin = cnt;
  }
}

__global__ void __launch_bounds__(TK_THREADS) k_observe_topk(TopkParams p) {
  extern __shared__ __align__(16) uint32_t s_bits[];     // [2][Wd]: key < T; key == T (ties); then [k] indices
  __shared__ TkShared S;
  const int b = blockIdx.y, ego = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int A = p.A, k = p.k, R = p.R, Wd = (R + 31) >> 5;
  uint32_t* bm = s_bits;
  uint32_t* tb = s_bits + Wd;
  int* list = (int*)(s_bits + 2 * Wd);                    // [k] selected indices, ascending
  const int64_t ro = (int64_t)b * p.row.stride_b;
  const int64_t oi = ((int64_t)b * A + ego) * k;          // rg_index / rg_type row
  float* feat = p.rg_feat + ((int64_t)b * A + ego) * 4 * k;
  auto pad_from = [&](int n0) {                           // D10 / D25
    for (int j = n0 + tid; j < k; j += TK_THREADS) {
      p.rg_index[oi + j] = -1; p.rg_type[oi + j] = 0;
      feat[j] = 0.f; feat[k + j] = 0.f; feat[2 * (int64_t)k + j] = 0.f; feat[3 * (int64_t)k + j] = 0.f;
    }
  };
  const WmPtGrid g = p.pt_grid[b];
  const int kk = min(k, g.nvalid);
  if (p.row.valid[ro + ego] == 0 || kk <= 0) { pad_from(0); return; }
  const float ex = p.row.x[ro + ego], ey = p.row.y[ro + ego];
  float sn, cs;
  sincosf(p.row.yaw[ro + ego], &sn, &cs);
  const float2* pxy = p.pt_xy + (int64_t)b * R;
  const int32_t* pidx = p.pt_idx + (int64_t)b * R;
  const int32_t* start = p.pt_start + (int64_t)b * (WM_PT_CELLS + 1);
  const int ci = min(g.nx - 1, max(0, (int)floorf((ex - g.x0) * g.inv_h)));
  const int cj = min(g.ny - 1, max(0, (int)floorf((ey - g.y0) * g.inv_h)));
  // float32 rounding of cell assignments (points and ego): far above an ulp of the coordinates
  const float tol = 2e-3f + 1e-6f * (fabsf(g.x0) + fabsf(g.y0) + (float)(g.nx + g.ny) * g.h);

  // points in the square of m rings around the ego's cell (rows are contiguous runs)
  auto square_count = [&](int m) {                        // warp 0
    const int i0 = max(ci - m, 0), i1 = min(ci + m, g.nx - 1), j0 = max(cj - m, 0), j1 = min(cj + m, g.ny - 1);
    int c = 0;
    for (int j = j0 + lane; j <= j1; j += 32) c += __ldg(start + j * g.nx + i1 + 1) - __ldg(start + j * g.nx + i0);
    return __reduce_add_sync(0xffffffffu, c);
  };
  if (warp == 0) {                                        // 0. the first square: ~1.6 k points
    const int want = min(g.nvalid, kk + (kk * 60) / 100);
    // lanes over m = 0..31 (independent loads), then one m at a time
    int c = 0;
    {
      const int m = lane;
      const int i0 = max(ci - m, 0), i1 = min(ci + m, g.nx - 1), j0 = max(cj - m, 0), j1 = min(cj + m, g.ny - 1);
      for (int j = j0; j <= j1; ++j) c += __ldg(start + j * g.nx + i1 + 1) - __ldg(start + j * g.nx + i0);
    }
    const uint32_t ok = __ballot_sync(0xffffffffu, c >= want);
    int m = ok ? __ffs(ok) - 1 : 32;
    c = __shfl_sync(0xffffffffu, c, m & 31);
    if (!ok) for (;; ++m) { c = square_count(m); if (c >= want || m >= WM_PT_NG) break; }
    if (lane == 0) { S.m = m; S.count = c; }
  }
  for (int i = tid; i < 2 * Wd; i += TK_THREADS) s_bits[i] = 0u;
  if (tid == 0) S.n_tie = 0;
  __syncthreads();

  // one pass over the points of the current square: f(key, sorted position)
  auto for_square = [&](auto&& f) {
    const int m = S.m;
    const int i0 = max(ci - m, 0), i1 = min(ci + m, g.nx - 1), j0 = max(cj - m, 0), j1 = min(cj + m, g.ny - 1);
    for (int j = j0; j <= j1; ++j) {
      const int s0 = __ldg(start + j * g.nx + i0), s1 = __ldg(start + j * g.nx + i1 + 1);
      for (int s = s0 + tid; s < s1; s += TK_THREADS) {
        const float2 pt = __ldg(pxy + s);
        const float dx = __fsub_rn(pt.x, ex), dy = __fsub_rn(pt.y, ey);
        f(__float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx))), s);
      }
    }
  };

  for (;;) {
    // ---- 1. level-0 histogram, bin of the kk-th key ----
    for (int i = tid; i < TK_BINS; i += TK_THREADS) S.hist[i] = 0u;
    if (tid == 0) { S.lo = 0u; S.hi = 0xffffffffu; S.c_less = 0; S.n_col = 0; S.shift = 0; }
    __syncthreads();
    for_square([&](uint32_t key, int) { atomicAdd(&S.hist[tk_bin0(key)], 1u); });
    __syncthreads();
    if (warp == 0) tk_locate(S, kk, true);
    __syncthreads();
    // ---- refine while the bin is too large for the collect buffer ----
    while (S.in_bin > TK_CAP && S.hi - S.lo > 1u) {
      const uint32_t lo = S.lo, hi = S.hi;
      const int shift = max(0, 32 - __clz(hi - lo - 1u) - 8);           // (span - 1) >> shift < 256
      __syncthreads();
      for (int i = tid; i < TK_BINS; i += TK_THREADS) S.hist[i] = 0u;
      if (tid == 0) S.shift = shift;
      __syncthreads();
      for_square([&](uint32_t key, int) { if (key >= lo && key < hi) atomicAdd(&S.hist[(key - lo) >> shift], 1u); });
      __syncthreads();
      if (warp == 0) tk_locate(S, kk - S.c_less, false);
      __syncthreads();
    }
    // ---- 2. collect the bin, then narrow [lo, hi) to one key value on the collected pairs ----
    {
      const uint32_t lo = S.lo, hi = S.hi;
      if (S.in_bin <= TK_CAP && hi - lo > 1u) for_square([&](uint32_t key, int s) {
        if (key >= lo && key < hi) { const int q = atomicAdd(&S.n_col, 1); if (q < TK_CAP) S.col[q] = make_uint2(key, (uint32_t)s); }
      });
      __syncthreads();
    }
    while (S.hi - S.lo > 1u) {                            // in_bin <= TK_CAP here: all of the range is in col
      const uint32_t lo = S.lo, hi = S.hi;
      const int shift = max(0, 32 - __clz(hi - lo - 1u) - 8), n_col = min(S.n_col, TK_CAP);
      __syncthreads();
      for (int i = tid; i < TK_BINS; i += TK_THREADS) S.hist[i] = 0u;
      if (tid == 0) S.shift = shift;
      __syncthreads();
      for (int i = tid; i < n_col; i += TK_THREADS) {
        const uint32_t key = S.col[i].x;
        if (key >= lo && key < hi) atomicAdd(&S.hist[(key - lo) >> shift], 1u);
      }
      __syncthreads();
      if (warp == 0) tk_locate(S, kk - S.c_less, false);
      __syncthreads();
    }
    if (warp == 0) {
      const uint32_t T = S.lo;                            // the kk-th key; ties to take, in index order:
      const int r = kk - S.c_less;
      // ---- 3. is the square large enough? ----
      const int m = S.m;
      const bool all = S.count >= g.nvalid;
      const float reach = (float)m * g.h - tol;
      const float dT = sqrtf(__uint_as_float(T)) * 1.000001f;
      int again = 0;
      if (!all && !(dT < reach)) {
        int m2 = max(m + 1, (int)ceilf((dT + tol) * g.inv_h) + 1);
        m2 = min(m2, WM_PT_NG);
        const int c = square_count(m2);
        if (lane == 0) { S.m = m2; S.count = c; }
        again = 1;
      }
      if (lane == 0) { S.T = T; S.quota = r; S.again = again; }   // r = ties (key == T) to take, in index order
    }
    __syncthreads();
    if (!S.again) break;
    __syncthreads();
  }

  // ---- 4. mark the selected points over the roadgraph indices ----
  const uint32_t T = S.T;
  for_square([&](uint32_t key, int s) {
    if (key <= T) {
      const int idx = __ldg(pidx + s);
      atomicOr((key < T ? bm : tb) + (idx >> 5), 1u << (idx & 31));
      if (key == T) atomicAdd(&S.n_tie, 1);
    }
  });
  __syncthreads();
  // The first `quota` ties in index order join the selection.  Nearly always every tie is taken
  // (n_tie == quota); otherwise the tie words are trimmed in index order, word r * 128 + tid in round r.
  const int quota = S.quota, n_tie = S.n_tie;
  const bool trim = n_tie > quota;
  if (trim) {
    const int rounds = (Wd + TK_THREADS - 1) / TK_THREADS;
    int base = 0;
    for (int r = 0; r < rounds; ++r) {
      const int w = r * TK_THREADS + tid;
      uint32_t t = w < Wd ? tb[w] : 0u;
      const int n = __popc(t);
      int tot_r;
      const int left = quota - (base + tk_block_scan(n, S.scan, tot_r));
      if (left < n) { for (int drop = n - max(left, 0); drop > 0; --drop) t &= ~(0x80000000u >> __clz(t)); }   // keep the lowest bits
      if (w < Wd) bm[w] |= t;
      base += tot_r;
    }
    __syncthreads();
  }
  // ---- 5. the set bits in ascending index order -> list, then features with coalesced stores ----
  // Each warp owns a contiguous quarter of the words, its lanes interleaved over them (the selected
  // points cluster in index ranges - polylines near the ego - and this spreads a cluster over the
  // lanes); positions come from one exchange of the warp totals and shuffle scans, no block barrier.
  const int Q = (Wd + TK_THREADS / 32 - 1) / (TK_THREADS / 32), wb = warp * Q, we = min(wb + Q, Wd);
  {
    int c = 0;
    for (int w = wb + lane; w < we; w += 32) {
      uint32_t v = bm[w];
      if (!trim) { v |= tb[w]; bm[w] = v; }
      c += __popc(v);
    }
    c = __reduce_add_sync(0xffffffffu, c);
    if (lane == 0) S.scan[warp] = c;
  }
  __syncthreads();
  int run = 0, n_out = 0;
#pragma unroll
  for (int w = 0; w < TK_THREADS / 32; ++w) { const int t = S.scan[w]; if (w < warp) run += t; n_out += t; }
  for (int w0 = wb; w0 < we; w0 += 32) {
    const int w = w0 + lane;
    uint32_t bits = w < we ? bm[w] : 0u;
    const int n = __popc(bits);
    int inc = n;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
    int pos = run + inc - n;
    while (bits) { if (pos < k) list[pos] = w * 32 + __ffs(bits) - 1; ++pos; bits &= bits - 1; }
    run += __shfl_sync(0xffffffffu, inc, 31);
  }
  __syncthreads();
  n_out = min(n_out, k);
  const float *gx = p.x + (int64_t)b * R, *gy = p.y + (int64_t)b * R, *gdx = p.dir_x + (int64_t)b * R, *gdy = p.dir_y + (int64_t)b * R;
  const int32_t* gt = p.type + (int64_t)b * R;
  if (p.by_distance) {
    // WM_TOPK_BY_DISTANCE (D44): the selected points by ascending (key, index) - a bitonic sort of
    // (key bits << 32 | index) in shared memory, padded to a power of two with all-ones
    unsigned long long* sk = (unsigned long long*)(s_bits + ((2 * Wd + k + 1) & ~1));
    int P = 1;
    while (P < n_out) P <<= 1;
    for (int j = tid; j < P; j += TK_THREADS) {
      unsigned long long kv = ~0ull;
      if (j < n_out) {
        const int idx = list[j];
        const float dx = __fsub_rn(__ldg(gx + idx), ex), dy = __fsub_rn(__ldg(gy + idx), ey);
        kv = ((unsigned long long)__float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx))) << 32) | (unsigned)idx;
      }
      sk[j] = kv;
    }
    __syncthreads();
    for (int len = 2; len <= P; len <<= 1)
      for (int st = len >> 1; st > 0; st >>= 1) {
        for (int i = tid; i < (P >> 1); i += TK_THREADS) {
          const int lo = ((i & ~(st - 1)) << 1) | (i & (st - 1)), hi = lo | st;
          const bool up = (lo & len) == 0;
          const unsigned long long a = sk[lo], c = sk[hi];
          if ((a > c) == up) { sk[lo] = c; sk[hi] = a; }
        }
        __syncthreads();
      }
    for (int j = tid; j < n_out; j += TK_THREADS) list[j] = (int)(unsigned)(sk[j] & 0xffffffffull);
    __syncthreads();
  }
  for (int j = tid; j < n_out; j += TK_THREADS) {
    const int idx = list[j];
    const float dx = __fsub_rn(__ldg(gx + idx), ex), dy = __fsub_rn(__ldg(gy + idx), ey);
    const float ux = __ldg(gdx + idx), uy = __ldg(gdy + idx);
    p.rg_index[oi + j] = idx;
    p.rg_type[oi + j] = __ldg(gt + idx);
    feat[j] = fmaf(cs, dx, sn * dy);
    feat[k + j] = fmaf(cs, dy, -sn * dx);
    feat[2 * (int64_t)k + j] = fmaf(cs, ux, sn * uy);
    feat[3 * (int64_t)k + j] = fmaf(cs, uy, -sn * ux);
  }
  pad_from(n_out);
}

cudaError_t wm_launch_observe_topk(wm_handle* h, const wm_traj& sim, const wm_roadgraph& rg, int t,
                                   int32_t* rg_index, float* rg_feat, int32_t* rg_type, cudaStream_t s) {
  TopkParams p;
  p.row = wm_make_row(sim, t);
  p.A = sim.A; p.R = rg.R; p.k = h->cfg.topk; p.by_distance = h->cfg.topk_order == WM_TOPK_BY_DISTANCE;
  p.pt_xy = h->pt_xy; p.pt_idx = h->pt_idx; p.pt_start = h->pt_start; p.pt_grid = h->pt_grid;
  p.x = rg.x; p.y = rg.y; p.dir_x = rg.dir_x; p.dir_y = rg.dir_y; p.type = rg.type;
  p.rg_index = rg_index; p.rg_feat = rg_feat; p.rg_type = rg_type;
  size_t smem = (2 * (size_t)((rg.R + 31) / 32) + (size_t)h->cfg.topk) * sizeof(uint32_t);
  if (p.by_distance) {                                        // + the sort keys: 8 B x the power of two >= k
    size_t P = 1;
    while (P < (size_t)h->cfg.topk) P <<= 1;
    smem = ((smem + 7) & ~(size_t)7) + P * sizeof(unsigned long long);
  }
  if (smem > 200 * 1024) return cudaErrorInvalidValue;       // R > 819 200 points per scenario
  if (smem > 40 * 1024) {                                     // per-device attribute: set whenever a launch needs it (cheap)
    cudaError_t e = cudaFuncSetAttribute(k_observe_topk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  k_observe_topk<<<dim3(sim.A, sim.B), TK_THREADS, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
