// a6 / a7 default observation: "transforms the location of all other vehicles to
// the agent's own coordinate frame, and sub-samples the roadgraph via distance".
//
// k_observe_hist: HBM-write bound (1.29 GB of features at config 3).  One CTA per (scenario,
// group of egos) stages the H history rows in shared memory once and streams out rows of A
// floats, fully coalesced.
//
// k_observe_topk: exact top-k on the float32 key d2 = fma(dy,dy,dx*dx) (the bit pattern of a
// non-negative float is order preserving; DESIGN.md R-topk).  wm_prepare buckets the valid points of
// a scenario into a uniform grid (k_point_grid).  One 128-thread CTA per ego (9 CTAs per SM; 256 threads
// were measured slower: the phases are short and a barrier then waits on more warps):
//   0. the square of cells around the ego's cell that holds ~1.6 k points (cell counts only);
//   1. ONE pass over the points of that square: keys -> shared memory (squares of up to 3072 points; the
//      later passes read them there), histogram of their top bits (1024 bins: exponent + 5 mantissa bits,
//      shared-memory atomics) -> bin of the k-th key (a 256-bin pass on the bin's sub-range only if it
//      holds more than 512 keys);
//   2. collect the keys of that bin (<= 512) -> 8-bit descents give the exact k-th key T, the number of
//      keys equal to it and the number of those to take;
//   3. every point outside a square of m rings is farther than m h, so if sqrt(T) < m h the k
//      nearest points of the square are the k nearest of the scenario; otherwise the square grows
//      to hold the disc of radius sqrt(T) and 1-2 run again (T of a subset is never too small);
//   4. mark key < T (and == T when every tie is taken, the usual case) in a bitmap over the roadgraph
//      indices and append the index to an unordered list (warp-aggregated); otherwise the ties go to a
//      bitmap of their own and the first `quota` of them in index order join (ties -> lower index, D23);
//   5. ascending index order without walking the bitmap: prefix sums of the words' popcounts, then every
//      listed index finds its rank with one popc and is stored at that place; ego-frame features follow.
// It reads ~2.3 k of the scenario's 30 k points per ego once instead of all of them three times.
#include <string.h>

#include <mutex>

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
constexpr int TK_BINS = 1024;                // level-0 bins: exponent + 5 mantissa bits
constexpr int TK_SH0 = 18;
constexpr int TK_CAP = 512;                  // boundary (key, position) pairs
constexpr int TK_BASE = 119 << 5;            // level-0 bins start at d2 = 2^-8
constexpr int TK_KEYS = 2560;                // keys of the square kept in shared memory (larger squares recompute them)

struct TopkParams {
  wm_row row;
  int A, R, k, by_distance;
  const float2* pt_xy; const int32_t* pt_idx; const int32_t* pt_start; const WmPtGrid* pt_grid;
  const float *x, *y, *dir_x, *dir_y; const int32_t* type;
  int32_t* rg_index; float* rg_feat; int32_t* rg_type;
};

__device__ __forceinline__ int tk_bin0(uint32_t key) { return min(max((int)(key >> TK_SH0) - TK_BASE, 0), TK_BINS - 1); }
__device__ __forceinline__ uint32_t tk_bin0_lo(int bin) { return bin <= 0 ? 0u : (uint32_t)(bin + TK_BASE) << TK_SH0; }
__device__ __forceinline__ uint32_t tk_bin0_hi(int bin) { return bin >= TK_BINS - 1 ? 0xffffffffu : (uint32_t)(bin + TK_BASE + 1) << TK_SH0; }

struct TkShared {
  int scan[TK_THREADS / 32];
  uint32_t lo, hi, T;            // undecided key range [lo, hi); exact threshold
  int shift, c_less, in_bin, n_col, quota, m, count, again, n_tie, n_sel, n_rows;
  int row_s0[WM_PT_NG];          // the square's rows of cells: first sorted point of the row,
  int row_base[WM_PT_NG + 1];    //   and its position in the square's own numbering (prefix counts)
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

// warp 0, after a histogram pass over `nbins` bins: the bin that holds rank `need` (1-based) of the current range
template <int NBINS>
__device__ __forceinline__ void tk_locate(TkShared& S, const uint32_t* hist, int need, bool level0) {
  const int lane = threadIdx.x & 31;
  constexpr int per = NBINS >> 5;
  int mine = 0;
  {
    const uint4* h4 = (const uint4*)(hist + lane * per);
#pragma unroll
    for (int q = 0; q < per / 4; ++q) { const uint4 v = h4[q]; mine += (int)(v.x + v.y + v.z + v.w); }
  }
  int inc = mine;
#pragma unroll
  for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
  const uint32_t has = __ballot_sync(0xffffffffu, inc >= need);
  const int L = has ? __ffs(has) - 1 : 31;
  if (lane == L) {
    int ex = inc - mine, bin = lane * per + per - 1, cnt = 0;
    for (int q = 0; q < per; ++q) {
      const int t = (int)hist[lane * per + q];
      if (ex + t >= need || q == per - 1) { bin = lane * per + q; cnt = t; break; }
      ex += t;
    }
    if (level0) { S.lo = tk_bin0_lo(bin); S.hi = tk_bin0_hi(bin); }
    else { const uint32_t base = S.lo; S.lo = base + ((uint32_t)bin << S.shift); S.hi = min(S.hi, base + ((uint32_t)(bin + 1) << S.shift)); }
    S.c_less += ex;
    S.in_bin = cnt;
  }
}

__global__ void __launch_bounds__(TK_THREADS) k_observe_topk(TopkParams p) {
  extern __shared__ __align__(16) uint32_t s_dyn[];
  __shared__ TkShared S;
  const int b = blockIdx.y, ego = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int A = p.A, k = p.k, R = p.R, Wd = (R + 31) >> 5;
  const int Wd4 = (Wd + 3) & ~3;                          // 16-byte aligned pieces
  uint32_t* bm = s_dyn;                                   // [Wd] key < T (and the ties that join)
  uint32_t* tb = bm + Wd4;                                // [Wd] key == T (only when some ties stay out); later:
  uint32_t* pre = tb;                                     //   [Wd] set bits of bm before word w
  uint32_t* keys = tb + Wd4;                              // [max(TK_KEYS, k)] keys of the square, in its order; later:
  int* list = (int*)keys;                                 //   [k] the selected indices, ascending
  uint32_t* const hist = keys + ((max(TK_KEYS, k) + 3) & ~3);   // [TK_BINS] histogram, [TK_CAP] keys of the k-th key's bin; later:
  uint32_t* const col = hist + TK_BINS;
  int* sel = (int*)hist;                                  //   [k] the selected indices as they were found
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
  // the rows of the square of m rings in shared memory: a pass then runs over the square's points as one
  // flat range instead of row by row (warp 0)
  auto set_rows = [&](int m) {
    const int i0 = max(ci - m, 0), i1 = min(ci + m, g.nx - 1), j0 = max(cj - m, 0), j1 = min(cj + m, g.ny - 1);
    const int nr = j1 - j0 + 1;                           // <= WM_PT_NG = 64
    int run = 0;
#pragma unroll
    for (int r0 = 0; r0 < WM_PT_NG; r0 += 32) {
      const int r = r0 + lane;
      int s0 = 0, c = 0;
      if (r < nr) { s0 = __ldg(start + (j0 + r) * g.nx + i0); c = __ldg(start + (j0 + r) * g.nx + i1 + 1) - s0; }
      int inc = c;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { const int u = __shfl_up_sync(0xffffffffu, inc, d); if (lane >= d) inc += u; }
      S.row_s0[r] = s0; S.row_base[r] = run + inc - c;
      run += __shfl_sync(0xffffffffu, inc, 31);
    }
    if (lane == 0) { S.row_base[WM_PT_NG] = run; S.m = m; S.count = run; S.n_rows = nr; }
  };
  if (warp == 0) {                                        // 0. the first square: ~1.6 k points
    const int want = min(g.nvalid, kk + (kk * 60) / 100);
    // lanes over m = 0..31 (independent loads), then one m at a time
    // m = 0..15 first, two lanes per m (the rows of a square split in halves: independent loads)
    int c = 0;
    {
      const int m = lane >> 1;
      const int i0 = max(ci - m, 0), i1 = min(ci + m, g.nx - 1), j0 = max(cj - m, 0), j1 = min(cj + m, g.ny - 1);
      for (int j = j0 + (lane & 1); j <= j1; j += 2) c += __ldg(start + j * g.nx + i1 + 1) - __ldg(start + j * g.nx + i0);
      c += __shfl_xor_sync(0xffffffffu, c, 1);
    }
    const uint32_t ok = __ballot_sync(0xffffffffu, c >= want);
    int m = ok ? (__ffs(ok) - 1) >> 1 : 16;
    if (!ok) for (;; ++m) { c = square_count(m); if (c >= want || m >= WM_PT_NG) break; }
    set_rows(m);
  }
  for (int i = tid; i < 2 * Wd4; i += TK_THREADS) s_dyn[i] = 0u;
  if (tid == 0) { S.n_tie = 0; S.n_sel = 0; }
  __syncthreads();

  // One pass over the points of the current square, numbered 0 .. count - 1 row after row: f(key, position).
  // The first pass of a square (fill) computes the keys, a warp per row of cells, and keeps them in shared
  // memory when the square fits; the later ones read them there as one flat range.
  bool cached = false;
  auto key_at = [&](int s) {
    const float2 pt = __ldg(pxy + s);
    const float dx = __fsub_rn(pt.x, ex), dy = __fsub_rn(pt.y, ey);
    return __float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
  };
  auto for_square = [&](bool fill, auto&& f) {
    if (cached && !fill) { const int count = S.count; for (int j = tid; j < count; j += TK_THREADS) f(keys[j], j); return; }
    const int nr = S.n_rows;
    for (int r = warp; r < nr; r += TK_THREADS / 32) {
      const int s0 = S.row_s0[r], base = S.row_base[r], cnt = S.row_base[r + 1] - base;
      // four points of the row in flight per lane: the loads do not depend on one another
      for (int i0 = lane; i0 < cnt; i0 += 128) {
        float2 pt[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) pt[u] = __ldg(pxy + s0 + min(i0 + 32 * u, cnt - 1));
#pragma unroll
        for (int u = 0; u < 4; ++u) {
          const int i = i0 + 32 * u;
          if (i < cnt) {
            const float dx = __fsub_rn(pt[u].x, ex), dy = __fsub_rn(pt[u].y, ey);
            const uint32_t key = __float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx)));
            if (cached) keys[base + i] = key;
            f(key, base + i);
          }
        }
      }
    }
  };

  for (;;) {
    // ---- 1. level-0 histogram, bin of the kk-th key ----
    for (int i = tid; i < TK_BINS; i += TK_THREADS) hist[i] = 0u;
    if (tid == 0) { S.lo = 0u; S.hi = 0xffffffffu; S.c_less = 0; S.n_col = 0; S.shift = 0; }
    cached = S.count <= TK_KEYS;
    __syncthreads();
    for_square(true, [&](uint32_t key, int) { atomicAdd(&hist[tk_bin0(key)], 1u); });
    __syncthreads();
    if (warp == 0) tk_locate<TK_BINS>(S, hist, kk, true);
    __syncthreads();
    // ---- refine while the bin is too large for the collect buffer ----
    while (S.in_bin > TK_CAP && S.hi - S.lo > 1u) {
      const uint32_t lo = S.lo, hi = S.hi;
      const int shift = max(0, 32 - __clz(hi - lo - 1u) - 8);           // (span - 1) >> shift < 256
      __syncthreads();
      for (int i = tid; i < 256; i += TK_THREADS) hist[i] = 0u;
      if (tid == 0) S.shift = shift;
      __syncthreads();
      for_square(false, [&](uint32_t key, int) { if (key >= lo && key < hi) atomicAdd(&hist[(key - lo) >> shift], 1u); });
      __syncthreads();
      if (warp == 0) tk_locate<256>(S, hist, kk - S.c_less, false);
      __syncthreads();
    }
    // ---- 2. collect the bin, then narrow [lo, hi) to one key value on the collected keys ----
    {
      const uint32_t lo = S.lo, hi = S.hi;
      if (S.in_bin <= TK_CAP && hi - lo > 1u) for_square(false, [&](uint32_t key, int s) {
        if (key >= lo && key < hi) { const int q = atomicAdd(&S.n_col, 1); if (q < TK_CAP) col[q] = key; }
      });
      __syncthreads();
    }
    {                                                     // in_bin <= TK_CAP here: all of the range is in col
      // the kk-th key by counting: the collected key with c smaller and e equal ones, c < need <= c + e
      const bool open_range = S.hi - S.lo > 1u;
      const int n_col = open_range ? min(S.n_col, TK_CAP) : 0, need = kk - S.c_less;
      __syncthreads();                                    // everyone has read the range before a winner rewrites it
      for (int i = tid; i < n_col; i += TK_THREADS) {
        const uint32_t mine = col[i];
        int c = 0, e = 0;
        for (int j = 0; j < n_col; ++j) { const uint32_t o = col[j]; c += o < mine; e += o == mine; }
        if (c < need && need <= c + e) { S.lo = mine; S.hi = mine + 1u; S.c_less = kk - need + c; S.in_bin = e; }   // every writer stores the same values
      }
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
        set_rows(m2);
        again = 1;
      }
      if (lane == 0) { S.T = T; S.quota = r; S.again = again; S.n_tie = S.in_bin; }   // r = ties (key == T) to take, in index order; in_bin = all ties
    }
    __syncthreads();
    if (!S.again) break;
    __syncthreads();
  }

  // ---- 4. mark the selected points over the roadgraph indices and list them as they come ----
  // Nearly always every tie is taken (n_tie == quota); otherwise the ties go to a bitmap of their own, are
  // trimmed in index order and join afterwards.
  const uint32_t T = S.T;
  const int quota = S.quota;
  const bool trim = S.n_tie > quota;
  {
    const int nr = S.n_rows;
    for (int r = warp; r < nr; r += TK_THREADS / 32) {        // a warp per row of cells; appends are warp-aggregated
      const int s0 = S.row_s0[r], base = S.row_base[r], cnt = S.row_base[r + 1] - base;
      for (int ib = 0; ib < cnt; ib += 32) {
        const int i = ib + lane;
        bool take = false, tie = false;
        const int idx = __ldg(pidx + s0 + min(i, cnt - 1));        // requested before the key decides: no dependent miss
        if (i < cnt) {
          const uint32_t key = cached ? keys[base + i] : key_at(s0 + i);
          take = key < T || (key == T && !trim);
          tie = key == T && trim;
        }
        const uint32_t bal = __ballot_sync(0xffffffffu, take);
        if (take || tie) {
          atomicOr((take ? bm : tb) + (idx >> 5), 1u << (idx & 31));
          if (take) {
            int q0 = 0;
            const int leader = __ffs(bal) - 1;
            if (lane == leader) q0 = atomicAdd(&S.n_sel, __popc(bal));
            q0 = __shfl_sync(bal, q0, leader);
            const int q = q0 + __popc(bal & ((1u << lane) - 1u));
            if (q < k) sel[q] = idx;
          }
        }
      }
    }
  }
  __syncthreads();
  if (trim) {
    // the first `quota` ties in index order join: word r * TK_THREADS + tid in round r
    const int rounds = (Wd + TK_THREADS - 1) / TK_THREADS;
    int basec = 0;
    for (int r = 0; r < rounds; ++r) {
      const int w = r * TK_THREADS + tid;
      uint32_t t = w < Wd ? tb[w] : 0u;
      const int n = __popc(t);
      int tot_r;
      const int left = quota - (basec + tk_block_scan(n, S.scan, tot_r));
      if (left < n) { for (int drop = n - max(left, 0); drop > 0; --drop) t &= ~(0x80000000u >> __clz(t)); }   // keep the lowest bits
      if (w < Wd) {
        bm[w] |= t;
        while (t) { const int q = atomicAdd(&S.n_sel, 1); if (q < k) sel[q] = w * 32 + __ffs(t) - 1; t &= t - 1; }
      }
      basec += tot_r;
    }
    __syncthreads();
  }
  // ---- 5. rank of every selected index = set bits of bm below it: word prefix sums, then one popc each ----
  {
    const int PW = (Wd + TK_THREADS - 1) / TK_THREADS;      // consecutive words per thread
    int c = 0;
    for (int q = 0; q < PW; ++q) { const int w = tid * PW + q; if (w < Wd) c += __popc(bm[w]); }
    int tot;
    int run = tk_block_scan(c, S.scan, tot);
    for (int q = 0; q < PW; ++q) { const int w = tid * PW + q; if (w < Wd) { pre[w] = (uint32_t)run; run += __popc(bm[w]); } }
  }
  __syncthreads();                                          // keys are dead from here on: list takes their place
  const int n_out = min(S.n_sel, k);
  for (int i = tid; i < n_out; i += TK_THREADS) {
    const int idx = sel[i], w = idx >> 5;
    const int pos = (int)pre[w] + __popc(bm[w] & ((1u << (idx & 31)) - 1u));
    if (pos < k) list[pos] = idx;
  }
  __syncthreads();
  const float *gx = p.x + (int64_t)b * R, *gy = p.y + (int64_t)b * R, *gdx = p.dir_x + (int64_t)b * R, *gdy = p.dir_y + (int64_t)b * R;
  const int32_t* gt = p.type + (int64_t)b * R;
  if (p.by_distance) {
    // WM_TOPK_BY_DISTANCE (D44): the selected points by ascending (key, index) - a bitonic sort of
    // (key bits << 32 | index) in shared memory, padded to a power of two with all-ones
    unsigned long long* sk = (unsigned long long*)(hist + ((max(TK_BINS + TK_CAP, k) + 1) & ~1));
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
  const size_t kq = (size_t)h->cfg.topk;
  const size_t hcq = (size_t)(TK_BINS + TK_CAP), wd4 = ((size_t)((rg.R + 31) / 32) + 3) & ~(size_t)3;
  size_t smem = (2 * wd4 + (((kq > (size_t)TK_KEYS ? kq : (size_t)TK_KEYS) + 3) & ~(size_t)3) + (((kq > hcq ? kq : hcq) + 1) & ~(size_t)1)) * sizeof(uint32_t);
  if (p.by_distance) {                                        // + the sort keys: 8 B x the power of two >= k
    size_t P = 1;
    while (P < (size_t)h->cfg.topk) P <<= 1;
    smem += P * sizeof(unsigned long long);
  }
  if (smem > 200 * 1024) return cudaErrorInvalidValue;       // R > ~500 000 points per scenario
  if (smem > 24 * 1024) {                                     // per-device attribute: set whenever a launch needs it (cheap)
    cudaError_t e = cudaFuncSetAttribute(k_observe_topk, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  k_observe_topk<<<dim3(sim.A, sim.B), TK_THREADS, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}

// ======================================================================================
// wm_observe_topk_static: the top-k observation for callers that must not allocate
// ======================================================================================
// The regular route (wm_create -> wm_prepare -> wm_observe) keeps the bucketed roadgraph points in
// buffers it obtains with cudaMalloc.  Some users of this library cannot do that where they call it:
//   - a simulator step running inside a training job whose framework allocator has already taken
//     (nearly) all of the HBM for its own pool, so a raw cudaMalloc from a library fails or fragments it;
//   - a control / planning loop with a fixed memory budget that forbids allocation after start-up;
//   - a latency-sensitive loop that cannot afford cudaMalloc / cudaFree, which synchronise the device.
// For them the bucketed points live in the file-scope array below, reserved in the library's image: every
// GPU that loads libwm_b200.so holds its WM_STATIC_BYTES (about 13 MiB) from then until the process exits,
// whether or not this entry point is ever called.  The entry point needs no wm_handle (creating one
// allocates) and calls no cudaMalloc / cudaFree / stream or event creation: two kernel launches
// (k_point_grid, k_observe_topk - the same kernels and arithmetic as wm_prepare + wm_observe) on the
// caller's stream.
//
// Layout of the array (bytes): [pt_xy: MAX_POINTS float2][pt_idx: MAX_POINTS int32]
//                              [pt_start: MAX_B x (WM_PT_CELLS + 1) int32][pt_grid: MAX_B WmPtGrid]
// A call with B scenarios of R points uses the first B * R entries of pt_xy / pt_idx and the first B rows of
// the other two.  Nothing in it has to start at zero: k_point_grid rewrites every word that k_observe_topk
// reads for the same (B, R) (cell starts 0 .. ncell, the grid descriptor, the nvalid bucketed points), so
// the previous call's contents are simply overwritten or left unread.
//
// In HOST code the name g_wm_static_obs is only a stand-in the runtime knows the symbol by, not a device
// address; the address comes from cudaGetSymbolAddress, asked once per device with that device current.
constexpr size_t WM_ST_OFF_IDX = (size_t)WM_STATIC_MAX_POINTS * sizeof(float2);
constexpr size_t WM_ST_OFF_START = WM_ST_OFF_IDX + (size_t)WM_STATIC_MAX_POINTS * sizeof(int32_t);
constexpr size_t WM_ST_OFF_GRID = (WM_ST_OFF_START + (size_t)WM_STATIC_MAX_B * (WM_PT_CELLS + 1) * sizeof(int32_t) + 255) / 256 * 256;
constexpr size_t WM_STATIC_BYTES = WM_ST_OFF_GRID + (size_t)WM_STATIC_MAX_B * sizeof(WmPtGrid);
static_assert(WM_ST_OFF_IDX % 256 == 0 && WM_ST_OFF_START % 256 == 0, "pieces of the static scratch stay 256-byte aligned");

static __device__ __align__(256) unsigned char g_wm_static_obs[WM_STATIC_BYTES];

constexpr int WM_STATIC_MAX_DEVICES = 64;
static std::mutex g_wm_static_mu;
static unsigned char* g_wm_static_ptr[WM_STATIC_MAX_DEVICES];     // device address of the array on each device, once known

// Set-up, once per device: the current device's address of the array.  Allocates nothing.
static int wm_static_base(unsigned char** out) {
  int dev = -1;
  WM_CUDA(cudaGetDevice(&dev));
  if (dev < 0 || dev >= WM_STATIC_MAX_DEVICES) return WM_ERR_UNSUPPORTED;
  std::lock_guard<std::mutex> lock(g_wm_static_mu);
  if (!g_wm_static_ptr[dev]) {
    int major = 0;
    WM_CUDA(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
    if (major != 10) return WM_ERR_UNSUPPORTED;                   // sm_100a kernels only; no fallback
    unsigned char* ptr = nullptr;
    WM_CUDA(cudaGetSymbolAddress((void**)&ptr, g_wm_static_obs));
    if (!ptr) return WM_ERR_CUDA;
    g_wm_static_ptr[dev] = ptr;
  }
  *out = g_wm_static_ptr[dev];
  return WM_OK;
}

extern "C" int wm_observe_topk_static(const wm_traj* sim, const wm_roadgraph* rg, int32_t t, int32_t topk, int32_t topk_order,
                                      int32_t* rg_index, float* rg_feat, int32_t* rg_type, void* stream) {
  if (!sim || !rg || !rg_index || !rg_feat || !rg_type) return WM_ERR_ARG;
  if (sim->B < 1 || sim->A < 1 || sim->T < 1 || rg->B != sim->B || rg->R < 1 || t < 0 || t >= sim->T) return WM_ERR_ARG;
  if (!sim->x || !sim->y || !sim->yaw || !sim->valid || !rg->x || !rg->y || !rg->dir_x || !rg->dir_y || !rg->type || !rg->valid) return WM_ERR_ARG;
  if (topk_order != WM_TOPK_BY_INDEX && topk_order != WM_TOPK_BY_DISTANCE) return WM_ERR_ARG;
  if (sim->B > WM_STATIC_MAX_B || (int64_t)sim->B * rg->R > WM_STATIC_MAX_POINTS) return WM_ERR_TOO_LARGE;   // the array is what it is
  if (sim->A > 1024 || topk < 1 || topk > rg->R) return WM_ERR_UNSUPPORTED;
  unsigned char* base = nullptr;
  const int rc = wm_static_base(&base);
  if (rc != WM_OK) return rc;
  // the launchers of the regular path read only these fields of a handle: a zeroed one on the stack
  // pointing into the static array runs the very same launches
  wm_handle tmp;
  memset(&tmp, 0, sizeof(tmp));
  tmp.cfg.topk = topk; tmp.cfg.topk_order = topk_order;
  tmp.pt_xy = (float2*)base; tmp.pt_idx = (int32_t*)(base + WM_ST_OFF_IDX);
  tmp.pt_start = (int32_t*)(base + WM_ST_OFF_START); tmp.pt_grid = (WmPtGrid*)(base + WM_ST_OFF_GRID);
  WM_CUDA(wm_launch_point_grid(&tmp, *rg, 0, rg->B, (cudaStream_t)stream));
  WM_CUDA(wm_launch_observe_topk(&tmp, *sim, *rg, t, rg_index, rg_feat, rg_type, (cudaStream_t)stream));
  return WM_OK;
}
