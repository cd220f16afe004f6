// a8 closed-loop rollout ("Rollout ... faster than running Step 80 times"), fused
// into TWO kernels that run back to back in one CUDA graph:
//
//   k_rollout_dyn      one thread per (scenario, agent): the serial chain of n_steps successor states
//                      (a1/a2, shared arithmetic with k_step: wm_device.cuh), log playback (D8), sim rows
//                      -> HBM, log divergence (a5) and ADE.  The successor state depends on the state and
//                      the action only, never on a metric, so the whole trajectory is laid down first.
//                      HBM bound: ~51 B per agent-step.
//   k_rollout_metrics  one CTA per (scenario, block of S steps), scheduled scenario-major: overlap (a3)
//                      and offroad (a4) of the block's rows and the any-flags.  Every (scenario, block)
//                      is independent, so nothing in this kernel is serial; consecutive CTAs belong to
//                      the same scenario, so only ~B/10 scenarios are in flight at a time and their
//                      search data (cell headers, pair records) stays in L2 instead of being re-fetched
//                      from HBM (the single-kernel version of round 1 kept 740 scenarios in flight:
//                      L2 hit rate 29 %, DRAM traffic 1.96 x the compulsory bytes).
//
//   metrics kernel, per CTA:
//   phase A  all threads          : rows of the block -> per-step slots in shared memory (centre, sin/cos,
//                                   half extents); then one thread per agent: its bounding box over the
//                                   block into a spatial hash (warps 0-3, while the others start phase B)
//   phase B  warp tasks, any warp : (agent, S steps) -> its 4 S box corners, one per lane: candidate
//                                   walk of the corner's grid cell (wm_grid.cuh).  The lanes of a task
//                                   follow one agent through consecutive steps, so they walk the
//                                   same few cells: equal list lengths, the same cache lines.  Corners
//                                   off the grid or in a crowded cell are searched by the whole warp;
//                                   (32 agents) -> overlap flags of the block: each lane walks the
//                                   3 x 3 hash cells around its agent and lists the pairs whose
//                                   block bounding boxes meet; then one lane per (pair, step) runs
//                                   the circle and separating-axis tests
//   phase C  all threads          : metric rows of the block -> HBM, any-flags
//
// Overlap broad phase, once per block: an agent is hashed by the 24 m cell of the centre of its
// bounding box over the block (linked lists in shared memory).  Two agents whose boxes (inflated by
// the circumradius) have half extents <= 11.7 m can only overlap from adjacent cells; larger ones go
// to a list that every agent checks, and check every agent themselves.  A pair is always evaluated
// with the lower agent index in the i role, like k_overlap, so flags equal the stepwise kernels' bit
// for bit.
//
// Results are bit-identical to the stepwise graph (WM_ROLLOUT_STEPWISE), which runs the same device
// functions kernel by kernel.
#include "wm_device.cuh"
#include "wm_grid.cuh"

constexpr int FUSED_NT = 256;               // threads per CTA of the metrics kernel
constexpr int FUSED_MINB = 5;               // CTAs per SM it is compiled for (48 registers)
constexpr int FUSED_S = 8;                  // steps per block: 8, 4, 2 or 1 (fewer when A is large: shared memory)
constexpr float FUSED_HASH_H = 24.f;        // hash cell side, metres
constexpr float FUSED_EXT_MAX = 11.7f;      // half extent limit of hashed agents (< FUSED_HASH_H / 2, with margin)
constexpr uint32_t FUSED_EMPTY = 0xffffu;
constexpr int FUSED_PAD = 4;                // slot rows are Ap + 4 long: the 8 steps of an agent fall into 8 different banks
constexpr int FUSED_PL = 48;                // pair list entries per warp (overlap narrow phase)
constexpr int DYN_NT = 128;                 // threads per CTA of the dynamics kernel

struct FusedParams {
  wm_traj log, sim;
  int t0, n_steps, C, S;
  const float* actions;               // [B][n_steps][C][A]
  const uint8_t* av;                  // [B][n_steps][A]
  wm_rollout_out out;                 // any pointer may be NULL
  WmDynCfg dyn;
  const float4* segrec; const float4* segpair; const float4* segfin; const float4* chunks; const uint2* cells; const uint32_t* pool; const WmGrid* gridp;
  int seg_cap;
  unsigned long long* stats;
};

// shared-memory carve-up of the metrics kernel: per-agent block state, then S per-step slots
__host__ __device__ inline int fused_nbk(int Ap) { int n = 64; while (n < 2 * Ap) n <<= 1; return n; }
__host__ __device__ inline size_t fused_persist_bytes(int Ap) {
  return (size_t)Ap * (16 + 4 + 2 + 2 + 1) + (size_t)fused_nbk(Ap) * 4 + 64 + (FUSED_NT / 32) * (FUSED_PL + 1) * 4 + 16;
}
__host__ __device__ inline size_t fused_slot_bytes(int Ap) { return (size_t)(Ap + FUSED_PAD) * (7 * 4 + 2); }
static inline int fused_pick_S(int A) {
  const int Ap = (A + 31) / 32 * 32;
  const size_t budget = 45400;                            // 5 CTAs per SM when it fits (48 registers, FUSED_MINB)
  const size_t per = fused_persist_bytes(Ap), slot = fused_slot_bytes(Ap);
  const int fit = per + slot >= budget ? 1 : (int)((budget - per) / slot);
  int S = FUSED_S;
  while (S > 1 && S > fit) S >>= 1;
  return S;
}

struct FusedIn { float a0, a1, a2, lx, ly; uint8_t av, lv; };

__device__ __forceinline__ FusedIn fused_load_in(const FusedParams& p, int64_t sb, int64_t ab, int k, int a, int A, int C) {
  FusedIn r;
  const int64_t o = sb + (int64_t)(p.t0 + k + 1) * A + a;
  const int64_t ak = ab + k;
  // streamed once: evict-first loads
  r.av = __ldcs(p.av + ak * A + a);
  const float* act = p.actions + ak * C * A + a;
  r.a0 = __ldcs(act); r.a1 = __ldcs(act + A); r.a2 = C > 2 ? __ldcs(act + 2 * (int64_t)A) : 0.f;
  r.lx = __ldcs(p.log.x + o); r.ly = __ldcs(p.log.y + o); r.lv = __ldcs(p.log.valid + o);
  return r;
}

// ======================================================================================
// k_rollout_dyn: the trajectory (a1 / a2, D8, D9), log divergence (a5), ADE (D21)
// ======================================================================================
// DYN_C >= 0: the dynamics model is a compile-time constant
template <int DYN_C>
__global__ void __launch_bounds__(DYN_NT, 16) k_rollout_dyn(FusedParams p) {
  const int A = p.sim.A, nba = (A + DYN_NT - 1) / DYN_NT;
  const int b = blockIdx.x / nba, a = (blockIdx.x % nba) * DYN_NT + threadIdx.x;
  if (a >= A) return;
  WmDynCfg dyn = p.dyn;
  if (DYN_C >= 0) dyn.dynamics = DYN_C;
  const int C = DYN_C >= 0 ? (DYN_C == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3) : p.C;
  const int64_t TA = (int64_t)p.sim.T * A;
  const int64_t sb = (int64_t)b * TA;                // scenario offset in the trajectories
  const int64_t ab = (int64_t)b * p.n_steps;         // scenario offset in the action / metric rows, in rows
  const int64_t o0 = sb + (int64_t)p.t0 * A + a;
  bool v = p.sim.valid[o0] != 0;
  float x = 0.f, y = 0.f, th = 0.f, vx = 0.f, vy = 0.f, ln = 0.f, wd = 0.f, sn = 0.f, cs = 1.f;
  if (v) {
    x = p.sim.x[o0]; y = p.sim.y[o0]; th = p.sim.yaw[o0]; vx = p.sim.vel_x[o0]; vy = p.sim.vel_y[o0];
    ln = p.sim.length[o0]; wd = p.sim.width[o0];
    sincosf(th, &sn, &cs);
  }
  double sum = 0.0;                                   // sum of valid log divergences (D21)
  int cnt = 0;
  FusedIn in = fused_load_in(p, sb, ab, 0, a, A, C);
#pragma unroll 1
  for (int k = 0; k < p.n_steps; ++k) {
    const FusedIn cur = in;
    if (k + 1 < p.n_steps) in = fused_load_in(p, sb, ab, k + 1, a, A, C);     // prefetch: nothing below depends on it
    const int64_t o = sb + (int64_t)(p.t0 + k + 1) * A + a;
    const bool use_dyn = cur.av != 0 && v;                          // D8
    float xn, yn, thn, vxn, vyn, s1 = 0.f, c1 = 1.f;
    if (use_dyn) {
      wm_dyn_step(dyn, x, y, th, vx, vy, sn, cs, cur.a0, cur.a1, cur.a2, xn, yn, thn, vxn, vyn, s1, c1);
      v = true;                                                     // D9: keeps its box
    } else {                                                        // log playback, L164
      xn = cur.lx; yn = cur.ly; thn = p.log.yaw[o]; vxn = p.log.vel_x[o]; vyn = p.log.vel_y[o];
      ln = p.log.length[o]; wd = p.log.width[o];
      v = cur.lv != 0;
      if (v) sincosf(thn, &s1, &c1);
    }
    __stcs(p.sim.x + o, xn); __stcs(p.sim.y + o, yn); __stcs(p.sim.yaw + o, thn);
    __stcs(p.sim.vel_x + o, vxn); __stcs(p.sim.vel_y + o, vyn);
    __stcs(p.sim.length + o, ln); __stcs(p.sim.width + o, wd); __stcs(p.sim.valid + o, (uint8_t)v);
    const bool ldv = v && cur.lv != 0;                              // a5, L106
    const float d = ldv ? wm_logdiv(xn, yn, cur.lx, cur.ly) : 0.f;
    if (p.out.log_div) __stcs(p.out.log_div + (ab + k) * A + a, d);
    if (ldv) { sum += (double)d; cnt += 1; }
    x = xn; y = yn; th = thn; vx = vxn; vy = vyn; sn = s1; cs = c1;
  }
  const int64_t oa = (int64_t)b * A + a;
  if (p.out.ade) p.out.ade[oa] = cnt ? (float)(sum / cnt) : 0.f;
  if (p.out.any_overlap) p.out.any_overlap[oa] = 0;                 // the metrics kernel sets the flags that are 1
  if (p.out.any_offroad) p.out.any_offroad[oa] = 0;
}

// ======================================================================================
// k_rollout_dyn_bulk: the same trajectory kernel with its input rows staged by bulk (TMA) copies
// ======================================================================================
// One CTA per scenario, one thread per agent.  The inputs of DYN_SS consecutive steps - actions, action masks and
// the logged rows - are contiguous per array ([...][A] row-major), so thread 0 brings each of them into shared
// memory with ONE 1-D bulk copy (cp.async.bulk -> mbarrier), two stages ahead, and the threads read them there with
// 32-bit addresses and immediate offsets instead of ten global streams of 128-byte requests per warp with 64-bit
// address arithmetic each (k_rollout_dyn is bound by instruction issue and load latency, profiles/r02_k_rollout_ncu.md).
// The successor rows leave with plain streaming stores: staging them for bulk stores as well costs the shared
// memory that keeps enough CTAs resident (measured: 0.62 ms with both directions staged, 0.51 ms with the inputs
// only, 0.65 ms for k_rollout_dyn).  Needs A % 16 == 0 and 16-byte aligned arrays (bulk copies); other shapes take
// k_rollout_dyn.  Same device arithmetic: bit-identical rows.
constexpr int DYN_SS = 4;                   // steps per stage (2: 0.54 ms, 4: 0.51 ms, 6: 0.67 ms, 8: 0.87 ms)

struct DynBulkSmem { int act, av, lx, ly, lyaw, lvx, lvy, llen, lwid, lv, in_bytes; };   // byte offsets inside a stage buffer
__host__ __device__ inline DynBulkSmem dyn_bulk_layout(int A, int C) {
  DynBulkSmem m;
  const int row = A * 4 * DYN_SS, rowb = A * DYN_SS;
  int o = 0;
  m.act = o; o += C * row;
  m.lx = o; o += row; m.ly = o; o += row; m.lyaw = o; o += row; m.lvx = o; o += row; m.lvy = o; o += row;
  m.llen = o; o += row; m.lwid = o; o += row;
  m.av = o; o += rowb; m.lv = o; o += rowb;
  m.in_bytes = (o + 127) & ~127;
  return m;
}

template <int DYN_C>
__global__ void __launch_bounds__(1024) k_rollout_dyn_bulk(FusedParams p) {
  extern __shared__ __align__(128) unsigned char dsm[];
  __shared__ __align__(8) uint64_t bars[2];
  const int A = p.sim.A, b = blockIdx.x, a = threadIdx.x;
  WmDynCfg dyn = p.dyn;
  if (DYN_C >= 0) dyn.dynamics = DYN_C;
  const int C = DYN_C >= 0 ? (DYN_C == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3) : p.C;
  const DynBulkSmem m = dyn_bulk_layout(A, C);
  const int64_t TA = (int64_t)p.sim.T * A;
  const int64_t sb = (int64_t)b * TA;                // scenario offset in the trajectories
  const int64_t ab = (int64_t)b * p.n_steps;         // scenario offset in the action / metric rows, in rows
  const int n_stage = (p.n_steps + DYN_SS - 1) / DYN_SS;
  if (a == 0) { mbar_init(&bars[0], 1); mbar_init(&bars[1], 1); mbar_fence_init(); }
  __syncthreads();
  // producer (thread 0): the inputs of stage s -> buffer s & 1
  auto load_stage = [&](int s) {
    const int k0 = s * DYN_SS, ns = min(DYN_SS, p.n_steps - k0);
    unsigned char* d = dsm + (s & 1) * m.in_bytes;
    uint64_t* bar = &bars[s & 1];
    const uint32_t rf = (uint32_t)(ns * A * 4), rb = (uint32_t)(ns * A);
    mbar_expect_tx(bar, (uint32_t)(C + 7) * rf + 2u * rb);
    const int64_t ro = sb + (int64_t)(p.t0 + 1 + k0) * A;          // first logged row of the stage
    tma_load_1d(d + m.act, p.actions + (ab + k0) * C * A, (uint32_t)C * rf, bar);
    tma_load_1d(d + m.lx, p.log.x + ro, rf, bar);       tma_load_1d(d + m.ly, p.log.y + ro, rf, bar);
    tma_load_1d(d + m.lyaw, p.log.yaw + ro, rf, bar);   tma_load_1d(d + m.lvx, p.log.vel_x + ro, rf, bar);
    tma_load_1d(d + m.lvy, p.log.vel_y + ro, rf, bar);  tma_load_1d(d + m.llen, p.log.length + ro, rf, bar);
    tma_load_1d(d + m.lwid, p.log.width + ro, rf, bar);
    tma_load_1d(d + m.av, p.av + (ab + k0) * A, rb, bar);
    tma_load_1d(d + m.lv, p.log.valid + ro, rb, bar);
  };
  if (a == 0) { load_stage(0); if (n_stage > 1) load_stage(1); }
  // the state at t0
  bool v = false;
  float x = 0.f, y = 0.f, th = 0.f, vx = 0.f, vy = 0.f, ln = 0.f, wd = 0.f, sn = 0.f, cs = 1.f;
  if (a < A) {
    const int64_t o0 = sb + (int64_t)p.t0 * A + a;
    v = p.sim.valid[o0] != 0;
    if (v) {
      x = p.sim.x[o0]; y = p.sim.y[o0]; th = p.sim.yaw[o0]; vx = p.sim.vel_x[o0]; vy = p.sim.vel_y[o0];
      ln = p.sim.length[o0]; wd = p.sim.width[o0];
      sincosf(th, &sn, &cs);
    }
  }
  double sum = 0.0;                                   // sum of valid log divergences (D21)
  int cnt = 0;
  for (int s = 0; s < n_stage; ++s) {
    const int k0 = s * DYN_SS, ns = min(DYN_SS, p.n_steps - k0);
    const unsigned char* in = dsm + (s & 1) * m.in_bytes;
    mbar_wait(&bars[s & 1], (uint32_t)((s >> 1) & 1));
    if (a < A) {
      for (int j = 0; j < ns; ++j) {
        const int r = j * A + a;
        const float* act = (const float*)(in + m.act) + (size_t)j * C * A + a;
        const uint8_t avk = in[m.av + r], lvk = in[m.lv + r];
        const float lx = ((const float*)(in + m.lx))[r], ly = ((const float*)(in + m.ly))[r];
        const bool use_dyn = avk != 0 && v;                          // D8
        float xn, yn, thn, vxn, vyn, s1 = 0.f, c1 = 1.f;
        if (use_dyn) {
          wm_dyn_step(dyn, x, y, th, vx, vy, sn, cs, act[0], act[A], C > 2 ? act[2 * A] : 0.f, xn, yn, thn, vxn, vyn, s1, c1);
          v = true;                                                  // D9: keeps its box
        } else {                                                     // log playback, L164
          xn = lx; yn = ly; thn = ((const float*)(in + m.lyaw))[r]; vxn = ((const float*)(in + m.lvx))[r];
          vyn = ((const float*)(in + m.lvy))[r]; ln = ((const float*)(in + m.llen))[r]; wd = ((const float*)(in + m.lwid))[r];
          v = lvk != 0;
          if (v) sincosf(thn, &s1, &c1);
        }
        const bool ldv = v && lvk != 0;                              // a5, L106
        const float d = ldv ? wm_logdiv(xn, yn, lx, ly) : 0.f;
        const int64_t o = sb + (int64_t)(p.t0 + 1 + k0 + j) * A + a;
        __stcs(p.sim.x + o, xn); __stcs(p.sim.y + o, yn); __stcs(p.sim.yaw + o, thn);
        __stcs(p.sim.vel_x + o, vxn); __stcs(p.sim.vel_y + o, vyn);
        __stcs(p.sim.length + o, ln); __stcs(p.sim.width + o, wd); __stcs(p.sim.valid + o, (uint8_t)v);
        if (p.out.log_div) __stcs(p.out.log_div + (ab + k0 + j) * A + a, d);
        if (ldv) { sum += (double)d; cnt += 1; }
        x = xn; y = yn; th = thn; vx = vxn; vy = vyn; sn = s1; cs = c1;
      }
    }
    __syncthreads();                                   // everyone has read the buffer: it takes stage s + 2
    if (a == 0 && s + 2 < n_stage) load_stage(s + 2);
  }
  if (a < A) {
    const int64_t oa = (int64_t)b * A + a;
    if (p.out.ade) p.out.ade[oa] = cnt ? (float)(sum / cnt) : 0.f;
    if (p.out.any_overlap) p.out.any_overlap[oa] = 0;                 // the metrics kernel sets the flags that are 1
    if (p.out.any_offroad) p.out.any_offroad[oa] = 0;
  }
}

__device__ __forceinline__ int fused_cell(float v) {
  return (int)floorf(fminf(fmaxf(v * (1.f / FUSED_HASH_H), -1.0e9f), 1.0e9f));
}
__device__ __forceinline__ uint32_t fused_bucket(int ix, int iy, uint32_t mask) {
  return (((uint32_t)ix * 73856093u) ^ ((uint32_t)iy * 19349663u)) & mask;
}

// ======================================================================================
// k_rollout_metrics: overlap (a3) and offroad (a4) of one block of steps of one scenario
// ======================================================================================
// AP_C / S_C > 0: padded agent count and steps per block known at compile time (the shared-memory
// carve-up then folds into immediate offsets); 0: taken from the arguments.
template <int AP_C, int S_C, bool STATS>
__global__ void __launch_bounds__(FUSED_NT, FUSED_MINB) k_rollout_metrics(FusedParams p, int nblk) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int A = p.sim.A, nb = AP_C ? AP_C / 32 : (A + 31) / 32, Ap = nb * 32, Aps = Ap + FUSED_PAD, S = S_C ? S_C : p.S;
  const int NBK = fused_nbk(Ap);
  // ---- per-agent state of the block ----
  float4* s_bb = (float4*)smem_raw;                  // [Ap] bounding box over the block, inflated: x0, y0, x1, y1
  float* s_br = (float*)(s_bb + Ap);                 // [Ap] largest circumradius over the block, inflated
  uint32_t* heads = (uint32_t*)(s_br + Ap);          // [NBK] first agent of the bucket, FUSED_EMPTY if none
  int* s_nover = (int*)(heads + NBK);                // oversize count (+ padding to 64 B)
  uint32_t* s_pl = (uint32_t*)(s_nover + 16);        // [warps][FUSED_PL + 1] pairs whose block boxes meet: count, (lo << 16) | hi
  int* s_task = (int*)(s_pl + (FUSED_NT / 32) * (FUSED_PL + 1));            // corner task counter (+ padding to 16 B)
  uint16_t* nxt = (uint16_t*)(s_task + 4);           // [Ap] next agent of the same bucket
  uint16_t* over = nxt + Ap;                         // [Ap] agents too large for the hash
  uint8_t* s_bvalid = (uint8_t*)(over + Ap);         // [Ap] valid at some step of the block
  // ---- per-step slots ----
  float* px = (float*)(smem_raw + fused_persist_bytes(Ap));      // [S][Aps] each
  float* py = px + S * Aps;  float* pc = py + S * Aps;  float* ps = pc + S * Aps;
  float* phl = ps + S * Aps; float* phw = phl + S * Aps;
  float* psd = phw + S * Aps;                        // max signed corner distance (a4)
  uint8_t* pvalid = (uint8_t*)(psd + S * Aps);       // [S][Aps]
  uint8_t* pov = pvalid + S * Aps;                   // [S][Aps] overlap flag (a3)

  const int b = blockIdx.x / nblk, k0 = (blockIdx.x % nblk) * S, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int Sb = min(S, p.n_steps - k0);
  const int64_t TA = (int64_t)p.sim.T * A;
  const int64_t sb = (int64_t)b * TA + (int64_t)(p.t0 + 1 + k0) * A;      // first row of the block
  const int64_t ab = (int64_t)b * p.n_steps + k0;    // first metric row of the block
  const WmGridView gv = wm_grid_view(p.segrec, p.segpair, p.segfin, p.chunks, p.cells, p.pool, p.gridp, p.seg_cap, WM_POOL_CAP, b);

  // ================= phase A: rows of the block -> slots =================
  for (int e = tid; e < S * Ap; e += FUSED_NT) {
    const int s = AP_C ? e / AP_C : e / Ap, a = e - s * Ap, q = s * Aps + a;
    bool v = false;
    float x = 0.f, y = 0.f, hl = 0.f, hw = 0.f, sn = 0.f, cs = 1.f;       // invalid slots: finite zeros (D10)
    if (s < Sb && a < A) {
      const int64_t o = sb + (int64_t)s * A + a;
      v = __ldcs(p.sim.valid + o) != 0;
      if (v) {
        x = __ldcs(p.sim.x + o); y = __ldcs(p.sim.y + o);
        hl = 0.5f * __ldcs(p.sim.length + o); hw = 0.5f * __ldcs(p.sim.width + o);
        sincosf(__ldcs(p.sim.yaw + o), &sn, &cs);
      }
    }
    px[q] = x; py[q] = y; pc[q] = cs; ps[q] = sn; phl[q] = hl; phw[q] = hw; psd[q] = 0.f;
    pvalid[q] = (uint8_t)v; pov[q] = 0;
  }
  for (int i = tid; i < NBK; i += FUSED_NT) heads[i] = FUSED_EMPTY;
  if (tid == 0) { *s_task = 0; *s_nover = 0; }
  __syncthreads();
  // overlap broad phase of the block, one thread per agent (the first nb warps; the others go on to the
  // corner tasks): the agent's boxes all lie inside [bx0 - br, bx1 + br] x [..]
  if (warp < nb || nb > FUSED_NT / 32) {
    for (int a = tid; a < Ap; a += FUSED_NT) {
      float bx0 = 3.0e38f, by0 = 3.0e38f, bx1 = -3.0e38f, by1 = -3.0e38f, br = 0.f;
      for (int s = 0; s < Sb; ++s) {
        const int q = s * Aps + a;
        if (pvalid[q] != 0) {
          const float xn = px[q], yn = py[q], hl = phl[q], hw = phw[q];
          bx0 = fminf(bx0, xn); bx1 = fmaxf(bx1, xn); by0 = fminf(by0, yn); by1 = fmaxf(by1, yn);
          br = fmaxf(br, sqrtf(fmaf(hl, hl, hw * hw)));
        }
      }
      const bool bv = bx0 <= bx1;
      s_bvalid[a] = (uint8_t)bv;
      if (bv) {
        br = fmaf(br, 1.001f, 1e-3f);                                   // float32 rounding of the pair tests
        s_bb[a] = make_float4(bx0 - br, by0 - br, bx1 + br, by1 + br);
        s_br[a] = br;
        const float ext = 0.5f * fmaxf(bx1 - bx0, by1 - by0) + br;
        if (ext <= FUSED_EXT_MAX) {
          const uint32_t bk = fused_bucket(fused_cell(0.5f * (bx0 + bx1)), fused_cell(0.5f * (by0 + by1)), (uint32_t)NBK - 1u);
          nxt[a] = (uint16_t)atomicExch(&heads[bk], (uint32_t)a);
        } else {
          over[atomicAdd(s_nover, 1)] = (uint16_t)a;
        }
      }
    }
    // the warps that built the hash meet at a named barrier of their own
    const int nhw = min(nb, FUSED_NT / 32);
    asm volatile("bar.sync 1, %0;" ::"r"(nhw * 32) : "memory");
  }
  // ================= phase B: warp tasks =================
  // lanes of a corner task: 4 corners x S steps x (8 / S) agents
  const int kk = lane & 3, ls = (lane >> 2) & (S - 1), la = (lane >> 2) / S, apt = 8 / S;
  int n_eval = 0, n_slow = 0, n_corner = 0;
  const int n_ctask = Ap / apt;
  // ---- overlap flags of 32 agents at every step of the block (a3): the warps that built the hash ----
  // broad phase, one lane per agent i: the pairs (i, j > i) whose block boxes meet go to the
  // warp's list; narrow phase, one lane per (pair, step): the pair test of k_overlap
  if (warp < nb || nb > FUSED_NT / 32) {
    for (int task = warp; task < nb; task += FUSED_NT / 32) {
      const int i = task * 32 + lane;
      uint32_t* pl = s_pl + warp * (FUSED_PL + 1);
      auto narrow = [&](int lo, int hi, int s) {       // lo < hi: the lower index takes the i role of k_overlap
        const int ql = s * Aps + lo, qh = s * Aps + hi;
        if (pvalid[ql] == 0 || pvalid[qh] == 0) return;
        const float dx = px[qh] - px[ql], dy = py[qh] - py[ql];
        const float hll = phl[ql], hwl = phw[ql], hlh = phl[qh], hwh = phw[qh];
        if (wm_circles_touch(dx, dy, sqrtf(fmaf(hlh, hlh, hwh * hwh)) + sqrtf(fmaf(hll, hll, hwl * hwl))) &&
            wm_sat_overlap(dx, dy, pc[ql], ps[ql], hll, hwl, pc[qh], ps[qh], hlh, hwh)) { pov[ql] = 1; pov[qh] = 1; }
      };
      __syncwarp();
      if (lane == 0) pl[0] = 0;
      __syncwarp();
      if (s_bvalid[i] != 0) {                         // per lane: no warp-level operation inside
        const float4 bi = s_bb[i];
        auto test = [&](int j) {
          if (j <= i) return;
          const float4 bj = s_bb[j];
          if (bi.x > bj.z || bj.x > bi.z || bi.y > bj.w || bj.y > bi.w) return;     // boxes of the block apart
          const uint32_t slot = atomicAdd(&pl[0], 1u);
          if (slot < (uint32_t)FUSED_PL) pl[1 + slot] = ((uint32_t)i << 16) | (uint32_t)j;
          else for (int s = 0; s < Sb; ++s) narrow(i, j, s);                        // list full: in place
        };
        if (0.5f * fmaxf(bi.z - bi.x, bi.w - bi.y) <= FUSED_EXT_MAX) {
          const int ix = fused_cell(0.5f * (bi.x + bi.z)), iy = fused_cell(0.5f * (bi.y + bi.w));
          uint32_t j = FUSED_EMPTY;
          for (int probe = 0; ;) {                    // one flat loop over the 9 cells and their lists
            if (j == FUSED_EMPTY) {
              if (probe == 9) break;
              j = heads[fused_bucket(ix + probe % 3 - 1, iy + probe / 3 - 1, (uint32_t)NBK - 1u)];
              ++probe;
              continue;
            }
            test((int)j);
            j = nxt[j];
          }
          const int no = *s_nover;
          for (int e = 0; e < no; ++e) test((int)over[e]);
        } else {
          for (int j = i + 1; j < A; ++j) if (s_bvalid[j] != 0) test(j);
        }
      }
      __syncwarp();
      const int np = (int)min(pl[0], (uint32_t)FUSED_PL);
      for (int it = lane; it < np * S; it += 32) {
        const uint32_t pr = pl[1 + it / S];
        const int s = it & (S - 1);
        if (s < Sb) narrow((int)(pr >> 16), (int)(pr & 0xffffu), s);
      }
    }
  }
  // ---- the 4 corners of one agent (8 / S agents) at every step of the block (a4) ----
  // a corner task's lane: agent slot q, validity, centre, half extents, corner offset
  auto corner = [&](int task, int& q, bool& v, float& cx, float& cy, float& hl, float& hw, float& offx, float& offy) {
    const int a = task * apt + la;
    q = ls * Aps + a;
    v = ls < Sb && pvalid[q] != 0;
    cx = px[q]; cy = py[q]; hl = phl[q]; hw = phw[q];
    float ax, ay, bx, by;
    wm_box_offsets_h(ps[q], pc[q], hl, hw, ax, ay, bx, by);
    const float ox = (kk & 1) ? bx : ax, oy = (kk & 1) ? by : ay;
    offx = (kk & 2) ? -ox : ox; offy = (kk & 2) ? -oy : oy;
  };
  // the cell header of the NEXT task's corner is requested at the end of a task, ahead of the shared
  // counter's round trip, together with the task's corner set-up, which the walk then finds in registers
  int q = 0; bool v = false; float cx = 0.f, cy = 0.f, hl = 0.f, hw = 0.f, offx = 0.f, offy = 0.f;
  auto header = [&](int task) {
    if (task >= n_ctask) return make_uint2(0u, 0u);
    corner(task, q, v, cx, cy, hl, hw, offx, offy);
    return wm_grid_header(gv, v, cx, cy, offx, offy);
  };
  // the shared counter is bumped by lane 0 at the START of a task and its answer is only read at the end:
  // the atomic's round trip hides under the walk
  int tn = 0;
  if (lane == 0) tn = atomicAdd(s_task, 1);
  int task = __shfl_sync(0xffffffffu, tn, 0);
  uint2 hd = header(task);
  while (task < n_ctask) {
    if (lane == 0) tn = atomicAdd(s_task, 1);
    if (__any_sync(0xffffffffu, v)) {                               // psd of invalid slots is never read
      float best; uint32_t bso;
      const bool slow = wm_grid_fast_hd(gv, hd, cx, cy, offx, offy, best, bso, n_eval);
      n_slow += slow; n_corner += v;
      uint32_t todo = __ballot_sync(0xffffffffu, slow);
      while (todo) {                                  // boxes with corners off the grid / in a crowded cell
        const int g4 = (__ffs(todo) - 1) & ~3;
        const uint32_t gm = (todo >> g4) & 15u;
        todo &= ~(15u << g4);
        const float acx = __shfl_sync(0xffffffffu, cx, g4), acy = __shfl_sync(0xffffffffu, cy, g4);
        const float fax = __shfl_sync(0xffffffffu, offx, g4), fay = __shfl_sync(0xffffffffu, offy, g4);
        const float fbx = __shfl_sync(0xffffffffu, offx, g4 + 1), fby = __shfl_sync(0xffffffffu, offy, g4 + 1);
        const float ahl = __shfl_sync(0xffffffffu, hl, g4), ahw = __shfl_sync(0xffffffffu, hw, g4);
        const float o4x[4] = {fax, fbx, -fax, -fbx}, o4y[4] = {fay, fby, -fay, -fby};
        float b4[4]; int i4[4], ne = 0;
        wm_grid_search_warp4(gv, acx, acy, o4x, o4y, sqrtf(fmaf(ahl, ahl, ahw * ahw)), b4, i4, ne);
        if ((lane & ~3) == g4 && ((gm >> kk) & 1u)) {
          best = kk == 0 ? b4[0] : kk == 1 ? b4[1] : kk == 2 ? b4[2] : b4[3];
          bso = wm_bso_of(kk == 0 ? i4[0] : kk == 1 ? i4[1] : kk == 2 ? i4[2] : i4[3]);
        }
        if (lane == 0) n_eval += ne;
      }
      float m = v ? wm_grid_finish(gv, cx, cy, offx, offy, best, bso) : 0.f;
      m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 1));               // D18: max over the 4 corners
      m = fmaxf(m, __shfl_xor_sync(0xffffffffu, m, 2));
      if (kk == 0 && v) psd[q] = m;
    }
    task = __shfl_sync(0xffffffffu, tn, 0); hd = header(task);
  }
  __syncthreads();
  // ================= phase C: metric rows of the block (D18, D19, D10) =================
  for (int e = tid; e < Sb * Ap; e += FUSED_NT) {
    const int s = AP_C ? e / AP_C : e / Ap, a = e - s * Ap;
    if (a >= A) continue;
    const int q = s * Aps + a;
    const int64_t o = (ab + s) * A + a;
    const bool vv = pvalid[q] != 0;
    const float m = vv ? psd[q] : 0.f;
    const uint8_t fo = pov[q], ff = (uint8_t)(vv && m > 0.f);
    if (p.out.overlap) __stcs(p.out.overlap + o, fo);
    if (p.out.offroad_dist) __stcs(p.out.offroad_dist + o, m);
    if (p.out.offroad) __stcs(p.out.offroad + o, ff);
    // aggregates: k_rollout_dyn cleared them; every writer stores the same 1
    if (fo && p.out.any_overlap) p.out.any_overlap[(int64_t)b * A + a] = 1;
    if (ff && p.out.any_offroad) p.out.any_offroad[(int64_t)b * A + a] = 1;
  }
  if (STATS && p.stats) {
    const unsigned ne = __reduce_add_sync(0xffffffffu, (unsigned)n_eval), ns = __reduce_add_sync(0xffffffffu, (unsigned)n_slow);
    const unsigned nc = __reduce_add_sync(0xffffffffu, (unsigned)n_corner);
    if (lane == 0 && nc) {
      atomicAdd(&p.stats[0], (unsigned long long)ne);
      atomicAdd(&p.stats[1], (unsigned long long)nc * (unsigned long long)max(gv.g.nseg, 0));
      atomicAdd(&p.stats[2], (unsigned long long)ns);
      atomicAdd(&p.stats[3], (unsigned long long)nc);
    }
  }
}

// scenarios per launch such that the pair records of a launch span less than 4 GB (32-bit offsets in the walk)
static inline int fused_launch_batch(int64_t seg_cap) {
  const int64_t per = seg_cap * 24;                   // bytes of pair records per scenario
  int64_t n = per > 0 ? (int64_t)0xffffffffLL / per : 1 << 30;
  if (n < 1) n = 1;
  return (int)(n > (1 << 30) ? (1 << 30) : n);
}

static cudaError_t fused_launch_part(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                     const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                     int b0, cudaStream_t s, cudaEvent_t* ev = nullptr);

cudaError_t wm_launch_rollout_fused_timed(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                          const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                          cudaEvent_t* ev, cudaStream_t s) {
  if (sim.B > fused_launch_batch((int64_t)h->seg_tiles * WM_TILE_SEGS)) return cudaErrorInvalidValue;   // one launch pair only
  return fused_launch_part(h, log, sim, t0, n_steps, actions, action_valid, out, 0, s, ev);
}

cudaError_t wm_launch_rollout_fused(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                    const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                    int b0, cudaStream_t s) {
  const int nbmax = fused_launch_batch((int64_t)h->seg_tiles * WM_TILE_SEGS);
  if (sim.B <= nbmax) return fused_launch_part(h, log, sim, t0, n_steps, actions, action_valid, out, b0, s);
  const int C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  for (int c0 = 0; c0 < sim.B; c0 += nbmax) {          // very large batches: scenario ranges, one launch pair each
    const int nb = sim.B - c0 < nbmax ? sim.B - c0 : nbmax;
    const int64_t oT = (int64_t)c0 * sim.T * sim.A, oW = (int64_t)c0 * n_steps * sim.A, oA = (int64_t)c0 * sim.A;
    wm_traj cl = log, cs = sim;
    cl.B = nb; cs.B = nb;
    cl.x += oT; cl.y += oT; cl.yaw += oT; cl.vel_x += oT; cl.vel_y += oT; cl.length += oT; cl.width += oT; cl.valid += oT;
    cs.x += oT; cs.y += oT; cs.yaw += oT; cs.vel_x += oT; cs.vel_y += oT; cs.length += oT; cs.width += oT; cs.valid += oT;
    wm_rollout_out co = out;
    if (co.overlap) co.overlap += oW;
    if (co.offroad) co.offroad += oW;
    if (co.offroad_dist) co.offroad_dist += oW;
    if (co.log_div) co.log_div += oW;
    if (co.any_overlap) co.any_overlap += oA;
    if (co.any_offroad) co.any_offroad += oA;
    if (co.ade) co.ade += oA;
    const cudaError_t e = fused_launch_part(h, cl, cs, t0, n_steps, actions + oW * C, action_valid + oW, co, b0 + c0, s);
    if (e != cudaSuccess) return e;
  }
  return cudaSuccess;
}

static cudaError_t fused_launch_part(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                     const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                     int b0, cudaStream_t s, cudaEvent_t* ev) {
  FusedParams p;
  p.log = log; p.sim = sim; p.t0 = t0; p.n_steps = n_steps;
  p.C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  p.S = fused_pick_S(sim.A);
  p.actions = actions; p.av = action_valid; p.out = out;
  p.dyn = WmDynCfg{h->cfg.dynamics, h->cfg.dt, h->cfg.max_accel, h->cfg.max_curvature};
  p.seg_cap = h->seg_tiles * WM_TILE_SEGS;
  const int64_t cap = p.seg_cap;
  p.segrec = h->segrec + b0 * cap * 2; p.segpair = h->segpair + b0 * (cap / 2) * 3; p.segfin = h->segfin + b0 * cap;
  p.chunks = h->chunks + b0 * (cap / WM_CHUNK); p.cells = h->cells + (int64_t)b0 * WM_GRID_CELLS;
  p.pool = h->pool + (int64_t)b0 * WM_POOL_CAP; p.gridp = h->gridp + b0;
  p.stats = h->stats_on ? h->cull_stats : nullptr;
  // ---- the trajectory ----
  const int nba = (sim.A + DYN_NT - 1) / DYN_NT;
  const int64_t n_dyn = (int64_t)sim.B * nba;
  cudaError_t e = cudaSuccess;
  if (ev && (e = cudaEventRecord(ev[0], s)) != cudaSuccess) return e;
  // bulk-copy staging needs 16-byte aligned rows of every array
  bool bulk = sim.A % 16 == 0 && sim.A <= 1024;
  {
    const void* ptrs[] = {log.x, log.y, log.yaw, log.vel_x, log.vel_y, log.length, log.width, log.valid, sim.x, sim.y, sim.yaw,
                          sim.vel_x, sim.vel_y, sim.length, sim.width, sim.valid, actions, action_valid, out.log_div};
    for (const void* q : ptrs) bulk = bulk && ((uintptr_t)q & 15u) == 0;
  }
  const DynBulkSmem bm = dyn_bulk_layout(sim.A, p.C);
  const size_t dsmem = 2 * (size_t)bm.in_bytes;
  bulk = bulk && dsmem <= 200 * 1024;
  if (bulk) {
    const unsigned nt = (unsigned)((sim.A + 31) / 32 * 32);
    if (h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE) {
      e = cudaFuncSetAttribute(k_rollout_dyn_bulk<WM_DYN_INVERTIBLE_BICYCLE>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsmem);
      if (e != cudaSuccess) return e;
      k_rollout_dyn_bulk<WM_DYN_INVERTIBLE_BICYCLE><<<(unsigned)sim.B, nt, dsmem, s>>>(p);
    } else {
      e = cudaFuncSetAttribute(k_rollout_dyn_bulk<-1>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)dsmem);
      if (e != cudaSuccess) return e;
      k_rollout_dyn_bulk<-1><<<(unsigned)sim.B, nt, dsmem, s>>>(p);
    }
  } else if (h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE) k_rollout_dyn<WM_DYN_INVERTIBLE_BICYCLE><<<(unsigned)n_dyn, DYN_NT, 0, s>>>(p);
  else k_rollout_dyn<-1><<<(unsigned)n_dyn, DYN_NT, 0, s>>>(p);
  h->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (ev && (e = cudaEventRecord(ev[1], s)) != cudaSuccess) return e;
  // ---- its metrics ----
  const int Ap = (sim.A + 31) / 32 * 32;
  const size_t smem = fused_persist_bytes(Ap) + (size_t)p.S * fused_slot_bytes(Ap);
  const int nblk = (n_steps + p.S - 1) / p.S;
  const int64_t n_cta = (int64_t)sim.B * nblk;
  if (n_cta > 0x7fffffffLL) return cudaErrorInvalidConfiguration;
  // the opt-in above 48 KB is a per-device attribute: set it at every launch (cheap), so that a second
  // handle on another device gets it too
  e = cudaFuncSetAttribute(k_rollout_metrics<0, 0, true>, cudaFuncAttributeMaxDynamicSharedMemorySize,
                           (int)(fused_persist_bytes(1024) + fused_slot_bytes(1024)));
  if (e != cudaSuccess) return e;
  if (Ap == 128 && p.S == 8 && !p.stats) k_rollout_metrics<128, 8, false><<<(unsigned)n_cta, FUSED_NT, smem, s>>>(p, nblk);     // the pair counters compiled out
  else if (Ap == 128 && p.S == 8) k_rollout_metrics<128, 8, true><<<(unsigned)n_cta, FUSED_NT, smem, s>>>(p, nblk);
  else if (Ap == 32 && p.S == 8) k_rollout_metrics<32, 8, true><<<(unsigned)n_cta, FUSED_NT, smem, s>>>(p, nblk);
  else k_rollout_metrics<0, 0, true><<<(unsigned)n_cta, FUSED_NT, smem, s>>>(p, nblk);
  h->launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) return e;
  if (ev) e = cudaEventRecord(ev[2], s);
  return e;
}
