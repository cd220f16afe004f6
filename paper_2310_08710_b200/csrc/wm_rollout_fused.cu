// a8 closed-loop rollout ("Rollout ... faster than running Step 80 times"), fused:
// ONE kernel runs all n_steps of a scenario — dynamics (a1/a2), log divergence (a5), pairwise
// overlap (a3), offroad (a4) and the aggregates — with the scenario's state resident in shared
// memory, one CTA per scenario.  Per step the CTA only streams what is compulsory: the action
// row and log row t+1 in, sim row t+1 and the metric rows out (~10 KB); the candidate road-edge
// records of the grid search (wm_grid.cuh) stay hot in L1/L2 across steps because an agent moves
// at most a few metres per step.
//
//   phase A  one thread per agent : metric rows of the previous step (overlap flag, max over the
//            4 corner distances), successor state (shared arithmetic with k_step:
//            wm_device.cuh), sim row t+1 -> HBM, log divergence, sin/cos, half extents, corner
//            offsets -> shared memory
//   phase B1 one thread per corner: candidate walk of the corner's grid cell; corners that need
//            the full search (off the grid, crowded cell) go to a shared-memory queue
//            one warp per (tile, quarter) of the A x A matrix: separating-axis test, any-flags
//   phase B2 the queued corners, one warp each, spread over all warps of the CTA
//
// Bound: compulsory HBM bytes (~10 KB per scenario-step) against the per-step latency chain of a
// CTA (2 barriers, the dependent loads of the grid walk); see DESIGN.md.
// Results are bit-identical to the stepwise graph (WM_ROLLOUT_STEPWISE), which runs the same
// device functions kernel by kernel.
#include "wm_device.cuh"
#include "wm_grid.cuh"

#ifndef FUSED_NT
#define FUSED_NT 512
#endif
#ifndef FUSED_MINB
#define FUSED_MINB 2
#endif
constexpr int FUSED_SUB = 4;          // an overlap tile is split into 4 tasks of 8 rows

struct FusedParams {
  wm_traj log, sim;
  int t0, n_steps, C;
  const float* actions;               // [B][n_steps][C][A]
  const uint8_t* av;                  // [B][n_steps][A]
  wm_rollout_out out;                 // any pointer may be NULL
  WmDynCfg dyn;
  const float4* segrec; const float4* chunks; const uint4* cells; const uint32_t* pool; const WmGrid* gridp;
  int seg_cap;
  unsigned long long* stats;
};

__host__ __device__ inline size_t fused_smem_bytes(int A) {
  const size_t Ap = (size_t)((A + 31) / 32) * 32;
  return Ap * (16 * 4 + 8 + 4 + 4 + 16 + 4 + 4 + 1 + 1 + 1 + 1) + (Ap / 32) * 4 + 64;
}

// metric rows of step k for agent a, from what phase B left in shared memory (D18, D19, D10)
__device__ __forceinline__ void fused_flush_metrics(const FusedParams& p, int64_t rb, int k, int a, int A,
                                                    const uint8_t* s_valid, const uint32_t* s_ov, const float* s_csd,
                                                    uint8_t* s_anyov, uint8_t* s_anyoff) {
  const int64_t o = rb + (int64_t)k * A + a;
  const uint8_t fo = (uint8_t)(s_ov[a] != 0);
  if (p.out.overlap) p.out.overlap[o] = fo;
  s_anyov[a] |= fo;
  const bool v = s_valid[a] != 0;
  const float4 cd = *(const float4*)(s_csd + 4 * a);
  const float m = fmaxf(fmaxf(cd.x, cd.y), fmaxf(cd.z, cd.w));                 // D18: max over the 4 corners
  const uint8_t ff = (uint8_t)(v && m > 0.f);                                  // D19
  if (p.out.offroad_dist) p.out.offroad_dist[o] = v ? m : 0.f;
  if (p.out.offroad) p.out.offroad[o] = ff;
  s_anyoff[a] |= ff;
}

__global__ void __launch_bounds__(FUSED_NT, FUSED_MINB) k_rollout_fused(FusedParams p) {
  extern __shared__ __align__(16) unsigned char smem_raw[];
  const int A = p.sim.A, nb = (A + 31) / 32, Ap = nb * 32;
  double* s_sum = (double*)smem_raw;                 // [Ap] sum of valid log divergences (D21)
  float* sx = (float*)(s_sum + Ap);
  float* sy = sx + Ap;    float* syaw = sy + Ap;   float* svx = syaw + Ap;  float* svy = svx + Ap;
  float* slen = svy + Ap; float* swid = slen + Ap;
  float* sc = swid + Ap;  float* ss = sc + Ap;     float* shl = ss + Ap;    float* shw = shl + Ap;
  float* oax = shw + Ap;  float* oay = oax + Ap;   float* obx = oay + Ap;   float* oby = obx + Ap;
  float* srad = oby + Ap;                            // [Ap] circumradius of the box
  int* s_cnt = (int*)(srad + Ap);                    // [Ap] count of valid log divergences
  uint32_t* s_ov = (uint32_t*)(s_cnt + Ap);          // [Ap] overlap flag of the current step
  float* s_csd = (float*)(s_ov + Ap);                // [4 Ap] signed distance of every corner, current step
  int* s_q = (int*)(s_csd + 4 * Ap);                 // [Ap] queue of agents that need the warp search
  uint32_t* s_qm = (uint32_t*)(s_q + Ap);            // [Ap] which corners of the agent (4 bits; 0 = not queued)
  uint32_t* s_vw = s_qm + Ap;                        // [nb] validity ballot words
  uint8_t* s_valid = (uint8_t*)(s_vw + nb);          // [Ap]
  uint8_t* s_anyov = s_valid + Ap;                   // [Ap]
  uint8_t* s_anyoff = s_anyov + Ap;                  // [Ap]

  __shared__ int s_nq;
  const int b = blockIdx.x, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
  const int64_t TA = (int64_t)p.sim.T * A;
  const int64_t sb = (int64_t)b * TA;                // scenario offset in the trajectories
  const int64_t rb = (int64_t)b * p.n_steps * A;     // scenario offset in the metric rows
  const WmGridView gv = wm_grid_view(p.segrec, p.chunks, p.cells, p.pool, p.gridp, p.seg_cap, WM_POOL_CAP, b);

  // ---- prologue: row t0 of the simulated trajectory -> shared memory ----
  for (int a = tid; a < Ap; a += FUSED_NT) {
    const int64_t o = sb + (int64_t)p.t0 * A + a;
    const bool v = a < A && p.sim.valid[o] != 0;
    float x = 0.f, y = 0.f, th = 0.f, vx = 0.f, vy = 0.f, ln = 0.f, wd = 0.f, sn = 0.f, cs = 1.f;
    if (v) {
      x = p.sim.x[o]; y = p.sim.y[o]; th = p.sim.yaw[o]; vx = p.sim.vel_x[o]; vy = p.sim.vel_y[o];
      ln = p.sim.length[o]; wd = p.sim.width[o];
      sincosf(th, &sn, &cs);
    }
    sx[a] = x; sy[a] = y; syaw[a] = th; svx[a] = vx; svy[a] = vy; slen[a] = ln; swid[a] = wd;
    sc[a] = cs; ss[a] = sn; s_valid[a] = v;
    s_sum[a] = 0.0; s_cnt[a] = 0; s_ov[a] = 0; s_anyov[a] = 0; s_anyoff[a] = 0; s_qm[a] = 0;
  }
  __syncthreads();

  int n_eval = 0, n_slow = 0, n_corner = 0;
  for (int k = 0; k < p.n_steps; ++k) {
    const int t1 = p.t0 + k + 1;
    // ================= phase A: one thread per agent =================
    if (tid == 0) s_nq = 0;               // last read in phase B2 of the previous step, before its closing barrier
    for (int a = tid; a < Ap; a += FUSED_NT) {
      if (k > 0 && a < A) fused_flush_metrics(p, rb, k - 1, a, A, s_valid, s_ov, s_csd, s_anyov, s_anyoff);
      s_ov[a] = 0;
      bool vn = false;
      float cs = 1.f, sn = 0.f, hl = 0.f, hw = 0.f, xn = 0.f, yn = 0.f;
      if (a < A) {
        const int64_t o = sb + (int64_t)t1 * A + a;
        const int64_t ak = (int64_t)b * p.n_steps + k;
        const bool use_dyn = p.av[ak * A + a] != 0 && s_valid[a] != 0;          // D8
        const float lx = p.log.x[o], ly = p.log.y[o];
        const uint8_t lvalid = p.log.valid[o];
        float thn, vxn, vyn, ln, wd;
        if (use_dyn) {
          const float* act = p.actions + ak * p.C * A + a;
          const float a2 = p.C > 2 ? act[2 * (int64_t)A] : 0.f;
          wm_dyn_step(p.dyn, sx[a], sy[a], syaw[a], svx[a], svy[a], ss[a], sc[a], act[0], act[A], a2, xn, yn, thn,
                      vxn, vyn, sn, cs);
          ln = slen[a]; wd = swid[a];
          vn = true;                                                            // D9
        } else {                                                                // log playback, L164
          xn = lx; yn = ly; thn = p.log.yaw[o]; vxn = p.log.vel_x[o]; vyn = p.log.vel_y[o];
          ln = p.log.length[o]; wd = p.log.width[o];
          vn = lvalid != 0;
          if (vn) sincosf(thn, &sn, &cs);
        }
        p.sim.x[o] = xn; p.sim.y[o] = yn; p.sim.yaw[o] = thn; p.sim.vel_x[o] = vxn; p.sim.vel_y[o] = vyn;
        p.sim.length[o] = ln; p.sim.width[o] = wd; p.sim.valid[o] = (uint8_t)vn;
        const bool ldv = vn && lvalid != 0;                                     // a5, L106
        const float d = ldv ? wm_logdiv(xn, yn, lx, ly) : 0.f;
        if (p.out.log_div) p.out.log_div[rb + (int64_t)k * A + a] = d;
        if (ldv) { s_sum[a] += (double)d; s_cnt[a] += 1; }
        sx[a] = xn; sy[a] = yn; syaw[a] = thn; svx[a] = vxn; svy[a] = vyn; slen[a] = ln; swid[a] = wd;
        if (vn) { hl = 0.5f * ln; hw = 0.5f * wd; } else { cs = 1.f; sn = 0.f; xn = 0.f; yn = 0.f; }
      }
      float ax = 0.f, ay = 0.f, bx = 0.f, by = 0.f;
      if (vn) wm_box_offsets_sc(sn, cs, slen[a], swid[a], ax, ay, bx, by);
      else { sx[a] = xn; sy[a] = yn; }                  // invalid slots: finite zeros for the overlap loads (D10)
      sc[a] = cs; ss[a] = sn; shl[a] = hl; shw[a] = hw; srad[a] = sqrtf(fmaf(hl, hl, hw * hw));
      oax[a] = ax; oay[a] = ay; obx[a] = bx; oby[a] = by;
      s_valid[a] = vn;
      const uint32_t w = __ballot_sync(0xffffffffu, vn);
      if (lane == 0) s_vw[a >> 5] = w;
    }
    __syncthreads();
    // ================= phase B1: corners (a4), candidate walk =================
    for (int c0 = 0; c0 < 4 * Ap; c0 += FUSED_NT) {
      if (c0 + (tid & ~31) >= 4 * Ap) continue;                                 // warp-uniform (4 Ap % 128 == 0)
      const int c = c0 + tid, a = c >> 2, kk = c & 3;
      const bool v = s_valid[a] != 0;
      const float ox = (kk & 1) ? obx[a] : oax[a], oy = (kk & 1) ? oby[a] : oay[a];
      const float offx = (kk & 2) ? -ox : ox, offy = (kk & 2) ? -oy : oy;
      float best; int bs;
      const bool slow = wm_grid_fast(gv, v, sx[a], sy[a], offx, offy, best, bs, n_eval);
      n_slow += slow; n_corner += v;
      if (slow) { if (atomicOr(&s_qm[a], 1u << kk) == 0u) s_q[atomicAdd(&s_nq, 1)] = a; }
      else s_csd[c] = v ? wm_grid_finish(gv, sx[a], sy[a], offx, offy, best, bs) : 0.f;
    }
    // ================= phase B: pairs (a3) =================
    const int ntask = nb * (nb + 1) / 2 * FUSED_SUB;
    for (int task = warp; task < ntask; task += FUSED_NT / 32) {
      const int tile = task / FUSED_SUB, q = task % FUSED_SUB;
      int I = 0, rem = tile;
      while (rem >= nb - I) { rem -= nb - I; ++I; }
      const int J = I + rem;
      const uint32_t vi = s_vw[I] & (0xffu << (q * 8)), vj = s_vw[J];
      if (vi == 0 || vj == 0) continue;
      const int j = J * 32 + lane;
      const float xj = sx[j], yj = sy[j], cj = sc[j], sj = ss[j], hlj = shl[j], hwj = shw[j], rj = srad[j];
      const bool jv = (vj >> lane) & 1u;
      bool any_j = false;
      for (int ii = q * 8; ii < q * 8 + 8; ++ii) {
        if (!((vi >> ii) & 1u)) continue;               // warp-uniform skip of invalid i
        const int i = I * 32 + ii;
        const float dx = xj - sx[i], dy = yj - sy[i];
        bool ov = jv && i != j && wm_circles_touch(dx, dy, rj + srad[i]);
        if (!__any_sync(0xffffffffu, ov)) continue;     // far apart
        ov = ov && wm_sat_overlap(dx, dy, sc[i], ss[i], shl[i], shw[i], cj, sj, hlj, hwj);
        any_j |= ov;
        if (__any_sync(0xffffffffu, ov) && lane == 0) s_ov[i] = 1u;
      }
      if (any_j) s_ov[j] = 1u;
    }
    __syncthreads();
    // ================= phase B2: queued agents, one warp each =================
    const int nq = s_nq;
    for (int i = warp; i < nq; i += FUSED_NT / 32) {
      const int a = s_q[i];
      const uint32_t qm = s_qm[a];
      const float offx[4] = {oax[a], obx[a], -oax[a], -obx[a]}, offy[4] = {oay[a], oby[a], -oay[a], -oby[a]};
      float best[4]; int bs[4], ne = 0;
      wm_grid_search_warp4(gv, sx[a], sy[a], offx, offy, srad[a], best, bs, ne);
      if (lane < 4) {
        const float ox = lane == 0 ? offx[0] : lane == 1 ? offx[1] : lane == 2 ? offx[2] : offx[3];
        const float oy = lane == 0 ? offy[0] : lane == 1 ? offy[1] : lane == 2 ? offy[2] : offy[3];
        const float bb = lane == 0 ? best[0] : lane == 1 ? best[1] : lane == 2 ? best[2] : best[3];
        const int bi = lane == 0 ? bs[0] : lane == 1 ? bs[1] : lane == 2 ? bs[2] : bs[3];
        if ((qm >> lane) & 1u) s_csd[4 * a + lane] = wm_grid_finish(gv, sx[a], sy[a], ox, oy, bb, bi);
      }
      if (lane == 0) { s_qm[a] = 0; n_eval += ne; }
    }
    __syncthreads();
  }

  // ---- epilogue: last overlap row, aggregates (D21) ----
  for (int a = tid; a < A; a += FUSED_NT) {
    fused_flush_metrics(p, rb, p.n_steps - 1, a, A, s_valid, s_ov, s_csd, s_anyov, s_anyoff);
    const int64_t o = (int64_t)b * A + a;
    if (p.out.any_overlap) p.out.any_overlap[o] = s_anyov[a];
    if (p.out.any_offroad) p.out.any_offroad[o] = s_anyoff[a];
    if (p.out.ade) p.out.ade[o] = s_cnt[a] ? (float)(s_sum[a] / s_cnt[a]) : 0.f;
  }
  if (p.stats) {
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

cudaError_t wm_launch_rollout_fused(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t0, int n_steps,
                                    const float* actions, const uint8_t* action_valid, const wm_rollout_out& out,
                                    cudaStream_t s) {
  FusedParams p;
  p.log = log; p.sim = sim; p.t0 = t0; p.n_steps = n_steps;
  p.C = h->cfg.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  p.actions = actions; p.av = action_valid; p.out = out;
  p.dyn = WmDynCfg{h->cfg.dynamics, h->cfg.dt, h->cfg.max_accel, h->cfg.max_curvature};
  p.segrec = h->segrec; p.chunks = h->chunks; p.cells = h->cells; p.pool = h->pool; p.gridp = h->gridp;
  p.seg_cap = h->seg_tiles * WM_TILE_SEGS;
  p.stats = h->stats_on ? h->cull_stats : nullptr;
  const size_t smem = fused_smem_bytes(sim.A);
  static bool configured = false;
  if (!configured) {
    cudaError_t e = cudaFuncSetAttribute(k_rollout_fused, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)fused_smem_bytes(1024));
    if (e != cudaSuccess) return e;
    configured = true;
  }
  k_rollout_fused<<<sim.B, FUSED_NT, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
