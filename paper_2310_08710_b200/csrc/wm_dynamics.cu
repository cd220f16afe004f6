// reset (a0), dynamics step (a1, a2) with optional fused log divergence (a5), aggregates (a8).
// One thread per (scenario, agent): these kernels move ~12 KB per scenario-step and are
// HBM/latency bound; rows are time-major so a warp touches one contiguous 128 B line per field.
#include "wm_device.cuh"

// ---------------------------------------------------------------------------------------
// a0 reset(scenario), PAPER.md L122 / L78.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_reset(wm_traj log, wm_traj sim, int history) {
  // one CTA per (scenario, chunk of 1024 row elements): no per-element division; rows [0, history) are
  // copied, the rest cleared.  HBM-write bound (the whole simulated trajectory is written once).
  const int64_t TA = (int64_t)sim.T * sim.A, HA = (int64_t)history * sim.A;
  const int64_t base = (int64_t)blockIdx.y * TA;
  for (int64_t e = (int64_t)blockIdx.x * 1024 + threadIdx.x; e < TA; e += (int64_t)gridDim.x * 1024) {
#pragma unroll
    for (int q = 0; q < 4; ++q) {
      const int64_t r = e + q * 256;
      if (r >= TA) break;
      const int64_t i = base + r;
      const bool c = r < HA;
      sim.x[i] = c ? log.x[i] : 0.f;
      sim.y[i] = c ? log.y[i] : 0.f;
      sim.yaw[i] = c ? log.yaw[i] : 0.f;
      sim.vel_x[i] = c ? log.vel_x[i] : 0.f;
      sim.vel_y[i] = c ? log.vel_y[i] : 0.f;
      sim.length[i] = c ? log.length[i] : 0.f;
      sim.width[i] = c ? log.width[i] : 0.f;
      sim.valid[i] = c ? log.valid[i] : (uint8_t)0;
    }
  }
}

cudaError_t wm_launch_reset(wm_handle* h, const wm_traj& log, const wm_traj& sim, int history, cudaStream_t s) {
  const int64_t TA = (int64_t)sim.T * sim.A;
  int gx = (int)((TA + 1023) / 1024);
  if (gx > 64) gx = 64;
  k_reset<<<dim3(gx, sim.B), 256, 0, s>>>(log, sim, history);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// a1 / a2 step(state, action); Eq. 2 (L339-L350) and Eq. 1 (L324-L333).
// ---------------------------------------------------------------------------------------
struct StepParams {
  wm_row cur;       // sim row t
  wm_row nxt_log;   // log row t+1
  wm_row_mut nxt;   // sim row t+1
  const float* action; int64_t act_stride_b;
  const uint8_t* av;   int64_t av_stride_b;
  float* ld_dist; uint8_t* ld_valid; int64_t ld_stride_b;
  int B, A, dynamics;
  float dt, max_accel, max_curvature;
};

__global__ void __launch_bounds__(256) k_step(StepParams p) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= (int64_t)p.B * p.A) return;
  const int b = (int)(i / p.A), a = (int)(i % p.A);
  const int64_t c = (int64_t)b * p.cur.stride_b + a;       // same offset in all three rows
  const bool use_dyn = p.av[(int64_t)b * p.av_stride_b + a] != 0 && p.cur.valid[c] != 0;
  const float lx = p.nxt_log.x[c], ly = p.nxt_log.y[c];
  const uint8_t lvalid = p.nxt_log.valid[c];
  float xn, yn, thn, vxn, vyn, ln, wn;
  uint8_t vn;
  if (use_dyn) {
    const float x = p.cur.x[c], y = p.cur.y[c], th = p.cur.yaw[c];
    const float vx = p.cur.vel_x[c], vy = p.cur.vel_y[c];
    const float* act = p.action + (int64_t)b * p.act_stride_b + a;
    float sn, cs, s1, c1;
    sincosf(th, &sn, &cs);
    const WmDynCfg dc{p.dynamics, p.dt, p.max_accel, p.max_curvature};
    const float a2 = p.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 0.f : act[2 * (int64_t)p.A];
    wm_dyn_step(dc, x, y, th, vx, vy, sn, cs, act[0], act[p.A], a2, xn, yn, thn, vxn, vyn, s1, c1);
    ln = p.cur.length[c];
    wn = p.cur.width[c];
    vn = 1;                                            // D9
  } else {                                             // log playback, L164 / D8
    xn = lx; yn = ly; thn = p.nxt_log.yaw[c];
    vxn = p.nxt_log.vel_x[c]; vyn = p.nxt_log.vel_y[c];
    ln = p.nxt_log.length[c]; wn = p.nxt_log.width[c];
    vn = lvalid;
  }
  p.nxt.x[c] = xn; p.nxt.y[c] = yn; p.nxt.yaw[c] = thn;
  p.nxt.vel_x[c] = vxn; p.nxt.vel_y[c] = vyn;
  p.nxt.length[c] = ln; p.nxt.width[c] = wn; p.nxt.valid[c] = vn;
  if (p.ld_dist) {                                     // fused a5 on row t+1, L106
    const bool v = vn != 0 && lvalid != 0;
    float d = 0.f;
    if (v) d = wm_logdiv(xn, yn, lx, ly);
    p.ld_dist[(int64_t)b * p.ld_stride_b + a] = d;
    if (p.ld_valid) p.ld_valid[(int64_t)b * p.ld_stride_b + a] = v;
  }
}

cudaError_t wm_launch_step(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t,
                           const float* action, int64_t act_stride_b, const uint8_t* av,
                           int64_t av_stride_b, float* ld_dist, uint8_t* ld_valid,
                           int64_t ld_stride_b, cudaStream_t s) {
  StepParams p;
  p.cur = wm_make_row(sim, t);
  p.nxt_log = wm_make_row(log, t + 1);
  p.nxt = wm_make_row_mut(sim, t + 1);
  p.action = action; p.act_stride_b = act_stride_b;
  p.av = av; p.av_stride_b = av_stride_b;
  p.ld_dist = ld_dist; p.ld_valid = ld_valid; p.ld_stride_b = ld_stride_b;
  p.B = sim.B; p.A = sim.A; p.dynamics = h->cfg.dynamics;
  p.dt = h->cfg.dt; p.max_accel = h->cfg.max_accel; p.max_curvature = h->cfg.max_curvature;
  const int64_t n = (int64_t)sim.B * sim.A;
  k_step<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// a5 log divergence.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_logdiv(wm_row lg, wm_row sm, int B, int A, float* dist, uint8_t* valid, int64_t stride_b) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= (int64_t)B * A) return;
  const int b = (int)(i / A), a = (int)(i % A);
  const int64_t cs = (int64_t)b * sm.stride_b + a, cl = (int64_t)b * lg.stride_b + a;
  const bool v = sm.valid[cs] != 0 && lg.valid[cl] != 0;
  float d = 0.f;
  if (v) d = wm_logdiv(sm.x[cs], sm.y[cs], lg.x[cl], lg.y[cl]);
  dist[(int64_t)b * stride_b + a] = d;
  if (valid) valid[(int64_t)b * stride_b + a] = v;
}

cudaError_t wm_launch_logdiv(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t, float* dist,
                             uint8_t* valid, int64_t stride_b, cudaStream_t s) {
  const int64_t n = (int64_t)sim.B * sim.A;
  k_logdiv<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(wm_make_row(log, t), wm_make_row(sim, t), sim.B, sim.A, dist, valid, stride_b);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// a8 aggregates over the n_steps metric rows (D21): any-overlap, any-offroad, ADE.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_aggregate(int B, int A, int n_steps, wm_rollout_out out, const uint8_t* ld_valid) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= (int64_t)B * A) return;
  const int b = (int)(i / A), a = (int)(i % A);
  uint8_t ov = 0, off = 0;
  double sum = 0.0;
  int cnt = 0;
  for (int s = 0; s < n_steps; ++s) {
    const int64_t o = ((int64_t)b * n_steps + s) * A + a;
    if (out.overlap) ov |= out.overlap[o];
    if (out.offroad) off |= out.offroad[o];
    if (out.log_div && ld_valid[o]) { sum += (double)out.log_div[o]; cnt++; }
  }
  if (out.any_overlap) out.any_overlap[i] = ov;
  if (out.any_offroad) out.any_offroad[i] = off;
  if (out.ade) out.ade[i] = cnt ? (float)(sum / cnt) : 0.f;
}

cudaError_t wm_launch_aggregate(wm_handle* h, int B, int A, int n_steps, const wm_rollout_out& out,
                                const uint8_t* ld_valid_rows, cudaStream_t s) {
  const int64_t n = (int64_t)B * A;
  k_aggregate<<<(unsigned)((n + 255) / 256), 256, 0, s>>>(B, A, n_steps, out, ld_valid_rows);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Expert actor (L204; L335, Eq. 3) and kinematic-infeasibility metric (L104): one thread per
// (scenario, step, agent); two state rows in, one action / metric row out.  HBM bound.
// ---------------------------------------------------------------------------------------
struct InvParams {
  wm_traj tr;
  int t, n_steps, dynamics;
  float dt, max_accel, max_curvature;
  float* action; uint8_t* valid;                // expert: [B][n][C][A], [B][n][A]
  float* accel; float* curvature; uint8_t* flag;   // metric: [B][n][A]
};

constexpr int INV_CHUNK = 8;      // consecutive steps per thread: every state row is loaded once

template <bool METRIC>
__global__ void __launch_bounds__(256) k_inverse(InvParams p) {
  const int A = p.tr.A, nchunk = (p.n_steps + INV_CHUNK - 1) / INV_CHUNK;
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= (int64_t)p.tr.B * nchunk * A) return;
  const int a = (int)(i % A), ch = (int)((i / A) % nchunk), b = (int)(i / ((int64_t)A * nchunk));
  const int s0 = ch * INV_CHUNK, s1 = min(s0 + INV_CHUNK, p.n_steps);
  const bool delta = !METRIC && p.dynamics != WM_DYN_INVERTIBLE_BICYCLE;
  const int C = p.dynamics == WM_DYN_INVERTIBLE_BICYCLE ? 2 : 3;
  int64_t r = ((int64_t)b * p.tr.T + (METRIC ? p.t + s0 - 1 : p.t + s0)) * A + a;      // first row of the chunk
  // loads are unconditional (independent of `valid`, so they pipeline); an invalid slot's values
  // never reach an output (D10): every use below is behind v
  const float* pa = delta ? p.tr.x : p.tr.vel_x;
  const float* pb = delta ? p.tr.y : p.tr.vel_y;
  bool v0 = p.tr.valid[r] != 0;
  float th = p.tr.yaw[r], vx = pa[r], vy = pb[r];
  float x = vx, y = vy;
#pragma unroll
  for (int s = s0; s < s0 + INV_CHUNK; ++s) {
    if (s >= s1) break;
    r += A;
    const bool v1 = p.tr.valid[r] != 0;
    const float th1 = p.tr.yaw[r], vx1 = pa[r], vy1 = pb[r];
    const float x1 = vx1, y1 = vy1;
    const bool v = v0 && v1;
    const int64_t o = ((int64_t)b * p.n_steps + s) * A + a;
    if (METRIC) {
      float acc = 0.f, kap = 0.f;
      if (v) wm_inverse_bicycle(p.dt, th, vx, vy, vx1, vy1, acc, kap);
      if (p.accel) p.accel[o] = acc;
      if (p.curvature) p.curvature[o] = kap;
      p.flag[o] = (uint8_t)(v && (fabsf(acc) > p.max_accel || fabsf(kap) > p.max_curvature));
    } else {
      float* act = p.action + (((int64_t)b * p.n_steps + s) * C) * A + a;
      float a0 = 0.f, a1 = 0.f, a2 = 0.f;
      if (v) {
        if (!delta) wm_inverse_bicycle(p.dt, th, vx, vy, vx1, vy1, a0, a1);
        else {                                                 // L335 in the body frame (D2)
          float sn = 0.f, cs = 1.f;                            // DeltaGlobal: the plain difference
          if (p.dynamics == WM_DYN_DELTA_LOCAL) sincosf(th, &sn, &cs);
          const float Dx = x1 - x, Dy = y1 - y;
          a0 = fmaf(cs, Dx, sn * Dy); a1 = fmaf(cs, Dy, -sn * Dx); a2 = th1 - th;
        }
      }
      act[0] = a0; act[A] = a1;
      if (C == 3) act[2 * (int64_t)A] = a2;
      p.valid[o] = (uint8_t)v;
    }
    v0 = v1; th = th1; vx = vx1; vy = vy1; x = x1; y = y1;
  }
}

cudaError_t wm_launch_expert(wm_handle* h, const wm_traj& tr, int t, int n_steps, float* action, uint8_t* valid, cudaStream_t s) {
  InvParams p{tr, t, n_steps, h->cfg.dynamics, h->cfg.dt, h->cfg.max_accel, h->cfg.max_curvature, action, valid, nullptr, nullptr, nullptr};
  const int64_t n = (int64_t)tr.B * ((n_steps + INV_CHUNK - 1) / INV_CHUNK) * tr.A;
  k_inverse<false><<<(unsigned)((n + 255) / 256), 256, 0, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}

cudaError_t wm_launch_kinematic(wm_handle* h, const wm_traj& tr, int t, int n_steps, float* accel, float* curvature,
                                uint8_t* flag, cudaStream_t s) {
  InvParams p{tr, t, n_steps, h->cfg.dynamics, h->cfg.dt, h->cfg.max_accel, h->cfg.max_curvature, nullptr, nullptr, accel, curvature, flag};
  const int64_t n = (int64_t)tr.B * ((n_steps + INV_CHUNK - 1) / INV_CHUNK) * tr.A;
  k_inverse<true><<<(unsigned)((n + 255) / 256), 256, 0, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Route-progress ratio, PAPER.md L96 (readings D33-D35).  One warp per agent: three closest-point
// searches over the agent's P path points (the simulated position and the first / last valid logged
// position) in one pass, lanes over points, (key, index) argmin by shuffles with the lower index
// winning ties.  Reads 9 B per path point once per agent: HBM bound.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_route_progress(wm_traj log, wm_traj sim, int t, wm_paths pa, float* ratio, uint8_t* valid) {
  // one CTA per (scenario, 32 consecutive agents): the first / last valid logged row of the 32 agents
  // from coalesced 32-byte pieces of the valid plane (lane = agent, warps over rows), then 4 agents per warp
  __shared__ int s_tf[32], s_tl[32];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int A = sim.A, T = sim.T, b = blockIdx.y, a0 = blockIdx.x * 32;
  if (threadIdx.x < 32) { s_tf[threadIdx.x] = 0x7fffffff; s_tl[threadIdx.x] = -1; }
  __syncthreads();
  {
    int tf = 0x7fffffff, tl = -1;                            // D34
    if (a0 + lane < A)
      for (int k = warp; k < T; k += 8)
        if (log.valid[((int64_t)b * T + k) * A + a0 + lane] != 0) { tf = min(tf, k); tl = max(tl, k); }
    if (tl >= 0) { atomicMin(&s_tf[lane], tf); atomicMax(&s_tl[lane], tl); }
  }
  __syncthreads();
  for (int q = 0; q < 4; ++q) {
    const int ai = warp * 4 + q, a = a0 + ai;
    if (a >= A) break;                                       // warp-uniform
    const int tf = s_tf[ai], tl = s_tl[ai];
    const int64_t rs = ((int64_t)b * T + t) * A + a;
    const bool sv = sim.valid[rs] != 0 && tl >= 0;
    float qx[3] = {0.f, 0.f, 0.f}, qy[3] = {0.f, 0.f, 0.f};
    if (sv) {
      const int64_t r0 = ((int64_t)b * T + tf) * A + a, r1 = ((int64_t)b * T + tl) * A + a;
      qx[0] = sim.x[rs]; qy[0] = sim.y[rs]; qx[1] = log.x[r0]; qy[1] = log.y[r0]; qx[2] = log.x[r1]; qy[2] = log.y[r1];
    }
    const int64_t po = ((int64_t)b * pa.A + a) * pa.P;
    unsigned long long best[3] = {~0ull, ~0ull, ~0ull};     // (key bits << 32) | index: keys are >= +0, so the bits order as floats
    if (sv)
      for (int i = lane; i < pa.P; i += 32) {
        if (pa.valid[po + i] == 0) continue;
        const float px = pa.x[po + i], py = pa.y[po + i];
#pragma unroll
        for (int c = 0; c < 3; ++c) {
          const float dx = __fsub_rn(px, qx[c]), dy = __fsub_rn(py, qy[c]);
          const unsigned long long kv = ((unsigned long long)__float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx))) << 32) | (unsigned)i;
          best[c] = min(best[c], kv);                        // ties -> lower index (D33)
        }
      }
#pragma unroll
    for (int c = 0; c < 3; ++c)
#pragma unroll
      for (int d = 16; d > 0; d >>= 1) best[c] = min(best[c], __shfl_xor_sync(0xffffffffu, best[c], d));
    if (lane == 0) {
      float r = 0.f;
      uint8_t v = 0;
      if (sv && best[0] != ~0ull) {
        const float dx = pa.arc_len[po + (int)(best[0] & 0xffffffffu)], dp = pa.arc_len[po + (int)(best[1] & 0xffffffffu)],
                    dq = pa.arc_len[po + (int)(best[2] & 0xffffffffu)];
        if (dq != dp) { r = (dx - dp) / (dq - dp); v = 1; }   // D35
      }
      ratio[(int64_t)b * A + a] = r;
      valid[(int64_t)b * A + a] = v;
    }
  }
}

cudaError_t wm_launch_route_progress(wm_handle* h, const wm_traj& log, const wm_traj& sim, int t, const wm_paths& pa, float* ratio,
                                     uint8_t* valid, cudaStream_t s) {
  k_route_progress<<<dim3((sim.A + 31) / 32, sim.B), 256, 0, s>>>(log, sim, t, pa, ratio, valid);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// Off-route metric, PAPER.md L98 (reading D36: thresholds are arguments).  One warp per agent, lanes
// over the points of its on-route and off-route path; float32 keys, min by shuffles.
// ---------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_offroute(wm_traj sim, int t, wm_paths on, wm_paths off, int has_off, float max_dist,
                                                  float margin, float* dist_on, uint8_t* flag) {
  const int lane = threadIdx.x & 31;
  const int64_t w = (blockIdx.x * (int64_t)blockDim.x + threadIdx.x) >> 5;
  const int A = sim.A;
  if (w >= (int64_t)sim.B * A) return;
  const int b = (int)(w / A), a = (int)(w % A);
  const int64_t rs = ((int64_t)b * sim.T + t) * A + a;
  const bool sv = sim.valid[rs] != 0;
  const float qx = sv ? sim.x[rs] : 0.f, qy = sv ? sim.y[rs] : 0.f;
  uint32_t k_on = 0xffffffffu, k_off = 0xffffffffu;          // float bits of the smallest key (keys are >= +0)
  if (sv) {
    const int64_t po = ((int64_t)b * on.A + a) * on.P;
    for (int i = lane; i < on.P; i += 32)
      if (on.valid[po + i] != 0) {
        const float dx = __fsub_rn(on.x[po + i], qx), dy = __fsub_rn(on.y[po + i], qy);
        k_on = min(k_on, __float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx))));
      }
    if (has_off) {
      const int64_t pf = ((int64_t)b * off.A + a) * off.P;
      for (int i = lane; i < off.P; i += 32)
        if (off.valid[pf + i] != 0) {
          const float dx = __fsub_rn(off.x[pf + i], qx), dy = __fsub_rn(off.y[pf + i], qy);
          k_off = min(k_off, __float_as_uint(__fmaf_rn(dy, dy, __fmul_rn(dx, dx))));
        }
    }
  }
  k_on = __reduce_min_sync(0xffffffffu, k_on); k_off = __reduce_min_sync(0xffffffffu, k_off);
  if (lane == 0) {
    float d = 0.f;
    uint8_t f = 0;
    if (sv && k_on != 0xffffffffu) {
      d = __fsqrt_rn(__uint_as_float(k_on));
      const float d_off = k_off != 0xffffffffu ? __fsqrt_rn(__uint_as_float(k_off)) : __int_as_float(0x7f800000);
      f = (uint8_t)(d > max_dist || __fadd_rn(d_off, margin) < d);    // L98
    }
    if (dist_on) dist_on[(int64_t)b * A + a] = d;
    flag[(int64_t)b * A + a] = f;
  }
}

cudaError_t wm_launch_offroute(wm_handle* h, const wm_traj& sim, int t, const wm_paths& on, const wm_paths* off, float max_dist,
                               float margin, float* dist_on, uint8_t* flag, cudaStream_t s) {
  const int64_t warps = (int64_t)sim.B * sim.A;
  k_offroute<<<(unsigned)((warps + 7) / 8), 256, 0, s>>>(sim, t, on, off ? *off : on, off != nullptr, max_dist, margin, dist_on, flag);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// IDM reactive sim agent, PAPER.md L110-L112 + ref. [51]; readings D37-D41.  One warp per
// (scenario, agent): its path is staged in shared memory, every other agent is projected on it with
// lanes over the path segments (agents outside the path's bounding box + their lateral reach are
// skipped: they cannot be within it of any segment).  Projections and the lead decision are float32,
// operation for operation as DESIGN.md (D38, D39) lays them down.
// ---------------------------------------------------------------------------------------
struct IdmParams {
  wm_traj sim; int t; wm_paths pa; const uint8_t* idm_valid; wm_idm_params prm; float dt;
  float* accel; int32_t* lead;
};

struct IdmProj { int k; float u, d2, sigma; };

// all lanes get the same result; sp: the warp's staged path, [0,P) x, [P,2P) y, [2P,3P) arc, then P valid bytes
__device__ __forceinline__ IdmProj idm_project(const float* sp, const uint8_t* sv, int P, float qx, float qy) {
  const int lane = threadIdx.x & 31;
  unsigned long long best = ~0ull;
  for (int k = lane; k + 1 < P; k += 32) {
    if (sv[k] == 0 || sv[k + 1] == 0) continue;
    const float ex = __fsub_rn(sp[k + 1], sp[k]), ey = __fsub_rn(sp[P + k + 1], sp[P + k]);
    const float wx = __fsub_rn(qx, sp[k]), wy = __fsub_rn(qy, sp[P + k]);
    const float ee = __fmaf_rn(ey, ey, __fmul_rn(ex, ex)), dot = __fmaf_rn(wy, ey, __fmul_rn(wx, ex));
    float u = 0.f;
    if (ee > 0.f) u = fminf(fmaxf(__fdiv_rn(dot, ee), 0.f), 1.f);
    const float rx = __fmaf_rn(-u, ex, wx), ry = __fmaf_rn(-u, ey, wy);
    const float d2 = __fmaf_rn(ry, ry, __fmul_rn(rx, rx));
    best = min(best, ((unsigned long long)__float_as_uint(d2) << 32) | (unsigned)k);     // ties -> lower segment (D38)
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) best = min(best, __shfl_xor_sync(0xffffffffu, best, d));
  IdmProj r{-1, 0.f, __int_as_float(0x7f800000), 0.f};
  if (best != ~0ull) {
    const int k = (int)(best & 0xffffffffu);
    r.k = k; r.d2 = __uint_as_float((uint32_t)(best >> 32));
    const float ex = __fsub_rn(sp[k + 1], sp[k]), ey = __fsub_rn(sp[P + k + 1], sp[P + k]);
    const float wx = __fsub_rn(qx, sp[k]), wy = __fsub_rn(qy, sp[P + k]);
    const float ee = __fmaf_rn(ey, ey, __fmul_rn(ex, ex)), dot = __fmaf_rn(wy, ey, __fmul_rn(wx, ex));
    if (ee > 0.f) r.u = fminf(fmaxf(__fdiv_rn(dot, ee), 0.f), 1.f);
    r.sigma = __fmaf_rn(r.u, __fsub_rn(sp[2 * P + k + 1], sp[2 * P + k]), sp[2 * P + k]);
  }
  return r;
}

__global__ void __launch_bounds__(256) k_idm_step(IdmParams p) {
  extern __shared__ __align__(16) float s_path[];            // per warp: 3 P floats + P bytes (padded to 4)
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const int A = p.sim.A, T = p.sim.T, P = p.pa.P;
  const int64_t w = blockIdx.x * (int64_t)(blockDim.x >> 5) + warp;
  if (w >= (int64_t)p.sim.B * A) return;
  const int b = (int)(w / A), i = (int)(w % A);
  const int64_t o = (int64_t)b * A + i, r0 = ((int64_t)b * T + p.t) * A + i, r1 = r0 + A;
  if (lane == 0) { if (p.accel) p.accel[o] = 0.f; if (p.lead) p.lead[o] = -1; }
  if (p.idm_valid[o] == 0 || p.sim.valid[r0] == 0) return;     // warp-uniform
  const int stride = 3 * P + ((P + 3) >> 2);
  float* sp = s_path + (size_t)warp * stride;
  uint8_t* sv = (uint8_t*)(sp + 3 * P);
  const int64_t po = ((int64_t)b * p.pa.A + i) * P;
  float bx0 = 3.0e38f, by0 = 3.0e38f, bx1 = -3.0e38f, by1 = -3.0e38f;
  for (int k = lane; k < P; k += 32) {
    const uint8_t v = p.pa.valid[po + k];
    const float x = p.pa.x[po + k], y = p.pa.y[po + k];
    sp[k] = x; sp[P + k] = y; sp[2 * P + k] = p.pa.arc_len[po + k]; sv[k] = v;
    if (v) { bx0 = fminf(bx0, x); bx1 = fmaxf(bx1, x); by0 = fminf(by0, y); by1 = fmaxf(by1, y); }
  }
#pragma unroll
  for (int d = 16; d > 0; d >>= 1) {
    bx0 = fminf(bx0, __shfl_xor_sync(0xffffffffu, bx0, d)); by0 = fminf(by0, __shfl_xor_sync(0xffffffffu, by0, d));
    bx1 = fmaxf(bx1, __shfl_xor_sync(0xffffffffu, bx1, d)); by1 = fmaxf(by1, __shfl_xor_sync(0xffffffffu, by1, d));
  }
  __syncwarp();
  const float xi = p.sim.x[r0], yi = p.sim.y[r0], Li = p.sim.length[r0], Wi = p.sim.width[r0];
  const IdmProj self = idm_project(sp, sv, P, xi, yi);
  if (self.k < 0) return;                                      // D41: no path segment
  // ---- lead object (D39) ----
  int lead = -1;
  float gap = __int_as_float(0x7f800000);
  const int64_t rb = ((int64_t)b * T + p.t) * A;
  for (int jb = 0; jb < A; jb += 32) {                        // lanes over the other agents: who can matter at all?
    const int jl = jb + lane;
    bool pass = jl < A && jl != i && p.sim.valid[rb + jl] != 0;
    float xl = 0.f, yl = 0.f, wl = 0.f, ll = 0.f;
    if (pass) {
      xl = p.sim.x[rb + jl]; yl = p.sim.y[rb + jl]; wl = p.sim.width[rb + jl]; ll = p.sim.length[rb + jl];
      const float reach = fmaf(__fmul_rn(0.5f, __fadd_rn(Wi, wl)), 1.001f, 1e-3f);   // outside the inflated box: farther than lat_max from every segment
      pass = !(xl < bx0 - reach || xl > bx1 + reach || yl < by0 - reach || yl > by1 + reach);
    }
    uint32_t todo = __ballot_sync(0xffffffffu, pass);
    while (todo) {                                             // ascending j: ties -> lower index (D39)
      const int src = __ffs(todo) - 1;
      todo &= todo - 1;
      const float xj = __shfl_sync(0xffffffffu, xl, src), yj = __shfl_sync(0xffffffffu, yl, src);
      const float wj = __shfl_sync(0xffffffffu, wl, src), lj = __shfl_sync(0xffffffffu, ll, src);
      const float lat_max = __fmul_rn(0.5f, __fadd_rn(Wi, wj));
      const IdmProj pj = idm_project(sp, sv, P, xj, yj);
      if (!(pj.sigma > self.sigma) || pj.d2 > __fmul_rn(lat_max, lat_max)) continue;
      const float g = __fsub_rn(__fsub_rn(pj.sigma, self.sigma), __fmul_rn(0.5f, __fadd_rn(Li, lj)));
      if (g < gap) { gap = g; lead = jb + src; }
    }
  }
  if (lane != 0) return;
  // ---- IDM acceleration (ref. [51]) and the move along the path (D40) ----
  const wm_idm_params& q = p.prm;
  const float vx = p.sim.vel_x[r0], vy = p.sim.vel_y[r0], v = sqrtf(fmaf(vx, vx, vy * vy));
  float acc = 1.f - powf(v / q.v0, q.delta);
  if (lead >= 0) {
    const float lx = p.sim.vel_x[rb + lead], ly = p.sim.vel_y[rb + lead], vl = sqrtf(fmaf(lx, lx, ly * ly));
    const float sstar = q.s0 + fmaxf(0.f, fmaf(v, q.T, v * (v - vl) / (2.f * sqrtf(q.a_max * q.b))));
    const float sg = sstar / fmaxf(gap, 0.1f);
    acc -= sg * sg;
  }
  acc = fminf(fmaxf(acc * q.a_max, -q.b_max), q.a_max);
  const float v1 = fmaxf(0.f, fmaf(acc, p.dt, v));
  const float target = fmaf(0.5f * (v + v1), p.dt, self.sigma);
  int ks = -1;
  for (int k = self.k; k + 1 < P; ++k)
    if (sv[k] != 0 && sv[k + 1] != 0 && sp[2 * P + k + 1] > target) { ks = k; break; }
  float xn, yn, yawn;
  if (ks >= 0) {
    const float ex = sp[ks + 1] - sp[ks], ey = sp[P + ks + 1] - sp[P + ks];
    const float len = sp[2 * P + ks + 1] - sp[2 * P + ks];
    const float u = fminf(fmaxf((target - sp[2 * P + ks]) / len, 0.f), 1.f);
    xn = fmaf(u, ex, sp[ks]); yn = fmaf(u, ey, sp[P + ks]); yawn = atan2f(ey, ex);
  } else {                                                     // past the end: the last path point, yaw kept
    int kl = self.k + 1;
    for (int k = self.k + 1; k < P; ++k) { if (sv[k] != 0 && sv[k - 1] != 0) kl = k; else break; }
    xn = sp[kl]; yn = sp[P + kl]; yawn = p.sim.yaw[r0];
  }
  float sn, cs;
  sincosf(yawn, &sn, &cs);
  p.sim.x[r1] = xn; p.sim.y[r1] = yn; p.sim.yaw[r1] = yawn;
  p.sim.vel_x[r1] = v1 * cs; p.sim.vel_y[r1] = v1 * sn;
  p.sim.length[r1] = Li; p.sim.width[r1] = Wi; p.sim.valid[r1] = 1;
  if (p.accel) p.accel[o] = acc;
  if (p.lead) p.lead[o] = lead;
}

cudaError_t wm_launch_idm_step(wm_handle* h, const wm_traj& sim, int t, const wm_paths& pa, const uint8_t* idm_valid,
                               const wm_idm_params& prm, float* accel, int32_t* lead, cudaStream_t s) {
  IdmParams p{sim, t, pa, idm_valid, prm, h->cfg.dt, accel, lead};
  const int64_t warps = (int64_t)sim.B * sim.A;
  const size_t smem = 8 * (size_t)(3 * pa.P + ((pa.P + 3) >> 2)) * sizeof(float);
  if (smem > 200 * 1024) return cudaErrorInvalidValue;         // P > ~1900 points per path
  if (smem > 40 * 1024) {                          // per-device attribute: set whenever a launch needs it (cheap)
    cudaError_t e = cudaFuncSetAttribute(k_idm_step, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)smem);
    if (e != cudaSuccess) return e;
  }
  k_idm_step<<<(unsigned)((warps + 7) / 8), 256, smem, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}
