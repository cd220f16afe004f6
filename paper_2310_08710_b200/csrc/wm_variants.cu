// Variants of the hot path:
//   k_rollout_vjp   backward pass of the dynamics a1 / a2 for differentiable rollouts:
//                   the vector-Jacobian product of Eq. 2 (L339-L350) / Eq. 1 (L324-L333), chained in
//                   reverse over the rows of a rollout.  One thread per (scenario, agent); per step it
//                   reads one state row (yaw, v_x, v_y, valid: 13 B), the action and five cotangents and
//                   writes the action cotangents: HBM bound (~45 B per agent-step).
//   k_discretize    discretised action spaces (L204): nearest value of a uniform grid per channel,
//                   joint index + de-quantised action; k_from_index: the decode.
#include "wm_device.cuh"

// ---------------------------------------------------------------------------------------
// backward pass (readings D43: playback slots and clipped actions pass no gradient; dv/dv_x = 0 at v = 0;
// Eq. 1's v' = (x' - x)/dt differentiates as written)
// ---------------------------------------------------------------------------------------
struct VjpParams {
  wm_traj sim;
  int t0, n_steps, dynamics;
  float dt, max_accel, max_curvature;
  const float* actions;      // [B][n_steps][C][A]
  const uint8_t* av;         // [B][n_steps][A]
  const float* g_rows;       // [B][n_steps][5][A]
  float* g_actions;          // [B][n_steps][C][A]
  float* g_state0;           // [B][5][A], may be NULL
};

__global__ void __launch_bounds__(128) k_rollout_vjp(VjpParams p) {
  const int A = p.sim.A;
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= (int64_t)p.sim.B * A) return;
  const int b = (int)(i / A), a = (int)(i % A);
  const bool bicycle = p.dynamics == WM_DYN_INVERTIBLE_BICYCLE;
  const int C = bicycle ? 2 : 3;
  const float dt = p.dt, hdt2 = 0.5f * dt * dt;
  float gx = 0.f, gy = 0.f, gth = 0.f, gvx = 0.f, gvy = 0.f;       // cotangent of row t0+k+1, carried backwards
#pragma unroll 1
  for (int k = p.n_steps - 1; k >= 0; --k) {
    const int64_t rk = (int64_t)b * p.n_steps + k;
    const float* gr = p.g_rows + rk * 5 * A + a;
    gx += __ldcs(gr); gy += __ldcs(gr + A); gth += __ldcs(gr + 2 * (int64_t)A);
    gvx += __ldcs(gr + 3 * (int64_t)A); gvy += __ldcs(gr + 4 * (int64_t)A);
    const int64_t r0 = ((int64_t)b * p.sim.T + p.t0 + k) * A + a;
    const float* act = p.actions + rk * C * A + a;
    float* ga = p.g_actions + rk * C * A + a;
    const bool use_dyn = p.av[rk * A + a] != 0 && p.sim.valid[r0] != 0;       // D8
    float o0 = 0.f, o1 = 0.f, o2 = 0.f;
    if (!use_dyn) { gx = gy = gth = gvx = gvy = 0.f; }                          // the successor came from the log
    else {
      const float th = p.sim.yaw[r0];
      float s0, c0;
      sincosf(th, &s0, &c0);
      if (bicycle) {
        const float vx = p.sim.vel_x[r0], vy = p.sim.vel_y[r0];
        float acc = act[0], kappa = act[A];
        float da = 1.f, dk = 1.f;
        if (p.max_accel > 0.f) { if (fabsf(acc) > p.max_accel) da = 0.f; acc = fminf(fmaxf(acc, -p.max_accel), p.max_accel); }
        if (p.max_curvature > 0.f) { if (fabsf(kappa) > p.max_curvature) dk = 0.f; kappa = fminf(fmaxf(kappa, -p.max_curvature), p.max_curvature); }
        const float v = sqrtf(fmaf(vx, vx, vy * vy));
        const float adv = fmaf(v, dt, acc * hdt2);                    // v dt + a dt^2 / 2
        const float thn = fmaf(kappa, adv, th), vn = fmaf(acc, dt, v);
        float s1, c1;
        sincosf(thn, &s1, &c1);
        const float gvn = fmaf(gvx, c1, gvy * s1);
        const float gthn = fmaf(vn, fmaf(gvy, c1, -gvx * s1), gth);
        const float gv = fmaf(gthn * kappa, dt, gvn);
        o1 = gthn * adv * dk;
        o0 = (fmaf(gvn, dt, gthn * kappa * hdt2) + hdt2 * fmaf(gx, c0, gy * s0)) * da;
        const float nth = fmaf(acc * hdt2, fmaf(gy, c0, -gx * s0), gthn);
        const float ux = v > 0.f ? vx / v : 0.f, uy = v > 0.f ? vy / v : 0.f;
        gvx = fmaf(gx, dt, gv * ux); gvy = fmaf(gy, dt, gv * uy);
        gth = nth;                                                    // gx, gy pass through
      } else {
        const bool glob = p.dynamics == WM_DYN_DELTA_GLOBAL;
        const float c = glob ? 1.f : c0, s = glob ? 0.f : s0;
        const float dx = act[0], dy = act[A];
        const float hx = gx + gvx / dt, hy = gy + gvy / dt;           // cotangents of the world-frame delta
        o0 = fmaf(hx, c, hy * s); o1 = fmaf(hy, c, -hx * s); o2 = gth;
        if (!glob) gth += fmaf(hx, -fmaf(s, dx, c * dy), hy * fmaf(c, dx, -s * dy));
        gvx = 0.f; gvy = 0.f;
      }
    }
    __stcs(ga, o0); __stcs(ga + A, o1);
    if (C == 3) __stcs(ga + 2 * (int64_t)A, o2);
  }
  if (p.g_state0) {
    float* g0 = p.g_state0 + (int64_t)b * 5 * A + a;
    g0[0] = gx; g0[A] = gy; g0[2 * (int64_t)A] = gth; g0[3 * (int64_t)A] = gvx; g0[4 * (int64_t)A] = gvy;
  }
}

cudaError_t wm_launch_rollout_vjp(wm_handle* h, const wm_traj& sim, int t0, int n_steps, const float* actions, const uint8_t* av,
                                  const float* g_rows, float* g_actions, float* g_state0, cudaStream_t s) {
  VjpParams p{sim, t0, n_steps, h->cfg.dynamics, h->cfg.dt, h->cfg.max_accel, h->cfg.max_curvature, actions, av, g_rows, g_actions, g_state0};
  const int64_t n = (int64_t)sim.B * sim.A;
  k_rollout_vjp<<<(unsigned)((n + 127) / 128), 128, 0, s>>>(p);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// discretised action spaces (D42): bin = clamp(rint((v - lo) * inv_step), 0, n - 1) in float32,
// inv_step = fl((n - 1) / (hi - lo)); value = lo + bin * (hi - lo) / (n - 1) in double, rounded once
// ---------------------------------------------------------------------------------------
struct GridDev { int n[3]; float lo[3], hi[3]; };

// lo + bin * (hi - lo) / (n - 1) in double, every operation rounded on its own (no contraction), then one rounding to float32
__device__ __forceinline__ float grid_value(const GridDev& g, int c, int bin) {
  const double step = g.n[c] > 1 ? __ddiv_rn(__dsub_rn((double)g.hi[c], (double)g.lo[c]), (double)(g.n[c] - 1)) : 0.0;
  return (float)__dadd_rn((double)g.lo[c], __dmul_rn((double)bin, step));
}

__global__ void __launch_bounds__(256) k_discretize(GridDev g, int C, int64_t N, int A, const float* action, const uint8_t* valid,
                                                    int32_t* index, float* dequant) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= N * A) return;
  const int64_t r = i / A;
  const int a = (int)(i - r * A);
  const bool v = valid == nullptr || valid[i] != 0;
  int idx = 0;
  for (int c = 0; c < C; ++c) {
    const int64_t o = (r * C + c) * A + a;
    const int n = g.n[c];
    int bin = 0;
    if (v && n > 1) {
      const float inv_step = __fdiv_rn((float)(n - 1), __fsub_rn(g.hi[c], g.lo[c]));
      const float q = rintf(__fmul_rn(__fsub_rn(action[o], g.lo[c]), inv_step));        // round half to even
      bin = !(q == q) ? 0 : q <= 0.f ? 0 : q >= (float)(n - 1) ? n - 1 : (int)q;
    }
    idx = idx * n + bin;
    if (dequant) {
      dequant[o] = v ? grid_value(g, c, bin) : 0.f;
    }
  }
  index[i] = v ? idx : -1;
}

__global__ void __launch_bounds__(256) k_from_index(GridDev g, int C, int64_t N, int A, const int32_t* index, float* action) {
  const int64_t i = blockIdx.x * (int64_t)blockDim.x + threadIdx.x;
  if (i >= N * A) return;
  const int64_t r = i / A;
  const int a = (int)(i - r * A);
  int idx = index[i];
  int64_t total = 1;
  for (int c = 0; c < C; ++c) total *= g.n[c];
  if ((int64_t)idx >= total) idx = -1;                     // D45: not a bin of this grid -> no action, like index < 0
  for (int c = C - 1; c >= 0; --c) {
    const int64_t o = (r * C + c) * A + a;
    const int n = g.n[c];
    float val = 0.f;
    if (idx >= 0) {
      const int bin = idx % n;
      idx /= n;
      val = grid_value(g, c, bin);
    }
    action[o] = val;
  }
}

static GridDev grid_dev(const wm_action_grid& g) {
  GridDev d;
  for (int c = 0; c < 3; ++c) { d.n[c] = g.n[c]; d.lo[c] = g.lo[c]; d.hi[c] = g.hi[c]; }
  return d;
}

cudaError_t wm_launch_discretize(wm_handle* h, const wm_action_grid& g, int C, int64_t N, int A, const float* action,
                                 const uint8_t* valid, int32_t* index, float* dequant, cudaStream_t s) {
  k_discretize<<<(unsigned)((N * A + 255) / 256), 256, 0, s>>>(grid_dev(g), C, N, A, action, valid, index, dequant);
  h->launches++;
  return cudaGetLastError();
}

cudaError_t wm_launch_from_index(wm_handle* h, const wm_action_grid& g, int C, int64_t N, int A, const int32_t* index, float* action,
                                 cudaStream_t s) {
  k_from_index<<<(unsigned)((N * A + 255) / 256), 256, 0, s>>>(grid_dev(g), C, N, A, index, action);
  h->launches++;
  return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------
// wm_selftest_ffma: the FP32 peak of this GPU as a register-resident FMA loop can reach it (the
// denominator SURVEY 8(d) asks to MEASURE in the same run as the brute-force offroad kernel):
// 8 independent accumulator chains per thread, scalar FFMA or packed FFMA2, no memory traffic.
// ---------------------------------------------------------------------------------------
template <bool PACKED>
__global__ void __launch_bounds__(256) k_ffma_peak(int iters, float seed, float* sink) {
  float a = seed + (float)threadIdx.x * 1e-6f, b = 0.999f;
  if (PACKED) {
    wm_u64 acc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = pk2(a + (float)j, a - (float)j);
    const wm_u64 m = pk2(b, b), c = pk2(1e-3f, -1e-3f);
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] = fma2(acc[j], m, c);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) { float lo, hi; upk2(acc[j], lo, hi); s += lo + hi; }
    if (s == 12345.678f) sink[0] = s;                      // never true: keeps the loop alive
  } else {
    float acc[8];
#pragma unroll
    for (int j = 0; j < 8; ++j) acc[j] = a + (float)j;
    for (int i = 0; i < iters; ++i) {
#pragma unroll
      for (int u = 0; u < 4; ++u)
#pragma unroll
        for (int j = 0; j < 8; ++j) acc[j] = fmaf(acc[j], b, 1e-3f);
    }
    float s = 0.f;
#pragma unroll
    for (int j = 0; j < 8; ++j) s += acc[j];
    if (s == 12345.678f) sink[0] = s;
  }
}

// flops of one launch = CTAs * 256 threads * iters * 32 FMA (* 2 lanes when packed) * 2
cudaError_t wm_launch_ffma_peak(wm_handle* h, int packed, int ctas, int iters, float* sink, cudaStream_t s) {
  if (packed) k_ffma_peak<true><<<ctas, 256, 0, s>>>(iters, 1.0f, sink);
  else k_ffma_peak<false><<<ctas, 256, 0, s>>>(iters, 1.0f, sink);
  h->launches++;
  return cudaGetLastError();
}
