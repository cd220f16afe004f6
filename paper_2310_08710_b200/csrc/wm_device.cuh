// Per-agent / per-pair device arithmetic shared by the stepwise kernels (wm_dynamics.cu,
// wm_overlap.cu) and the fused rollout kernel (wm_rollout_fused.cu), so that both paths return
// bit-identical results (P14).
#pragma once
#include "wm_internal.cuh"

// a1 / a2: successor state of one controlled agent.  (sn, cs) = sincosf(th).  For the bicycle
// model (s1, c1) = sincosf(th') is returned as well (Eq. 2 needs it for the velocity).
// PAPER.md Eq. 2 (L339-L350), Eq. 1 (L324-L333) on the body-frame delta rotated by th (D2).
struct WmDynCfg { int dynamics; float dt, max_accel, max_curvature; };

__device__ __forceinline__ void wm_dyn_step(const WmDynCfg& k, float x, float y, float th, float vx, float vy, float sn,
                                            float cs, float a0, float a1, float a2, float& xn, float& yn, float& thn,
                                            float& vxn, float& vyn, float& s1, float& c1) {
  const float dt = k.dt;
  if (k.dynamics == WM_DYN_INVERTIBLE_BICYCLE) {
    float acc = a0, kappa = a1;
    if (k.max_accel > 0.f) acc = fminf(fmaxf(acc, -k.max_accel), k.max_accel);                    // D7
    if (k.max_curvature > 0.f) kappa = fminf(fmaxf(kappa, -k.max_curvature), k.max_curvature);
    const float v = sqrtf(fmaf(vx, vx, vy * vy));
    const float h = 0.5f * acc * dt * dt;            // a dt^2 / 2
    xn = x + fmaf(vx, dt, h * cs);                   // Eq. 2
    yn = y + fmaf(vy, dt, h * sn);                   // L341
    thn = fmaf(kappa, fmaf(v, dt, h), th);           // L343
    const float v1 = fmaf(acc, dt, v);               // L345
    sincosf(thn, &s1, &c1);
    vxn = v1 * c1;                                   // L347
    vyn = v1 * s1;                                   // L349
  } else {
    const float dx = a0, dy = a1, dyaw = a2;
    // explicit roundings: the compiler must not contract these differently in different kernels (P14)
    if (k.dynamics == WM_DYN_DELTA_GLOBAL) {                        // Eq. 1 literally: world-frame delta
      xn = __fadd_rn(x, dx);
      yn = __fadd_rn(y, dy);
    } else {
      xn = __fadd_rn(x, __fmaf_rn(cs, dx, -__fmul_rn(sn, dy)));   // Eq. 1 on the rotated delta (D2)
      yn = __fadd_rn(y, __fmaf_rn(sn, dx, __fmul_rn(cs, dy)));
    }
    thn = __fadd_rn(th, dyaw);
    vxn = __fdiv_rn(__fsub_rn(xn, x), dt);           // Eq. 1: on the stored float32 x' (D28)
    vyn = __fdiv_rn(__fsub_rn(yn, y), dt);
    sincosf(thn, &s1, &c1);
  }
}

// Bicycle inverse, Eq. 3 (L352-L359), readings D4 / D31 / D32: acceleration and steering
// curvature of the transition (th, vx, vy) -> (vx1, vy1).  Expert actor (L204) and kinematic
// infeasibility metric (L104) share it.
__device__ __forceinline__ void wm_inverse_bicycle(float dt, float th, float vx, float vy, float vx1, float vy1, float& acc,
                                                   float& kappa) {
  const float v = sqrtf(fmaf(vx, vx, vy * vy)), v1 = sqrtf(fmaf(vx1, vx1, vy1 * vy1));
  acc = (v1 - v) / dt;                                       // L354
  kappa = 0.f;
  if (!(v == 0.f && v1 == 0.f)) {                            // D31
    const float den = fmaf(v, dt, 0.5f * acc * dt * dt);     // L358
    float d = atan2f(vy1, vx1) - th;                         // D4
    d -= 6.28318530717958647692f * floorf((d + 3.14159265358979323846f) * 0.15915494309189533577f);   // D32: into [-pi, pi)
    kappa = d / den;
  }
}

// a5: displacement error, L106
__device__ __forceinline__ float wm_logdiv(float x, float y, float lx, float ly) {
  const float ex = x - lx, ey = y - ly;
  return sqrtf(fmaf(ex, ex, ey * ey));
}

// a3: strict positive-area overlap (D12): gap < 0 on all four edge-normal axes.
// (dx, dy) = c_j - c_i; (c, s) = cos/sin of each yaw; hl, hw half extents.
__device__ __forceinline__ bool wm_sat_overlap(float dx, float dy, float ci, float si, float hli, float hwi,
                                               float cj, float sj, float hlj, float hwj) {
  const float c = fabsf(fmaf(ci, cj, si * sj));      // |f_i . f_j| = |s_i . s_j|
  const float s = fabsf(fmaf(si, cj, -ci * sj));     // |f_i . s_j| = |s_i . f_j|
  const float g0 = fabsf(fmaf(dx, ci, dy * si)) - (hli + fmaf(hlj, c, hwj * s));    // axis f_i
  const float g1 = fabsf(fmaf(dy, ci, -dx * si)) - (hwi + fmaf(hlj, s, hwj * c));   // axis s_i
  const float g2 = fabsf(fmaf(dx, cj, dy * sj)) - (hlj + fmaf(hli, c, hwi * s));    // axis f_j
  const float g3 = fabsf(fmaf(dy, cj, -dx * sj)) - (hwj + fmaf(hli, s, hwi * c));   // axis s_j
  return fmaxf(fmaxf(g0, g1), fmaxf(g2, g3)) < 0.f;
}

// Conservative pre-test of a3: two boxes can only overlap if their centres are closer than the
// sum of their circumradii (rr = r_i + r_j).  The 1.001 factor and the absolute term keep the
// float32 test on the safe side, so skipping the separating-axis test never changes a result.
__device__ __forceinline__ bool wm_circles_touch(float dx, float dy, float rr) {
  return fmaf(dx, dx, dy * dy) <= fmaf(rr * rr, 1.001f, 1e-6f);
}
